// mvd_sep.cu -- separable fast path of the direct engine (sm_100a).
//
// When every PSF of a plan is an outer product, P_v[j][i] = u_v[j] w_v[i] (Gaussian PSFs are: BASELINE.json's configs
// 1, 2 and 4), the two correlations of a view update (a1 with the flipped PSF, a3 with the PSF as given)
// factor into a pass along x and a pass along z: 2 K FMAs per output instead of K^2.  Steps a1+a2 and a3+a4 stay two
// fused kernels exactly like mvd_direct.cu's, so HBM still sees 22 B per voxel-view-iteration -- about half of the
// FFT engine's 42 B -- and the FP32 pipe sees ~2 K (1 + 128 / TY) FMAs instead of K^2.
//
// One CTA (256 threads) owns a TY x 32 output tile of a PAIR of planes (float2 = (plane a, plane b), FFMA2 with the
// tap as broadcast operand), TY = 128 - (K - 1):
//   1. stage   the (128) x (32 + K - 1) source tile with its periodically wrapped halo, TRANSPOSED, in shared memory:
//              sT[x'][y'], pitch 129 float2, so that lanes along y' read consecutive 8-byte words (conflict-free)
//   2. x pass  thread (y' = tid % 128, strip = tid / 128) slides a K-tap window along x over 16 outputs of row y':
//              16 + K - 1 shared loads for 16 K FFMA2; result t[y'][x], pitch 33 float2
//   3. z pass  thread (x = tid % 32, strip = tid / 32) slides the window down its column over RY = ceil(TY / 8)
//              outputs: RY + K - 1 shared loads (lanes along x: conflict-free) for RY K FFMA2; epilogue a2 or a4
// K is a template parameter for the config sizes (fully unrolled windows); other K run in chunks of 8 taps.
#include <math.h>

#include <algorithm>
#include <vector>

#include "mvd_internal.cuh"

namespace {

constexpr int NT = 256;      // threads per CTA
constexpr int RS = 128;      // staged rows per tile (outputs + halo)
constexpr int TX = 32;       // output columns per tile
constexpr int RX = 16;       // outputs per thread in the x pass
constexpr int P1 = RS + 2;   // pitch of the transposed source tile (float2): 4 P1 = 8 mod 16, see the staging loop
constexpr int P2 = TX + 1;   // pitch of the intermediate (float2)
constexpr int NSTRIP = NT / TX;   // strips of the z pass

__device__ __forceinline__ float2 ffma2_b(float g, float2 w, float2 c) {
    float2 r;
    asm("{ .reg .b64 ra, rb, rc, rd; mov.b64 ra, {%2,%2}; mov.b64 rb, {%3,%4}; mov.b64 rc, {%5,%6}; "
        "fma.rn.f32x2 rd, ra, rb, rc; mov.b64 {%0,%1}, rd; }"
        : "=f"(r.x), "=f"(r.y) : "f"(g), "f"(w.x), "f"(w.y), "f"(c.x), "f"(c.y));
    return r;
}

// staged columns of a tile: the alignment shift of the vectorised staging + TX + K - 1, rounded up to whole float4 groups
__host__ __device__ constexpr int sep_swa(int K) { return ((4 - ((K - 1) / 2) % 4) % 4 + TX + K - 1 + 3) & ~3; }

__device__ __forceinline__ void cp_async16(float* dst, const float* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async4(float* dst, const float* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}

// acc[0 .. N) += sum_{j < JC} g[j] * win[m + j]: a JC-tap chunk of a sliding window, everything in registers
template <int N, int JC>
__device__ __forceinline__ void window_fma(float2 (&acc)[N], const float2 (&win)[N + JC - 1], const float (&g)[JC]) {
#pragma unroll
    for (int j = 0; j < JC; ++j)
#pragma unroll
        for (int m = 0; m < N; ++m) acc[m] = ffma2_b(g[j], win[m + j], acc[m]);
}

struct SepArgs {
    const float* src;        // psi (MODE 0) or r (MODE 1), [n][H][W]
    const float* taps;       // [2][Kp]: gz (z pass), gx (x pass) of this view and mode, zero-padded to Kp
    const uint16_t* phi;     // MODE 0: this view's planes
    float* dst;              // MODE 0: r; MODE 1: psi (read-modify-write)
    const float* wgt;        // MODE 1: nullptr or this view's weights (a4w)
    size_t phi_plane, phi_row;
    int W, H, K, Kp, n_planes, tiles_x, tiles_y, n_sm;
    float eps;
};

// KT > 0: K known at compile time, JC == KT (one fully unrolled window); KT == 0: runtime K in chunks of JC taps.
//
// PERSISTENT: one CTA per SM walks the tiles.  The source rows of the NEXT tile stream into a row-major landing
// buffer (`raw`, cp.async, 16 bytes at a time when W is a multiple of 4) while the current tile is computed, so no
// global-load latency is left on the critical path; each tile then costs one shared-memory transposition
// (raw -> sT, interleaving the two planes), the two passes and its stores.
template <int KT, int JC, int MODE, bool VEC, bool WGT>
__global__ void __launch_bounds__(NT, 1) sep_corr2_kernel(SepArgs a) {
    extern __shared__ __align__(16) float2 sep_smem[];
    const int K = KT > 0 ? KT : a.K, Kp = KT > 0 ? KT : a.Kp;
    const int c = (K - 1) / 2;
    const int TY = RS - (K - 1);               // output rows per tile
    constexpr int RYC = KT > 0 ? (RS - (KT - 1) + NSTRIP - 1) / NSTRIP : RS / NSTRIP;   // outputs per thread, z pass
    // The windows of the last strips reach a few rows / columns past the tile: those are zero-filled spares
    // (ZC spare columns of sT for the chunked runtime-K window, ZR spare rows of tt), so no load needs a guard.
    constexpr int ZC = KT > 0 ? 0 : 8, ZR = 16;
    const int SWA = sep_swa(K);                // staged columns: alignment shift + TX + K - 1, whole float4 groups
    const int RP = SWA + 4;                    // pitch of a landing row (floats): rows 8 apart fall into distinct 16-byte bank groups
    float2* sT = sep_smem;                            // [SWA + ZC][P1]   source tile, transposed, (plane a, plane b)
    float2* tt = sep_smem + (size_t)(SWA + ZC) * P1;  // [RS + ZR][P2]    result of the x pass
    float* raw = reinterpret_cast<float*>(tt + (size_t)(RS + ZR) * P2);   // [2][RS][RP]  landing buffer of the next tile
    float* sg = raw + (size_t)2 * RS * RP;            // [2][Kp] taps
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int k = tid; k < ZC * P1; k += NT) sT[(size_t)SWA * P1 + k] = make_float2(0.f, 0.f);
    for (int k = tid; k < ZR * P2; k += NT) tt[(size_t)RS * P2 + k] = make_float2(0.f, 0.f);
    for (int k = tid; k < 2 * Kp; k += NT) sg[k] = a.taps[k];

    const int W = a.W, H = a.H;
    const size_t npx = (size_t)W * H;
    // the staged columns start `shift` columns before x0 - c, at a multiple of 4 (x0 is a multiple of 32)
    const int shift = (4 - c % 4) % 4;
    const int G = SWA / 4;                     // float4 groups per staged row
    const int n_tiles = a.tiles_x * a.tiles_y * ((a.n_planes + 1) / 2);

    // rows of tile `t` -> raw: raw[p][ty][0 .. SWA) = src_p(y0 - c + ty, x0 - c - shift + ...), periodic
    auto issue = [&](int t) {
        const int tile_x = t % a.tiles_x, tile_y = (t / a.tiles_x) % a.tiles_y, pa = 2 * (t / (a.tiles_x * a.tiles_y));
        const size_t offa = (size_t)pa * npx, offb = pa + 1 < a.n_planes ? offa + npx : offa;
        const int xa = tile_x * TX - c - shift, ya = tile_y * TY - c;
        // lanes along a row (no division in the loop): warp w takes rows w, w + 8, ...
        int gy = (ya + warp) % H;
        if (gy < 0) gy += H;
        if (VEC) {
            const int grp = lane;                                  // G <= 24 groups per row: the other lanes idle
            int gx = (xa + 4 * min(grp, G - 1)) % W;
            if (gx < 0) gx += W;
            for (int ty = warp; ty < RS; ty += NT / 32) {
                if (grp < G) {
                    const size_t g = (size_t)gy * W + gx;
                    cp_async16(raw + (size_t)ty * RP + 4 * grp, a.src + offa + g);
                    cp_async16(raw + (size_t)(RS + ty) * RP + 4 * grp, a.src + offb + g);
                }
                gy += NT / 32;
                if (gy >= H) gy = H >= NT / 32 ? gy - H : gy % H;
            }
        } else {
            for (int tx = lane; tx < SWA; tx += 32) {
                int gx = (xa + tx) % W;
                if (gx < 0) gx += W;
                int gyy = gy;
                for (int ty = warp; ty < RS; ty += NT / 32) {
                    const size_t g = (size_t)gyy * W + gx;
                    cp_async4(raw + (size_t)ty * RP + tx, a.src + offa + g);
                    cp_async4(raw + (size_t)(RS + ty) * RP + tx, a.src + offb + g);
                    gyy += NT / 32;
                    if (gyy >= H) gyy = H >= NT / 32 ? gyy - H : gyy % H;
                }
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    int tile = blockIdx.x;
    if (tile < n_tiles) issue(tile);
    for (; tile < n_tiles; tile += gridDim.x) {
        int b = tile;
        const int tile_x = b % a.tiles_x; b /= a.tiles_x;
        const int tile_y = b % a.tiles_y; b /= a.tiles_y;      // b: pair
        const int pa = 2 * b;
        const bool has_b = pa + 1 < a.n_planes;
        const size_t offa = (size_t)pa * npx, offb = has_b ? offa + npx : offa;
        const int x0 = tile_x * TX, y0 = tile_y * TY;

        // The epilogue's operands (phi, or the old psi and the weights) are requested now, so that their latency hides
        // behind the passes (and no load has to wait for a store the compiler cannot prove independent).  Branch-free:
        // coordinates past the plane are clamped, the values discarded later; phi stays uint16 until then.
        const int ex = tid % TX, eys = (tid / TX) * RYC, gxo = x0 + ex;
        const int gxc = min(gxo, W - 1);
        float ea[MODE == 1 ? RYC : 1], eb[MODE == 1 ? RYC : 1], wa[WGT ? RYC : 1], wb[WGT ? RYC : 1];
        unsigned short ua[MODE == 0 ? RYC : 1], ub[MODE == 0 ? RYC : 1];
#pragma unroll
        for (int m = 0; m < RYC; ++m) {
            const int yc = min(y0 + eys + m, H - 1);
            const size_t q = (size_t)yc * W + gxc;
            if constexpr (MODE == 0) {
                const size_t f = (size_t)pa * a.phi_plane + (size_t)yc * a.phi_row + gxc;
                ua[m] = __ldg(a.phi + f);
                ub[m] = __ldg(a.phi + (has_b ? f + a.phi_plane : f));
            } else {
                ea[m] = a.dst[offa + q];
                eb[m] = a.dst[offb + q];
            }
        }
        if constexpr (WGT) {
#pragma unroll
            for (int m = 0; m < RYC; ++m) {
                const int yc = min(y0 + eys + m, H - 1);
                const size_t q = (size_t)yc * W + gxc;
                wa[m] = __ldg(a.wgt + offa + q);
                wb[m] = __ldg(a.wgt + offb + q);
            }
        }

        // 1. raw -> sT, transposed and interleaved.  A warp takes 8 rows x 4 groups at a time: its 16-byte loads hit
        // distinct bank groups (pitch RP), its transposed 8-byte stores 16 distinct banks per half-warp (rows: 8
        // consecutive words; groups: 4 P1 words apart = 8 banks further).
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();        // the landing buffer is complete; everybody is done with sT and tt of the previous tile
        for (int rb = warp; rb < RS / 8; rb += NT / 32) {
            const int ty = 8 * rb + (lane & 7);
            for (int g0 = 0; g0 < G; g0 += 4) {
                const int grp = min(g0 + (lane >> 3), G - 1);   // (groups past the end repeat the last one)
                const float4 va = *reinterpret_cast<const float4*>(raw + (size_t)ty * RP + 4 * grp);
                const float4 vb = *reinterpret_cast<const float4*>(raw + (size_t)(RS + ty) * RP + 4 * grp);
                float2* d = sT + (size_t)(4 * grp) * P1 + ty;
                d[0] = make_float2(va.x, vb.x);
                d[P1] = make_float2(va.y, vb.y);
                d[2 * P1] = make_float2(va.z, vb.z);
                d[3 * P1] = make_float2(va.w, vb.w);
            }
        }
        __syncthreads();        // sT is complete, the landing buffer is free
        if (tile + (int)gridDim.x < n_tiles) issue(tile + gridDim.x);

        {   // 2. x pass: t(ty, x) = sum_i gx[i] s(ty, x + i)
            const int ty = tid % RS, xs = (tid / RS) * RX;
            const float* gx = sg + Kp;
            const float2* col = sT + (size_t)(xs + shift) * P1 + ty;
            float2 acc[RX];
#pragma unroll
            for (int m = 0; m < RX; ++m) acc[m] = make_float2(0.f, 0.f);
            for (int jc = 0; jc < Kp; jc += JC) {
                float2 win[RX + JC - 1];
#pragma unroll
                for (int n = 0; n < RX + JC - 1; ++n) win[n] = col[(size_t)(jc + n) * P1];
                float g[JC];
#pragma unroll
                for (int j = 0; j < JC; ++j) g[j] = gx[jc + j];
                window_fma<RX, JC>(acc, win, g);
            }
#pragma unroll
            for (int m = 0; m < RX; ++m) tt[ty * P2 + xs + m] = acc[m];
        }
        __syncthreads();

        {   // 3. z pass: out(y, x) = sum_j gz[j] t(y + j, x); epilogue
            const int x = tid % TX, ys = (tid / TX) * RYC;
            const float* gz = sg;
            const float2* col = tt + (size_t)ys * P2 + x;
            float2 acc[RYC];
#pragma unroll
            for (int m = 0; m < RYC; ++m) acc[m] = make_float2(0.f, 0.f);
            for (int jc = 0; jc < Kp; jc += JC) {
                float2 win[RYC + JC - 1];
#pragma unroll
                for (int n = 0; n < RYC + JC - 1; ++n)
                    win[n] = (KT > 0 || ys + jc + n < RS + ZR) ? col[(size_t)(jc + n) * P2] : make_float2(0.f, 0.f);
                float g[JC];
#pragma unroll
                for (int j = 0; j < JC; ++j) g[j] = gz[jc + j];
                window_fma<RYC, JC>(acc, win, g);
            }
            if (gxo < W) {
#pragma unroll
                for (int m = 0; m < RYC; ++m) {
                    const int ly = ys + m, y = y0 + ly;
                    if (ly < TY && y < H) {
                        const size_t q = (size_t)y * W + gxo;
                        if constexpr (MODE == 0) {                                    // a2
                            a.dst[offa + q] = __fdividef((float)ua[m], fmaxf(acc[m].x, a.eps));      // 2 ulp, reading A16
                            if (has_b) a.dst[offb + q] = __fdividef((float)ub[m], fmaxf(acc[m].y, a.eps));
                        } else {                                                      // a4 (a4w: q <- w q + 1 - w)
                            float qa = acc[m].x, qb = acc[m].y;
                            if constexpr (WGT) {
                                qa = fmaf(wa[m], qa, 1.f - wa[m]);
                                qb = fmaf(wb[m], qb, 1.f - wb[m]);
                            }
                            a.dst[offa + q] = ea[m] * qa;
                            if (has_b) a.dst[offb + q] = eb[m] * qb;
                        }
                    }
                }
            }
        }
    }
}

size_t sep_smem_bytes(int K, int Kp) {
    const bool templated = Kp == K;
    return sizeof(float2) * ((size_t)(sep_swa(K) + (templated ? 0 : 8)) * P1 + (size_t)(RS + 16) * P2) +
           sizeof(float) * ((size_t)2 * RS * (sep_swa(K) + 4) + 2 * Kp);
}

template <int KT, int JC, int MODE, bool VEC, bool WGT = false>
int launch_sep_one(const SepArgs& a, size_t smem, unsigned grid, cudaStream_t st) {
    static size_t opted = 0;
    if (smem > opted) {
        cudaError_t e = cudaFuncSetAttribute(sep_corr2_kernel<KT, JC, MODE, VEC, WGT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return (int)e;
        opted = smem;
    }
    sep_corr2_kernel<KT, JC, MODE, VEC, WGT><<<grid, NT, smem, st>>>(a);
    return (int)cudaGetLastError();
}

template <int KT, int JC>
int launch_sep(int mode, const SepArgs& a, cudaStream_t st) {
    const size_t smem = sep_smem_bytes(a.K, a.Kp);
    const size_t n_tiles = (size_t)a.tiles_x * a.tiles_y * ((a.n_planes + 1) / 2);
    const unsigned grid = (unsigned)std::min<size_t>(n_tiles, (size_t)a.n_sm);
    const bool vec = a.W % 4 == 0 && ((uintptr_t)a.src & 15u) == 0;   // planes are W H floats apart: aligned too
    if (mode == 0) return vec ? launch_sep_one<KT, JC, 0, true>(a, smem, grid, st) : launch_sep_one<KT, JC, 0, false>(a, smem, grid, st);
    if (a.wgt) return vec ? launch_sep_one<KT, JC, 1, true, true>(a, smem, grid, st) : launch_sep_one<KT, JC, 1, false, true>(a, smem, grid, st);
    return vec ? launch_sep_one<KT, JC, 1, true>(a, smem, grid, st) : launch_sep_one<KT, JC, 1, false>(a, smem, grid, st);
}

}  // namespace

// P ~ u w^T ?  For an outer product the row sums are u (sum w) and the column sums w (sum u), so
// P = rowsum (x) colsum / total; accepted when the residual is below 1e-6 of ||P||_F (fp32 rounding of an exact
// outer product leaves ~3e-8).
bool sep_factor(const float* P, int K, std::vector<double>& u, std::vector<double>& w) {
    u.assign(K, 0.0);
    w.assign(K, 0.0);
    double total = 0.0, norm2 = 0.0;
    for (int j = 0; j < K; ++j)
        for (int i = 0; i < K; ++i) {
            const double p = P[(size_t)j * K + i];
            u[j] += p;
            w[i] += p;
            total += p;
            norm2 += p * p;
        }
    if (!(total > 0.0) || !(norm2 > 0.0)) return false;
    for (int i = 0; i < K; ++i) w[i] /= total;
    double res2 = 0.0;
    for (int j = 0; j < K; ++j)
        for (int i = 0; i < K; ++i) {
            const double d = (double)P[(size_t)j * K + i] - u[j] * w[i];
            res2 += d * d;
        }
    return res2 <= 1e-12 * norm2;
}

bool sep_psfs_separable(int n_views, const float* psfs, int K) {
    if (K < 3 || K > 65) return false;     // TY = 128 - (K - 1) >= 64 output rows per tile
    std::vector<double> u, w;
    for (int v = 0; v < n_views; ++v)
        if (!sep_factor(psfs + (size_t)v * K * K, K, u, w)) return false;
    return true;
}

// taps: [V][2 (a1, a3)][2 (gz, gx)][Kp]; a1 correlates with the FLIPPED factors (convolution), a3 with them as given
int sep_setup(mvd_handle* h, const float* host_psfs) {
    h->sep = false;
    if (h->KX || !sep_psfs_separable(h->V, host_psfs, h->K)) return MVD_OK;
    const int K = h->K;
    int JC, Kp;
    direct_choose_chunk(K, &JC, &Kp);
    const bool templated = K == 9 || K == 21 || K == 31 || K == 41 || K == 51;
    if (templated) Kp = K;
    else Kp = (K + 7) / 8 * 8;
    if (sep_smem_bytes(K, Kp) > 227u * 1024u) return MVD_OK;
    std::vector<float> taps((size_t)h->V * 4 * Kp, 0.f);
    std::vector<double> u, w;
    for (int v = 0; v < h->V; ++v) {
        sep_factor(host_psfs + (size_t)v * K * K, K, u, w);
        float* t = taps.data() + (size_t)v * 4 * Kp;
        for (int k = 0; k < K; ++k) {
            t[0 * Kp + k] = (float)u[K - 1 - k];   // a1 gz
            t[1 * Kp + k] = (float)w[K - 1 - k];   // a1 gx
            t[2 * Kp + k] = (float)u[k];           // a3 gz
            t[3 * Kp + k] = (float)w[k];           // a3 gx
        }
    }
    MVD_TRY(h, cudaMalloc((void**)&h->d_sep, taps.size() * sizeof(float)));
    MVD_TRY(h, cudaMemcpy(h->d_sep, taps.data(), taps.size() * sizeof(float), cudaMemcpyHostToDevice));
    h->sepKp = Kp;
    h->sep = true;
    return MVD_OK;
}

int sep_launch(int mode, const mvd_handle* h, int v, const float* src, const uint16_t* phi, float* dst, int n_planes,
               cudaStream_t st, size_t phi_plane, size_t phi_row, const float* wgt) {
    SepArgs a;
    a.src = src;
    a.taps = h->d_sep + ((size_t)v * 4 + (mode ? 2 : 0)) * h->sepKp;
    a.phi = phi;
    a.dst = dst;
    a.wgt = wgt;
    a.phi_plane = phi_plane;
    a.phi_row = phi_row;
    a.W = h->W; a.H = h->H; a.K = h->K; a.Kp = h->sepKp; a.n_planes = n_planes;
    a.tiles_x = (h->W + TX - 1) / TX;
    a.tiles_y = (h->H + (RS - (h->K - 1)) - 1) / (RS - (h->K - 1));
    a.eps = h->eps;
    a.n_sm = h->n_sm;
    switch (h->K) {
        case 9: return launch_sep<9, 9>(mode, a, st);
        case 21: return launch_sep<21, 21>(mode, a, st);
        case 31: return launch_sep<31, 31>(mode, a, st);
        case 41: return launch_sep<41, 41>(mode, a, st);
        case 51: return launch_sep<51, 51>(mode, a, st);
        default: return launch_sep<0, 8>(mode, a, st);
    }
}
