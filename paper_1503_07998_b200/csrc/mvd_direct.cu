// mvd_direct.cu -- direct (spatial-domain) engine of libmvd for sm_100a.
//
// Steps a1..a4 of the per-plane RL view update as two fused kernels:
//   kernel A  b = psi (*) P_v (periodic convolution, a1);  r = phi_v / max(b, eps) (a2)  -> r
//   kernel B  q = r (*) P_v^* (periodic correlation, a3);  psi <- psi . q (a4)           -> psi
// Both are the same correlation   out(y,x) = sum_{j,i} G[j][i] * src(y + j - c, x + i - c)   with
// G = P_v flipped in both axes for a1 (convolution) and G = P_v as given for a3.
//
// Mapping (B200): a CTA owns a BX x (BY*RY) output tile of one plane, stages the tile plus its
// wrapped halo in shared memory once, and each thread accumulates RY outputs of one image column in
// registers: for one PSF column i it reads a (RY+JC-1)-tall window of the staged column (one
// conflict-free LDS per value, lanes along x) and issues JC*RY FFMAs on it.  The FP32 FMA pipe is
// the bound (4 K^2 flop against 22 B of HBM traffic per voxel-view-iteration).
#include "mvd_internal.cuh"

namespace {

constexpr int BX = 64;   // tile width  (threads along x)
constexpr int BY = 4;    // thread rows
constexpr int RY = 16;   // outputs per thread along y
constexpr int TILE_H = BY * RY;

__device__ __forceinline__ int pmod(int a, int m) {
    int r = a % m;
    return r < 0 ? r + m : r;
}

// a0: psi_0 = mean of the views (exact sum in fp32: <= 2^16 * V < 2^24 for V <= 255)
__global__ void init_mean_kernel(const uint16_t* __restrict__ views, ViewLayout lay, int V, int W, int H,
                                 float* __restrict__ psi, size_t n) {
    const float inv_is_exact_division = (float)V;
    const size_t npx = (size_t)W * H;
    for (size_t p = blockIdx.x * (size_t)blockDim.x + threadIdx.x; p < n;
         p += (size_t)gridDim.x * blockDim.x) {
        const size_t plane = p / npx, rem = p % npx;
        const size_t q = plane * lay.plane + (rem / W) * lay.row + rem % W;
        float s = 0.f;
        for (int v = 0; v < V; ++v) s += (float)views[(size_t)v * lay.view + q];
        psi[p] = s / inv_is_exact_division;
    }
}

// KT > 0: PSF size known at compile time (immediate shared-memory offsets); KT == 0: runtime K.
// MODE 0: kernel A (ratio epilogue).  MODE 1: kernel B (multiplicative update epilogue).
template <int KT, int JC, int MODE>
__global__ void __launch_bounds__(BX* BY)
direct_corr_kernel(const float* __restrict__ src, const float* __restrict__ G,
                   const uint16_t* __restrict__ phi, float* __restrict__ dst, int W, int H, int Krt,
                   int Kp, float eps, int tiles_x, int tiles_y, size_t phi_plane, size_t phi_row) {
    extern __shared__ float smem[];
    const int K = KT > 0 ? KT : Krt;
    const int c = (K - 1) / 2;
    const int SW = (KT > 0 ? KT : Krt) + BX - 1;   // staged tile width (= pitch)
    const int SH = TILE_H + Kp - 1;                // staged rows, incl. zero rows for the padded PSF rows
    float* sG = smem;                              // [K][Kp]  G transposed: sG[i * Kp + j]
    float* s = smem + K * Kp;                      // [SH][SW]

    int t = blockIdx.x;
    const int tile_x = t % tiles_x; t /= tiles_x;
    const int tile_y = t % tiles_y; t /= tiles_y;
    const size_t plane_off = (size_t)t * W * H;
    const int x0 = tile_x * BX, y0 = tile_y * TILE_H;
    const int tid = threadIdx.y * BX + threadIdx.x;

    for (int k = tid; k < K * Kp; k += BX * BY) sG[k] = G[k];

    {   // stage the tile with periodic wrap: s[ty][tx] = src(y0 - c + ty, x0 - c + tx)
        const float* sp = src + plane_off;
        const int lane = tid & 31, warp = tid >> 5;
        const int real_rows = TILE_H + K - 1;
        for (int tx = lane; tx < SW; tx += 32) {
            const int gx = pmod(x0 - c + tx, W);
            int gy = pmod(y0 - c + warp, H);
            for (int ty = warp; ty < SH; ty += (BX * BY) / 32) {
                s[ty * SW + tx] = ty < real_rows ? sp[(size_t)gy * W + gx] : 0.f;
                gy += (BX * BY) / 32;
                while (gy >= H) gy -= H;
            }
        }
    }
    __syncthreads();

    float acc[RY];
#pragma unroll
    for (int m = 0; m < RY; ++m) acc[m] = 0.f;

    const float* sbase = s + (threadIdx.y * RY) * SW + threadIdx.x;
    for (int i = 0; i < K; ++i) {
        const float* sg = sG + i * Kp;
        const float* scol = sbase + i;
        for (int jc = 0; jc < Kp; jc += JC) {
            float w[RY + JC - 1];
#pragma unroll
            for (int n = 0; n < RY + JC - 1; ++n) w[n] = scol[(jc + n) * SW];
            float g[JC];
#pragma unroll
            for (int jj = 0; jj < JC; ++jj) g[jj] = sg[jc + jj];
#pragma unroll
            for (int jj = 0; jj < JC; ++jj)
#pragma unroll
                for (int m = 0; m < RY; ++m) acc[m] = fmaf(g[jj], w[m + jj], acc[m]);
        }
    }

    const int x = x0 + threadIdx.x;
    if (x < W) {
#pragma unroll
        for (int m = 0; m < RY; ++m) {
            const int y = y0 + threadIdx.y * RY + m;
            if (y < H) {
                const size_t p = plane_off + (size_t)y * W + x;
                if (MODE == 0) dst[p] = (float)phi[(size_t)t * phi_plane + (size_t)y * phi_row + x] / fmaxf(acc[m], eps);   // a2
                else           dst[p] = dst[p] * acc[m];                      // a4
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// The same correlation on TWO planes at once.  The staged tile holds (plane a, plane b) as float2, a
// thread keeps RY float2 accumulators, and the inner product is FFMA2 (fma.rn.f32x2) with the tap as a
// broadcast scalar: one issue slot and one shared-memory load now feed two FMAs, which moves the kernel
// from issue-bound (ncu round 1: 80 % issue slots, 60 % FMA pipe) towards the FMA pipe's own limit.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ float2 ffma2_bcast(float g, float2 w, float2 c) {
    float2 r;
    asm("{ .reg .b64 ra, rb, rc, rd; mov.b64 ra, {%2,%2}; mov.b64 rb, {%3,%4}; mov.b64 rc, {%5,%6}; "
        "fma.rn.f32x2 rd, ra, rb, rc; mov.b64 {%0,%1}, rd; }"
        : "=f"(r.x), "=f"(r.y) : "f"(g), "f"(w.x), "f"(w.y), "f"(c.x), "f"(c.y));
    return r;
}

template <int KT, int JC, int MODE>
__global__ void __launch_bounds__(BX* BY)
direct_corr2_kernel(const float* __restrict__ src, const float* __restrict__ G,
                    const uint16_t* __restrict__ phi, float* __restrict__ dst, int W, int H, int Krt,
                    int Kp, float eps, int tiles_x, int tiles_y, size_t phi_plane, size_t phi_row,
                    int n_planes) {
    extern __shared__ __align__(16) float smem[];
    const int K = KT > 0 ? KT : Krt;
    const int c = (K - 1) / 2;
    const int SW = (KT > 0 ? KT : Krt) + BX - 1;   // staged tile width (= pitch)
    const int SH = TILE_H + Kp - 1;                // staged rows, incl. zero rows for the padded PSF rows
    float* sG = smem;                              // [K][Kp]  G transposed: sG[i * Kp + j]
    float2* s = reinterpret_cast<float2*>(smem + ((K * Kp + 1) & ~1));   // [SH][SW] (a, b)

    int t = blockIdx.x;
    const int tile_x = t % tiles_x; t /= tiles_x;
    const int tile_y = t % tiles_y; t /= tiles_y;   // t: pair index
    const int pa = 2 * t;
    const bool has_b = pa + 1 < n_planes;
    const size_t offa = (size_t)pa * W * H, offb = has_b ? offa + (size_t)W * H : offa;
    const int x0 = tile_x * BX, y0 = tile_y * TILE_H;
    const int tid = threadIdx.y * BX + threadIdx.x;

    for (int k = tid; k < K * Kp; k += BX * BY) sG[k] = G[k];

    {   // stage the tile with periodic wrap: s[ty][tx] = src(y0 - c + ty, x0 - c + tx) of both planes
        const float* spa = src + offa;
        const float* spb = src + offb;
        const int lane = tid & 31, warp = tid >> 5;
        const int real_rows = TILE_H + K - 1;
        for (int tx = lane; tx < SW; tx += 32) {
            const int gx = pmod(x0 - c + tx, W);
            int gy = pmod(y0 - c + warp, H);
            for (int ty = warp; ty < SH; ty += (BX * BY) / 32) {
                s[ty * SW + tx] = ty < real_rows ? make_float2(spa[(size_t)gy * W + gx], spb[(size_t)gy * W + gx])
                                                 : make_float2(0.f, 0.f);
                gy += (BX * BY) / 32;
                while (gy >= H) gy -= H;
            }
        }
    }
    __syncthreads();

    float2 acc[RY];
#pragma unroll
    for (int m = 0; m < RY; ++m) acc[m] = make_float2(0.f, 0.f);

    const float2* sbase = s + (threadIdx.y * RY) * SW + threadIdx.x;
    for (int i = 0; i < K; ++i) {
        const float* sg = sG + i * Kp;
        const float2* scol = sbase + i;
        for (int jc = 0; jc < Kp; jc += JC) {
            float2 w[RY + JC - 1];
#pragma unroll
            for (int n = 0; n < RY + JC - 1; ++n) w[n] = scol[(jc + n) * SW];
            float g[JC];
#pragma unroll
            for (int jj = 0; jj < JC; ++jj) g[jj] = sg[jc + jj];
#pragma unroll
            for (int jj = 0; jj < JC; ++jj)
#pragma unroll
                for (int m = 0; m < RY; ++m) acc[m] = ffma2_bcast(g[jj], w[m + jj], acc[m]);
        }
    }

    const int x = x0 + threadIdx.x;
    if (x < W) {
#pragma unroll
        for (int m = 0; m < RY; ++m) {
            const int y = y0 + threadIdx.y * RY + m;
            if (y < H) {
                const size_t q = (size_t)y * W + x;
                if (MODE == 0) {                                              // a2
                    const size_t f = (size_t)pa * phi_plane + (size_t)y * phi_row + x;
                    dst[offa + q] = (float)phi[f] / fmaxf(acc[m].x, eps);
                    if (has_b) dst[offb + q] = (float)phi[f + phi_plane] / fmaxf(acc[m].y, eps);
                } else {                                                      // a4
                    dst[offa + q] = dst[offa + q] * acc[m].x;
                    if (has_b) dst[offb + q] = dst[offb + q] * acc[m].y;
                }
            }
        }
    }
}

inline size_t pair_smem_bytes(int K, int Kp) {
    return sizeof(float) * (size_t)((K * Kp + 1) & ~1) + sizeof(float2) * (size_t)(TILE_H + Kp - 1) * (K + BX - 1);
}

template <int KT, int JC>
int launch_pair2(int mode, const float* src, const float* G, const uint16_t* phi, float* dst,
                 int W, int H, int K, int Kp, float eps, int n_planes, cudaStream_t st,
                 size_t phi_plane, size_t phi_row) {
    const int tiles_x = (W + BX - 1) / BX, tiles_y = (H + TILE_H - 1) / TILE_H;
    const size_t smem = pair_smem_bytes(K, Kp);
    const long long grid = (long long)((n_planes + 1) / 2) * tiles_x * tiles_y;
    if (grid > 0x7fffffffLL) return (int)cudaErrorInvalidConfiguration;
    dim3 block(BX, BY);
    cudaError_t e;
    // the opt-in to > 48 KB of dynamic shared memory is raised once per kernel and size (not per launch)
    static size_t opted[2] = {0, 0};
    if (mode == 0) {
        auto k = direct_corr2_kernel<KT, JC, 0>;
        if (smem > opted[0]) {
            e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return (int)e;
            opted[0] = smem;
        }
        k<<<(unsigned)grid, block, smem, st>>>(src, G, phi, dst, W, H, K, Kp, eps, tiles_x, tiles_y, phi_plane, phi_row, n_planes);
    } else {
        auto k = direct_corr2_kernel<KT, JC, 1>;
        if (smem > opted[1]) {
            e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return (int)e;
            opted[1] = smem;
        }
        k<<<(unsigned)grid, block, smem, st>>>(src, G, phi, dst, W, H, K, Kp, eps, tiles_x, tiles_y, phi_plane, phi_row, n_planes);
    }
    return (int)cudaGetLastError();
}

template <int KT, int JC>
int launch_pair_member(int mode, const float* src, const float* G, const uint16_t* phi, float* dst,
                       int W, int H, int K, int Kp, float eps, int n_planes, cudaStream_t st,
                       size_t phi_plane, size_t phi_row) {
    const int tiles_x = (W + BX - 1) / BX, tiles_y = (H + TILE_H - 1) / TILE_H;
    const size_t smem = sizeof(float) * ((size_t)K * Kp + (size_t)(TILE_H + Kp - 1) * (K + BX - 1));
    const long long grid = (long long)n_planes * tiles_x * tiles_y;
    if (grid > 0x7fffffffLL) return (int)cudaErrorInvalidConfiguration;
    dim3 block(BX, BY);
    cudaError_t e;
    static size_t opted[2] = {0, 0};
    if (mode == 0) {
        auto k = direct_corr_kernel<KT, JC, 0>;
        if (smem > opted[0]) {
            e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return (int)e;
            opted[0] = smem;
        }
        k<<<(unsigned)grid, block, smem, st>>>(src, G, phi, dst, W, H, K, Kp, eps, tiles_x, tiles_y, phi_plane, phi_row);
    } else {
        auto k = direct_corr_kernel<KT, JC, 1>;
        if (smem > opted[1]) {
            e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return (int)e;
            opted[1] = smem;
        }
        k<<<(unsigned)grid, block, smem, st>>>(src, G, phi, dst, W, H, K, Kp, eps, tiles_x, tiles_y, phi_plane, phi_row);
    }
    return (int)cudaGetLastError();
}

int launch_corr(int mode, const mvd_handle* h, const float* src, const float* G, const uint16_t* phi,
                float* dst, int n_planes, cudaStream_t st, size_t phi_plane, size_t phi_row) {
    // two planes per thread whenever the float2 tile fits in shared memory; K as a template
    // parameter for the config sizes
    if (h->direct_pair) {
#define MVD_DIRECT_CASE(KT_, JC_)                                                                 \
    if (h->K == (KT_) && h->JC == (JC_))                                                          \
        return launch_pair2<KT_, JC_>(mode, src, G, phi, dst, h->W, h->H, h->K, h->Kp,             \
                                      h->eps, n_planes, st, phi_plane, phi_row);
        MVD_DIRECT_CASE(9, 9)
        MVD_DIRECT_CASE(21, 7)
        MVD_DIRECT_CASE(31, 8)
        MVD_DIRECT_CASE(41, 7)
        MVD_DIRECT_CASE(51, 17)
#undef MVD_DIRECT_CASE
        if (h->JC == 8)
            return launch_pair2<0, 8>(mode, src, G, phi, dst, h->W, h->H, h->K, h->Kp, h->eps, n_planes, st,
                                      phi_plane, phi_row);
    }
    return launch_pair_member<0, 8>(mode, src, G, phi, dst, h->W, h->H, h->K, h->Kp, h->eps,
                                    n_planes, st, phi_plane, phi_row);
}

}  // namespace

// Row chunk JC and padded row count Kp of the kernel that serves psf_size K.
int direct_choose_chunk(int K, int* JC, int* Kp) {
    int jc;
    switch (K) {
        case 9: jc = 9; break;      // row chunks sized for the two-plane kernel's register budget
        case 21: jc = 7; break;
        case 31: jc = 8; break;
        case 41: jc = 7; break;
        case 51: jc = 17; break;
        default: jc = 8; break;
    }
    *JC = jc;
    *Kp = ((K + jc - 1) / jc) * jc;
    return MVD_OK;
}

// Upload both coefficient arrays per view, transposed and zero-padded: G[v][which][i][j], j < Kp.
// host_xs (nullable): explicit back-projectors X_v, [V][KX][KX].  Step a3 is then the convolution with
// X_v, i.e. the correlation this kernel computes with the FLIPPED X_v.  Both kernels are laid, centred,
// into arrays of Kd = max(K, KX) taps (zero outside their support); h->K becomes Kd for this engine.
int direct_setup(mvd_handle* h, const float* host_psfs, const float* host_xs) {
    const int K0 = h->K, KX = host_xs ? h->KX : h->K;
    const int Kd = K0 > KX ? K0 : KX;
    std::vector<float> pad_p((size_t)h->V * Kd * Kd, 0.f), pad_b((size_t)h->V * Kd * Kd, 0.f);
    for (int v = 0; v < h->V; ++v) {
        const int op = (Kd - K0) / 2, ox = (Kd - KX) / 2;
        for (int j = 0; j < K0; ++j)
            for (int i = 0; i < K0; ++i) {
                const float p = host_psfs[((size_t)v * K0 + j) * K0 + i];
                pad_p[((size_t)v * Kd + j + op) * Kd + i + op] = p;
                if (!host_xs) pad_b[((size_t)v * Kd + j + op) * Kd + i + op] = p;   // a3 correlates with P_v
            }
        if (host_xs)
            for (int j = 0; j < KX; ++j)
                for (int i = 0; i < KX; ++i)   // correlation with flip(X_v) == convolution with X_v
                    pad_b[((size_t)v * Kd + (Kd - 1 - (j + ox))) * Kd + (Kd - 1 - (i + ox))] =
                        host_xs[((size_t)v * KX + j) * KX + i];
    }
    h->K = Kd;
    host_psfs = pad_p.data();
    const float* host_back = pad_b.data();
    direct_choose_chunk(h->K, &h->JC, &h->Kp);
    // two planes per thread whenever the float2 tile fits; the single-plane kernel works in row chunks of 8
    h->direct_pair = pair_smem_bytes(h->K, h->Kp) <= 227u * 1024u;
    if (!h->direct_pair) {
        h->JC = 8;
        h->Kp = (h->K + 7) / 8 * 8;
    }
    const int K = h->K, Kp = h->Kp;
    const size_t per = (size_t)K * Kp;
    // shared memory needed by one CTA must fit the 227 KB limit
    const size_t smem = sizeof(float) * (per + (size_t)(TILE_H + Kp - 1) * (K + BX - 1));
    if (smem > 227u * 1024u) return MVD_ERR_UNSUPPORTED;
    std::vector<float> g((size_t)h->V * 2 * per, 0.f);
    for (int v = 0; v < h->V; ++v) {
        const float* P = host_psfs + (size_t)v * K * K;
        const float* B = host_back + (size_t)v * K * K;
        float* blur = g.data() + ((size_t)v * 2 + 0) * per;
        float* back = g.data() + ((size_t)v * 2 + 1) * per;
        for (int j = 0; j < K; ++j)
            for (int i = 0; i < K; ++i) {
                blur[(size_t)i * Kp + j] = P[(size_t)(K - 1 - j) * K + (K - 1 - i)];   // a1: flipped
                back[(size_t)i * Kp + j] = B[(size_t)j * K + i];                       // a3: as given
            }
    }
    MVD_TRY(h, cudaMalloc((void**)&h->d_coef, g.size() * sizeof(float)));
    MVD_TRY(h, cudaMemcpy(h->d_coef, g.data(), g.size() * sizeof(float), cudaMemcpyHostToDevice));
    return MVD_OK;
}

size_t direct_scratch_bytes(const mvd_handle* h, int n_planes) {
    return sizeof(float) * (size_t)n_planes * h->W * h->H;
}

int direct_run(mvd_handle* h, Workspace& ws, const uint16_t* views, ViewLayout lay, float* out,
               int n_planes, cudaStream_t stream) {
    const size_t npx = (size_t)h->W * h->H;
    const size_t n = npx * n_planes;
    {
        LaunchScope ls(h, KC_INIT_MEAN, stream);
        const int threads = 256;
        const size_t want = (n + threads - 1) / threads;
        const unsigned grid = (unsigned)(want < (size_t)h->n_sm * 16 ? want : (size_t)h->n_sm * 16);
        init_mean_kernel<<<grid, threads, 0, stream>>>(views, lay, h->V, h->W, h->H, out, n);
    }
    MVD_TRY(h, cudaGetLastError());
    if (h->T == 0) return MVD_OK;
    int rc = ws_reserve(h, ws, direct_scratch_bytes(h, n_planes), 0);
    if (rc != MVD_OK) return rc;
    float* r = ws.a;
    const size_t per = (size_t)h->K * h->Kp;
    for (int t = 0; t < h->T; ++t)
        for (int v = 0; v < h->V; ++v) {
            const float* Gblur = h->d_coef + ((size_t)v * 2 + 0) * per;
            const float* Gback = h->d_coef + ((size_t)v * 2 + 1) * per;
            const uint16_t* phi = views + (size_t)v * lay.view;
            int e;
            {
                LaunchScope ls(h, KC_DIRECT_BLUR_RATIO, stream);
                e = launch_corr(0, h, out, Gblur, phi, r, n_planes, stream, lay.plane, lay.row);
            }
            MVD_TRY(h, (cudaError_t)e);
            {
                LaunchScope ls(h, KC_DIRECT_BACK_UPDATE, stream);
                e = launch_corr(1, h, r, Gback, nullptr, out, n_planes, stream, 0, 0);
            }
            MVD_TRY(h, (cudaError_t)e);
        }
    return MVD_OK;
}
