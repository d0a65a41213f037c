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
#include <algorithm>

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
                   int Kp, float eps, int tiles_x, int tiles_y, size_t phi_plane, size_t phi_row,
                   const float* __restrict__ wgt) {
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
                else {                                                        // a4 / a4w
                    float q = acc[m];
                    if (wgt) { const float w0 = __ldg(wgt + p); q = fmaf(w0, q, 1.f - w0); }
                    dst[p] = dst[p] * q;
                }
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

// One 64 x 64 output tile (tile_x, tile_y) of the plane pair (pa, pa + 1): stage, correlate, epilogue.
// `stage_G`: copy the coefficient array into shared memory first (false when the caller already did).
// CG: read src and the read-modify-write of dst through L2 only (ld.global.cg) -- the persistent repair kernel
// reads what other SMs wrote earlier in the SAME launch, which a stale L1 line must not serve.
// MODE 1 extras: wgt (nullable) = weights of this view, same layout as dst (a4w: q <- w q + 1 - w, reading W1).
template <int KT, int JC, int MODE, bool CG = false>
__device__ __forceinline__ void corr2_tile(float* smem, const float* __restrict__ src, const float* __restrict__ G,
                                           const uint16_t* __restrict__ phi, float* __restrict__ dst, int W, int H,
                                           int Krt, int Kp, float eps, int tile_x, int tile_y, int pa, bool has_b,
                                           size_t phi_plane, size_t phi_row, bool stage_G,
                                           const float* __restrict__ wgt = nullptr) {
    const int K = KT > 0 ? KT : Krt;
    const int c = (K - 1) / 2;
    const int SW = (KT > 0 ? KT : Krt) + BX - 1;   // staged tile width (= pitch)
    const int SH = TILE_H + Kp - 1;                // staged rows, incl. zero rows for the padded PSF rows
    float* sG = smem;                              // [K][Kp]  G transposed: sG[i * Kp + j]
    float2* s = reinterpret_cast<float2*>(smem + ((K * Kp + 1) & ~1));   // [SH][SW] (a, b)

    const size_t offa = (size_t)pa * W * H, offb = has_b ? offa + (size_t)W * H : offa;
    const int x0 = tile_x * BX, y0 = tile_y * TILE_H;
    const int tid = threadIdx.y * BX + threadIdx.x;

    if (stage_G)
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
                const size_t g = (size_t)gy * W + gx;
                s[ty * SW + tx] = ty >= real_rows ? make_float2(0.f, 0.f)
                                  : CG ? make_float2(__ldcg(spa + g), __ldcg(spb + g)) : make_float2(spa[g], spb[g]);
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
                    float qa = acc[m].x, qb = acc[m].y;
                    if (wgt) {                                                // a4w
                        const float w0 = __ldg(wgt + offa + q), w1 = has_b ? __ldg(wgt + offb + q) : 0.f;
                        qa = fmaf(w0, qa, 1.f - w0);
                        qb = fmaf(w1, qb, 1.f - w1);
                    }
                    dst[offa + q] = (CG ? __ldcg(dst + offa + q) : dst[offa + q]) * qa;
                    if (has_b) dst[offb + q] = (CG ? __ldcg(dst + offb + q) : dst[offb + q]) * qb;
                }
            }
        }
    }
}

template <int KT, int JC, int MODE>
__global__ void __launch_bounds__(BX* BY)
direct_corr2_kernel(const float* __restrict__ src, const float* __restrict__ G,
                    const uint16_t* __restrict__ phi, float* __restrict__ dst, int W, int H, int Krt,
                    int Kp, float eps, int tiles_x, int tiles_y, size_t phi_plane, size_t phi_row,
                    int n_planes, const float* __restrict__ wgt) {
    extern __shared__ __align__(16) float smem[];
    int t = blockIdx.x;
    const int tile_x = t % tiles_x; t /= tiles_x;
    const int tile_y = t % tiles_y; t /= tiles_y;   // t: pair index
    corr2_tile<KT, JC, MODE>(smem, src, G, phi, dst, W, H, Krt, Kp, eps, tile_x, tile_y, 2 * t,
                             2 * t + 1 < n_planes, phi_plane, phi_row, true, wgt);
}

// ---------------------------------------------------------------------------------------------
// Guard of the FFT engine: the plane pairs that the FFT engine flagged as
// ill-conditioned for fp32 transforms (a pixel with phi_v > 0 whose blur fell below the engine's noise
// threshold: step a2 then divides by round-off) are recomputed here from scratch, a0..a5, with the direct
// engine's arithmetic.  ONE persistent cooperative launch per chunk: every CTA reads the flags, returns at
// once when none is set (the normal case: one empty launch), and otherwise all CTAs share the tiles of the
// flagged pairs with a grid-wide barrier after every pass (the halo dependency between a2 and a3, and
// between a4 and the next a1).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint16_t to_u16(float x) { return (uint16_t)__float2uint_rn(fminf(x, 65535.f)); }

__device__ __forceinline__ void grid_barrier(unsigned* counter, unsigned target) {
    __syncthreads();
    if (threadIdx.x == 0 && threadIdx.y == 0) {
        __threadfence();
        atomicAdd(counter, 1u);
        while (*(volatile unsigned*)counter < target) {}
        __threadfence();
    }
    __syncthreads();
}

struct RepairArgs {
    const uint16_t* views;      // view 0 of plane 0 of the chunk
    ViewLayout lay;
    float* out;                 // [n_planes][H][W]: psi, iterated in place
    float* r;                   // ratio scratch, [n_planes][H][W] (the FFT engine's Z buffer, free by now)
    const float* coef;          // [V][2][K][Kp]
    const unsigned* flags;      // [pairs]
    unsigned* barrier;          // zeroed before the launch
    unsigned* total;            // per-handle count of pairs ever handed over (mvd_guard_flagged)
    const float* weights;       // nullptr or [V][n][H][W] (a4w)
    size_t w_view;
    uint16_t* out16;            // nullptr, or the uint16 output that receives the repaired planes (out is then scratch)
    float* acc;                 // nullptr: sequential update; else product form (PAPER.md:79 as printed): scratch like out, in
                                // which psi^t times the factors so far is built while kernel A keeps reading psi^t
    int n_planes, W, H, K, Kp, V, T;
    float eps;
};

template <int KT, int JC>
__global__ void __launch_bounds__(BX* BY) direct_repair_kernel(RepairArgs a) {
    extern __shared__ __align__(16) float smem[];
    __shared__ int s_list[512];
    __shared__ int s_n;
    const int pairs = (a.n_planes + 1) / 2;
    const int tid = threadIdx.y * BX + threadIdx.x;
    if (tid == 0) {
        int n = 0;
        for (int p = 0; p < pairs; ++p)
            if (a.flags[p]) {
                if (n < 512) s_list[n] = p;
                ++n;
            }
        s_n = n;
    }
    __syncthreads();
    const int nf = s_n < 512 ? s_n : 512;   // more than 512 flagged pairs per chunk cannot happen (chunks hold <= 512 pairs)
    if (nf == 0) return;
    if (blockIdx.x == 0 && tid == 0) atomicAdd(a.total, (unsigned)nf);

    const size_t npx = (size_t)a.W * a.H;
    const int tiles_x = (a.W + BX - 1) / BX, tiles_y = (a.H + TILE_H - 1) / TILE_H;
    const int tiles = tiles_x * tiles_y;
    unsigned epoch = 0;

    // a0 on the flagged pairs
    for (int k = 0; k < nf; ++k) {
        const int pa = 2 * s_list[k];
        const int np = pa + 1 < a.n_planes ? 2 : 1;
        for (size_t q = (size_t)blockIdx.x * (BX * BY) + tid; q < np * npx; q += (size_t)gridDim.x * (BX * BY)) {
            const size_t pl = q / npx, rem = q % npx;
            const size_t src = (pa + pl) * a.lay.plane + (rem / a.W) * a.lay.row + rem % a.W;
            float s = 0.f;
            for (int v = 0; v < a.V; ++v) s += (float)a.views[(size_t)v * a.lay.view + src];
            a.out[(size_t)(pa + pl) * npx + rem] = s / (float)a.V;
        }
    }
    grid_barrier(a.barrier, ++epoch * gridDim.x);

    // dst <- src on the flagged pairs (every CTA takes a share; the caller puts a grid barrier behind it)
    auto copy_flagged = [&](float* dst, const float* src) {
        for (int k = 0; k < nf; ++k) {
            const int pa = 2 * s_list[k];
            const int np = pa + 1 < a.n_planes ? 2 : 1;
            for (size_t q = (size_t)blockIdx.x * (BX * BY) + tid; q < np * npx; q += (size_t)gridDim.x * (BX * BY))
                dst[(size_t)pa * npx + q] = __ldcg(src + (size_t)pa * npx + q);
        }
    };
    const size_t per = (size_t)a.K * a.Kp;
    float* psi = a.out;     // psi^t
    float* acc = a.acc;     // product form: the estimate being built (the two swap roles after every iteration)
    for (int t = 0; t < a.T; ++t) {
        if (acc) {
            copy_flagged(acc, psi);
            grid_barrier(a.barrier, ++epoch * gridDim.x);
        }
        for (int v = 0; v < a.V; ++v) {
            const float* Gblur = a.coef + ((size_t)v * 2 + 0) * per;
            const float* Gback = a.coef + ((size_t)v * 2 + 1) * per;
            const uint16_t* phi = a.views + (size_t)v * a.lay.view;
            for (int w = blockIdx.x; w < nf * tiles; w += gridDim.x) {
                const int pa = 2 * s_list[w / tiles], tl = w % tiles;
                __syncthreads();   // the previous tile's shared memory is no longer read
                corr2_tile<KT, JC, 0, true>(smem, psi, Gblur, phi, a.r, a.W, a.H, a.K, a.Kp, a.eps, tl % tiles_x,
                                      tl / tiles_x, pa, pa + 1 < a.n_planes, a.lay.plane, a.lay.row, true);
            }
            grid_barrier(a.barrier, ++epoch * gridDim.x);
            for (int w = blockIdx.x; w < nf * tiles; w += gridDim.x) {
                const int pa = 2 * s_list[w / tiles], tl = w % tiles;
                __syncthreads();
                corr2_tile<KT, JC, 1, true>(smem, a.r, Gback, nullptr, acc ? acc : psi, a.W, a.H, a.K, a.Kp, a.eps, tl % tiles_x,
                                      tl / tiles_x, pa, pa + 1 < a.n_planes, 0, 0, true,
                                      a.weights ? a.weights + (size_t)v * a.w_view : nullptr);
            }
            grid_barrier(a.barrier, ++epoch * gridDim.x);
        }
        if (acc) {
            float* tmp = psi; psi = acc; acc = tmp;
        }
    }
    if (psi != a.out) {     // product form, odd iteration count: the result sits in the scratch
        copy_flagged(a.out, psi);
        grid_barrier(a.barrier, ++epoch * gridDim.x);
    }
    if (a.out16)
        for (int k = 0; k < nf; ++k) {
            const int pa = 2 * s_list[k];
            const int np = pa + 1 < a.n_planes ? 2 : 1;
            for (size_t q = (size_t)blockIdx.x * (BX * BY) + tid; q < np * npx; q += (size_t)gridDim.x * (BX * BY))
                a.out16[(size_t)pa * npx + q] = to_u16(__ldcg(a.out + (size_t)pa * npx + q));
        }
}

// ---------------------------------------------------------------------------------------------
// Planes that fit on chip: the WHOLE RL run (a0, T x V view updates, final store) of a plane pair in one CTA
// and one launch.  psi and r of the pair live in shared memory (4 fp32 planes), every pass stages its wrapped
// tile from there and runs the same register-blocked FFMA2 correlation as above, so the result is the direct
// engine's bit for bit; HBM sees the uint16 views and the final psi only ((2 V + 4) B per voxel per step instead
// of 22 B per voxel-view-iteration), and the 2 V T + 1 launches of the tiled kernels -- which bound small stacks
// such as config 1 (81 launches of ~4 us on 32 768 voxels) -- become one.
// ---------------------------------------------------------------------------------------------
struct SmallArgs {
    const uint16_t* views;
    ViewLayout lay;
    float* out;
    const float* coef;          // [V][2][K][Kp]
    int n_planes, W, H, K, Kp, V, T;
    float eps;
    int tile_floats;            // floats of the staging area (coefficients + wrapped float2 tile)
    const float* weights;       // nullptr or [V][n][H][W] (a4w)
    size_t w_view;
    uint16_t* out16;            // set instead of out for uint16 output
};

template <int KT, int JC>
__global__ void __launch_bounds__(BX* BY) direct_small_kernel(SmallArgs a) {
    extern __shared__ __align__(16) float smem[];
    const size_t npx = (size_t)a.W * a.H;
    float* psi = smem + a.tile_floats;          // [2][H][W]
    float* r = psi + 2 * npx;                   // [2][H][W]
    const int tid = threadIdx.y * BX + threadIdx.x;
    const int pairs = (a.n_planes + 1) / 2;
    const int tiles_x = (a.W + BX - 1) / BX, tiles_y = (a.H + TILE_H - 1) / TILE_H;
    const size_t per = (size_t)a.K * a.Kp;
    for (int pair = blockIdx.x; pair < pairs; pair += gridDim.x) {
        const int pa = 2 * pair;
        const bool has_b = pa + 1 < a.n_planes;
        const uint16_t* v0 = a.views + (size_t)pa * a.lay.plane;
        for (size_t q = tid; q < (has_b ? 2 : 1) * npx; q += BX * BY) {      // a0
            const size_t pl = q / npx, rem = q % npx;
            const size_t src = pl * a.lay.plane + (rem / a.W) * a.lay.row + rem % a.W;
            float s = 0.f;
            for (int v = 0; v < a.V; ++v) s += (float)v0[(size_t)v * a.lay.view + src];
            psi[q] = s / (float)a.V;
        }
        __syncthreads();
        for (int t = 0; t < a.T; ++t)
            for (int v = 0; v < a.V; ++v) {
                const float* Gblur = a.coef + ((size_t)v * 2 + 0) * per;
                const float* Gback = a.coef + ((size_t)v * 2 + 1) * per;
                const uint16_t* phi = v0 + (size_t)v * a.lay.view;
                for (int tl = 0; tl < tiles_x * tiles_y; ++tl) {
                    if (tl) __syncthreads();      // the staging area is no longer read
                    corr2_tile<KT, JC, 0>(smem, psi, Gblur, phi, r, a.W, a.H, a.K, a.Kp, a.eps, tl % tiles_x,
                                          tl / tiles_x, 0, has_b, a.lay.plane, a.lay.row, true);
                }
                __syncthreads();
                for (int tl = 0; tl < tiles_x * tiles_y; ++tl) {
                    if (tl) __syncthreads();
                    corr2_tile<KT, JC, 1>(smem, r, Gback, nullptr, psi, a.W, a.H, a.K, a.Kp, a.eps, tl % tiles_x,
                                          tl / tiles_x, 0, has_b, 0, 0, true,
                                          a.weights ? a.weights + (size_t)v * a.w_view + (size_t)pa * npx : nullptr);
                }
                __syncthreads();
            }
        for (size_t q = tid; q < (has_b ? 2 : 1) * npx; q += BX * BY) {
            if (a.out16) a.out16[(size_t)pa * npx + q] = to_u16(psi[q]);
            else a.out[(size_t)pa * npx + q] = psi[q];
        }
        __syncthreads();
    }
}

inline size_t pair_smem_bytes(int K, int Kp) {
    return sizeof(float) * (size_t)((K * Kp + 1) & ~1) + sizeof(float2) * (size_t)(TILE_H + Kp - 1) * (K + BX - 1);
}

template <int KT, int JC>
int launch_pair2(int mode, const float* src, const float* G, const uint16_t* phi, float* dst,
                 int W, int H, int K, int Kp, float eps, int n_planes, cudaStream_t st,
                 size_t phi_plane, size_t phi_row, const float* wgt) {
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
        k<<<(unsigned)grid, block, smem, st>>>(src, G, phi, dst, W, H, K, Kp, eps, tiles_x, tiles_y, phi_plane, phi_row, n_planes, wgt);
    } else {
        auto k = direct_corr2_kernel<KT, JC, 1>;
        if (smem > opted[1]) {
            e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return (int)e;
            opted[1] = smem;
        }
        k<<<(unsigned)grid, block, smem, st>>>(src, G, phi, dst, W, H, K, Kp, eps, tiles_x, tiles_y, phi_plane, phi_row, n_planes, wgt);
    }
    return (int)cudaGetLastError();
}

template <int KT, int JC>
int launch_pair_member(int mode, const float* src, const float* G, const uint16_t* phi, float* dst,
                       int W, int H, int K, int Kp, float eps, int n_planes, cudaStream_t st,
                       size_t phi_plane, size_t phi_row, const float* wgt) {
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
        k<<<(unsigned)grid, block, smem, st>>>(src, G, phi, dst, W, H, K, Kp, eps, tiles_x, tiles_y, phi_plane, phi_row, wgt);
    } else {
        auto k = direct_corr_kernel<KT, JC, 1>;
        if (smem > opted[1]) {
            e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return (int)e;
            opted[1] = smem;
        }
        k<<<(unsigned)grid, block, smem, st>>>(src, G, phi, dst, W, H, K, Kp, eps, tiles_x, tiles_y, phi_plane, phi_row, wgt);
    }
    return (int)cudaGetLastError();
}

int launch_corr(int mode, const mvd_handle* h, const float* src, const float* G, const uint16_t* phi,
                float* dst, int n_planes, cudaStream_t st, size_t phi_plane, size_t phi_row, const float* wgt) {
    // two planes per thread whenever the float2 tile fits in shared memory; K as a template
    // parameter for the config sizes
    if (h->direct_pair) {
#define MVD_DIRECT_CASE(KT_, JC_)                                                                 \
    if (h->dK == (KT_) && h->JC == (JC_))                                                         \
        return launch_pair2<KT_, JC_>(mode, src, G, phi, dst, h->W, h->H, h->dK, h->Kp,            \
                                      h->eps, n_planes, st, phi_plane, phi_row, wgt);
        MVD_DIRECT_CASE(9, 9)
        MVD_DIRECT_CASE(21, 7)
        MVD_DIRECT_CASE(31, 8)
        MVD_DIRECT_CASE(41, 7)
        MVD_DIRECT_CASE(51, 17)
#undef MVD_DIRECT_CASE
        if (h->JC == 8)
            return launch_pair2<0, 8>(mode, src, G, phi, dst, h->W, h->H, h->dK, h->Kp, h->eps, n_planes, st,
                                      phi_plane, phi_row, wgt);
    }
    return launch_pair_member<0, 8>(mode, src, G, phi, dst, h->W, h->H, h->dK, h->Kp, h->eps,
                                    n_planes, st, phi_plane, phi_row, wgt);
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
// into arrays of Kd = max(K, KX) taps (zero outside their support): h->dK taps.
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
    h->dK = Kd;
    host_psfs = pad_p.data();
    const float* host_back = pad_b.data();
    direct_choose_chunk(h->dK, &h->JC, &h->Kp);
    // two planes per thread whenever the float2 tile fits; the single-plane kernel works in row chunks of 8
    h->direct_pair = pair_smem_bytes(h->dK, h->Kp) <= 227u * 1024u;
    if (!h->direct_pair) {
        h->JC = 8;
        h->Kp = (h->dK + 7) / 8 * 8;
    }
    const int K = h->dK, Kp = h->Kp;
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

namespace {
size_t small_smem_bytes(const mvd_handle* h) {
    return pair_smem_bytes(h->dK, h->Kp) + sizeof(float) * 4 * (size_t)h->W * h->H;
}

template <int KT, int JC>
int launch_small(const mvd_handle* h, SmallArgs& a, cudaStream_t st) {
    const size_t smem = small_smem_bytes(h);
    static size_t opted = 0;
    auto k = direct_small_kernel<KT, JC>;
    if (smem > opted) {
        cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return (int)e;
        opted = smem;
    }
    const int pairs = (a.n_planes + 1) / 2;
    const int per_sm = (int)std::max<size_t>(1, (size_t)(228 * 1024) / (smem + 1024));
    const int grid = std::min(pairs, h->n_sm * per_sm);
    k<<<grid, dim3(BX, BY), smem, st>>>(a);
    return (int)cudaGetLastError();
}
}  // namespace

// The on-chip path serves a plan when psi, r (4 fp32 planes of the pair) and the staging tile fit one CTA.
bool direct_small_available(const mvd_handle* h) {
    return h->direct_pair && small_smem_bytes(h) <= 227u * 1024u;
}
static int direct_run_small(mvd_handle* h, const PlaneIO& io, int n_planes, cudaStream_t stream) {
    SmallArgs a;
    a.views = io.views; a.lay = io.lay; a.out = io.out; a.coef = h->d_coef;
    a.weights = io.weights; a.w_view = io.w_view; a.out16 = io.out16;
    a.n_planes = n_planes; a.W = h->W; a.H = h->H; a.K = h->dK; a.Kp = h->Kp; a.V = h->V; a.T = h->T; a.eps = h->eps;
    a.tile_floats = (int)(pair_smem_bytes(h->dK, h->Kp) / sizeof(float));
    int e;
    LaunchScope ls(h, KC_SMALL_RESIDENT, stream);
    if (h->dK == 9 && h->JC == 9) e = launch_small<9, 9>(h, a, stream);
    else if (h->dK == 21 && h->JC == 7) e = launch_small<21, 7>(h, a, stream);
    else if (h->dK == 31 && h->JC == 8) e = launch_small<31, 8>(h, a, stream);
    else e = launch_small<0, 8>(h, a, stream);
    return mvd_check(h, (cudaError_t)e);
}

size_t direct_scratch_bytes(const mvd_handle* h, int n_planes) {
    return sizeof(float) * (size_t)n_planes * h->W * h->H;
}

__global__ void convert_u16_kernel(const float* __restrict__ psi, uint16_t* __restrict__ out, size_t n) {
    for (size_t p = blockIdx.x * (size_t)blockDim.x + threadIdx.x; p < n; p += (size_t)gridDim.x * blockDim.x)
        out[p] = to_u16(psi[p]);
}

int direct_run(mvd_handle* h, Workspace& ws, const PlaneIO& io, int n_planes, cudaStream_t stream) {
    const size_t npx = (size_t)h->W * h->H;
    const size_t n = npx * n_planes;
    const bool product = h->update_mode == MVD_UPDATE_PRODUCT && h->T > 0;
    if (h->T > 0 && !product && direct_small_available(h)) return direct_run_small(h, io, n_planes, stream);
    // psi is iterated in place in the fp32 output; a uint16 output gets an fp32 scratch and one conversion pass
    int rc = ws_reserve(h, ws, h->T > 0 ? direct_scratch_bytes(h, n_planes) : 0, io.out16 ? sizeof(float) * n : 0);
    if (rc != MVD_OK) return rc;
    // Product form (PAPER.md:79 as printed): kernel A reads psi^t for every view, kernel B multiplies the factors into a
    // copy of it, which becomes psi^{t+1} after the last view; the two buffers then swap roles.
    if (product && (rc = ws_reserve_product(h, ws, sizeof(float) * n, 0)) != MVD_OK) return rc;
    float* psi = io.out16 ? ws.b : io.out;
    float* const result = psi;
    float* acc = ws.c;
    const unsigned egrid = (unsigned)std::min<size_t>((n + 255) / 256, (size_t)h->n_sm * 16);
    {
        LaunchScope ls(h, KC_INIT_MEAN, stream);
        init_mean_kernel<<<egrid, 256, 0, stream>>>(io.views, io.lay, h->V, h->W, h->H, psi, n);
    }
    MVD_TRY(h, cudaGetLastError());
    float* r = ws.a;
    const size_t per = (size_t)h->dK * h->Kp;
    for (int t = 0; t < h->T; ++t) {
        if (product) MVD_TRY(h, cudaMemcpyAsync(acc, psi, sizeof(float) * n, cudaMemcpyDeviceToDevice, stream));
        float* const upd = product ? acc : psi;     // what kernel B multiplies the factor into
        for (int v = 0; v < h->V; ++v) {
            const float* Gblur = h->d_coef + ((size_t)v * 2 + 0) * per;
            const float* Gback = h->d_coef + ((size_t)v * 2 + 1) * per;
            const uint16_t* phi = io.views + (size_t)v * io.lay.view;
            int e;
            const float* wv = io.weights ? io.weights + (size_t)v * io.w_view : nullptr;
            {
                LaunchScope ls(h, h->sep ? KC_SEP_BLUR_RATIO : KC_DIRECT_BLUR_RATIO, stream);
                e = h->sep ? sep_launch(0, h, v, psi, phi, r, n_planes, stream, io.lay.plane, io.lay.row, nullptr)
                           : launch_corr(0, h, psi, Gblur, phi, r, n_planes, stream, io.lay.plane, io.lay.row, nullptr);
            }
            MVD_TRY(h, (cudaError_t)e);
            {
                LaunchScope ls(h, h->sep ? KC_SEP_BACK_UPDATE : KC_DIRECT_BACK_UPDATE, stream);
                e = h->sep ? sep_launch(1, h, v, r, nullptr, upd, n_planes, stream, 0, 0, wv)
                           : launch_corr(1, h, r, Gback, nullptr, upd, n_planes, stream, 0, 0, wv);
            }
            MVD_TRY(h, (cudaError_t)e);
        }
        if (product) std::swap(psi, acc);
    }
    if (psi != result) MVD_TRY(h, cudaMemcpyAsync(result, psi, sizeof(float) * n, cudaMemcpyDeviceToDevice, stream));
    psi = result;
    if (io.out16) {
        LaunchScope ls(h, KC_INIT_MEAN, stream);
        convert_u16_kernel<<<egrid, 256, 0, stream>>>(psi, io.out16, n);
        MVD_TRY(h, cudaGetLastError());
    }
    return MVD_OK;
}

// ---------------------------------------------------------------------------------------------
// guard repair (called by the FFT engine after a chunk's last pass)
// ---------------------------------------------------------------------------------------------
namespace {
template <int KT, int JC>
int launch_repair(const mvd_handle* h, RepairArgs& a, cudaStream_t st) {
    const size_t smem = pair_smem_bytes(a.K, a.Kp);
    static size_t opted = 0;
    auto k = direct_repair_kernel<KT, JC>;
    if (smem > opted) {
        cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return (int)e;
        opted = smem;
    }
    void* args[] = {&a};
    // cooperative: all CTAs are resident at once, so the grid-wide barrier cannot deadlock
    return (int)cudaLaunchCooperativeKernel((void*)k, dim3(h->n_sm), dim3(BX, BY), args, smem, st);
}
}  // namespace

bool direct_repair_available(const mvd_handle* h) { return h->d_coef != nullptr && h->direct_pair; }

int direct_repair_launch(mvd_handle* h, const PlaneIO& io, float* psi, float* r_scratch,
                         const unsigned* flags, unsigned* barrier, int n_planes, cudaStream_t stream, float* acc) {
    RepairArgs a;
    a.acc = acc;
    a.views = io.views; a.lay = io.lay; a.out = psi; a.r = r_scratch; a.coef = h->d_coef; a.flags = flags;
    a.barrier = barrier; a.total = h->d_guard_total;
    a.weights = io.weights; a.w_view = io.w_view; a.out16 = io.out16;
    a.n_planes = n_planes; a.W = h->W; a.H = h->H; a.K = h->dK; a.Kp = h->Kp; a.V = h->V; a.T = h->T; a.eps = h->eps;
    int e;
    LaunchScope ls(h, KC_GUARD_REPAIR, stream);
    if (h->dK == 9 && h->JC == 9) e = launch_repair<9, 9>(h, a, stream);
    else if (h->dK == 21 && h->JC == 7) e = launch_repair<21, 7>(h, a, stream);
    else if (h->dK == 31 && h->JC == 8) e = launch_repair<31, 8>(h, a, stream);
    else if (h->dK == 41 && h->JC == 7) e = launch_repair<41, 7>(h, a, stream);
    else if (h->dK == 51 && h->JC == 17) e = launch_repair<51, 17>(h, a, stream);
    else e = launch_repair<0, 8>(h, a, stream);
    return mvd_check(h, (cudaError_t)e);
}

// ---------------------------------------------------------------------------------------------
// mvd_deconvolve_planes_noalloc -- the direct engine's tiled kernels with their ratio scratch r in a file-scope
// device array instead of the handle's cudaMalloc'ed workspace, for callers that cannot allocate (code under CUDA
// graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Nothing here calls cudaMalloc, cudaFree or
// an allocating library routine; every GPU that loads libmvd.so holds the array (16 MiB) until exit.
//
// The array's name is a host-side stand-in in host code, NOT a device address: the kernels get the pointer that
// cudaGetSymbolAddress returns, resolved once per device with that device current (first call of the entry point on
// that device -- make it outside stream capture).  Every call shares the array and it keeps the last call's
// contents: nothing has to start at zero (kernel A overwrites every element kernel B reads), but two calls that
// overlap on the GPU (different streams, no ordering between them) race on it.
// ---------------------------------------------------------------------------------------------
static __device__ __align__(256) float g_noalloc_r[MVD_NOALLOC_MAX_VOXELS];

namespace {
constexpr int kMaxDevices = 64;
float* g_noalloc_ptr[kMaxDevices] = {};       // per device: the array's device address
}  // namespace

int mvd_deconvolve_planes_noalloc(mvd_handle* h, const uint16_t* dev_views_u16, float* dev_out_f32, int n_planes,
                                  void* stream) {
    if (!h || !dev_views_u16 || !dev_out_f32 || n_planes < 0) return MVD_ERR_INVALID;
    if (n_planes == 0) return MVD_OK;
    if (h->path != MVD_PATH_DIRECT || h->padded || h->update_mode != MVD_UPDATE_SEQUENTIAL || !h->d_coef)
        return MVD_ERR_UNSUPPORTED;
    const size_t npx = (size_t)h->W * h->H;
    const size_t n = npx * (size_t)n_planes;
    if (n > (size_t)MVD_NOALLOC_MAX_VOXELS) return MVD_ERR_TOO_LARGE;
    cudaStream_t st = (cudaStream_t)stream;

    int dev = -1;
    MVD_TRY(h, cudaGetDevice(&dev));
    if (dev != h->device || dev < 0 || dev >= kMaxDevices) return MVD_ERR_INVALID;   // the handle's device must be current
    if (!g_noalloc_ptr[dev]) {
        float* p = nullptr;
        MVD_TRY(h, cudaGetSymbolAddress((void**)&p, g_noalloc_r));
        if (!p) return MVD_ERR_CUDA;
        g_noalloc_ptr[dev] = p;
    }
    float* r = g_noalloc_ptr[dev];
    float* psi = dev_out_f32;                       // iterated in place in the caller's output

    const ViewLayout lay{(size_t)n_planes * npx, npx, (size_t)h->W};
    const unsigned egrid = (unsigned)std::min<size_t>((n + 255) / 256, (size_t)h->n_sm * 16);
    init_mean_kernel<<<egrid, 256, 0, st>>>(dev_views_u16, lay, h->V, h->W, h->H, psi, n);   // a0
    h->launches++;
    MVD_TRY(h, cudaGetLastError());
    const size_t per = (size_t)h->dK * h->Kp;
    for (int t = 0; t < h->T; ++t)
        for (int v = 0; v < h->V; ++v) {
            const float* Gblur = h->d_coef + ((size_t)v * 2 + 0) * per;
            const float* Gback = h->d_coef + ((size_t)v * 2 + 1) * per;
            const uint16_t* phi = dev_views_u16 + (size_t)v * lay.view;
            int e = launch_corr(0, h, psi, Gblur, phi, r, n_planes, st, lay.plane, lay.row, nullptr);    // a1 + a2 -> r
            h->launches++;
            MVD_TRY(h, (cudaError_t)e);
            e = launch_corr(1, h, r, Gback, nullptr, psi, n_planes, st, 0, 0, nullptr);                  // a3 + a4
            h->launches++;
            MVD_TRY(h, (cudaError_t)e);
        }
    return MVD_OK;
}
