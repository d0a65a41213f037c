// mvd_fft.cu -- host side of the FFT engine: supported lengths, twiddle tables, optical transfer
// functions, and the launch sequence of one chunk of planes (see mvd_fft_kernels.cuh for the kernels).
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "mvd_fft_kernels.cuh"
#include "mvd_internal.cuh"

using mvdfft::PlanInfo;
using mvdfft::RowArgs;
using mvdfft::SizeOps;

namespace {

// The two generations lay the spectrum out differently (v2: tile-major), so a plane uses v2 kernels
// only when BOTH of its lengths have them.
const SizeOps* find_ops_v1(int N) {
    if (const SizeOps* o = mvd_fft_ops_small(N)) return o;
    if (const SizeOps* o = mvd_fft_ops_mid(N)) return o;
    if (const SizeOps* o = mvd_fft_ops_more_a(N)) return o;
    if (const SizeOps* o = mvd_fft_ops_more_b(N)) return o;
    return mvd_fft_ops_large(N);
}
bool use_v2(int W, int H) {
    const SizeOps* r = mvd_fft_ops_v2(W);
    const SizeOps* c = mvd_fft_ops_v2(H);
    return r && c && r->rows && c->cols;
}
const SizeOps* find_row_ops(int W, int H) { return use_v2(W, H) ? mvd_fft_ops_v2(W) : find_ops_v1(W); }
const SizeOps* find_col_ops(int W, int H) { return use_v2(W, H) ? mvd_fft_ops_v2(H) : find_ops_v1(H); }

// Per-thread twiddles of a plan, [(s-1) E + e][TPF], s >= 1:
//   element e of thread t in stage s belongs to butterfly j = t + u TPF, input m  (e = u + m E/R),
//   and is multiplied by exp(-2 pi i m k / (Ns R)),  k = j mod Ns  (inverse transforms conjugate it).
std::vector<float2> make_twiddles(int N, const PlanInfo& p) {
    std::vector<float2> tw((size_t)std::max(p.S - 1, 0) * p.E * p.TPF);
    int Ns = p.radices[0];
    for (int s = 1; s < p.S; ++s) {
        const int R = p.radices[s], NB = p.E / R;
        for (int e = 0; e < p.E; ++e) {
            const int u = e % NB, m = e / NB;
            for (int t = 0; t < p.TPF; ++t) {
                const int j = t + u * p.TPF, k = j % Ns;
                const double ang = -2.0 * M_PI * (double)((long long)m * k) / (double)((long long)Ns * R);
                tw[((size_t)(s - 1) * p.E + e) * p.TPF + t] = make_float2((float)cos(ang), (float)sin(ang));
            }
        }
        Ns *= R;
    }
    (void)N;
    return tw;
}

// OTF, phase 1: G[j][kx] = sum_i P[j][i] exp(-2 pi i kx (i - c) / W)        (fp64)
__global__ void otf_rows_kernel(const float* __restrict__ P, int K, int W, double2* __restrict__ G) {
    const int kx = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (kx >= W) return;
    const int c = (K - 1) / 2;
    double re = 0.0, im = 0.0;
    for (int i = 0; i < K; ++i) {
        long long ph = ((long long)kx * (i - c)) % W;
        if (ph < 0) ph += W;
        double s, co;
        sincospi(-2.0 * (double)ph / (double)W, &s, &co);
        const double p = (double)P[j * K + i];
        re += p * co;
        im += p * s;
    }
    G[(size_t)j * W + kx] = make_double2(re, im);
}

// OTF, phase 2: O[ky][kx] = (1 / (W H)) sum_j G[j][kx] exp(-2 pi i ky (j - c) / H)   -> fp32
__global__ void otf_cols_kernel(const double2* __restrict__ G, int K, int W, int H, float2* __restrict__ O,
                                int tile_major, float* __restrict__ Oreal) {
    const int kx = blockIdx.x * blockDim.x + threadIdx.x, ky = blockIdx.y;
    if (kx >= W) return;
    const int c = (K - 1) / 2;
    double re = 0.0, im = 0.0;
    for (int j = 0; j < K; ++j) {
        long long ph = ((long long)ky * (j - c)) % H;
        if (ph < 0) ph += H;
        double s, co;
        sincospi(-2.0 * (double)ph / (double)H, &s, &co);
        const double2 g = G[(size_t)j * W + kx];
        re += g.x * co - g.y * s;
        im += g.x * s + g.y * co;
    }
    const double sc = 1.0 / ((double)W * (double)H);
    const size_t idx = tile_major ? ((size_t)(kx >> 4) * H + ky) * 16 + (kx & 15) : (size_t)ky * W + kx;
    if (Oreal) Oreal[idx] = (float)(re * sc);     // centro-symmetric PSF: the imaginary part is round-off only
    else O[idx] = make_float2((float)(re * sc), (float)(im * sc));
}

// Product-form runs are not repaired (the repair kernel implements the sequential update): the flagged plane pairs are
// only counted, so that mvd_guard_flagged tells the caller which stacks to rerun on the direct engine.
__global__ void guard_count_kernel(const unsigned* __restrict__ flags, int pairs, unsigned* __restrict__ total) {
    unsigned n = 0;
    for (int p = threadIdx.x; p < pairs; p += blockDim.x) n += flags[p] ? 1u : 0u;
    n = __reduce_add_sync(0xffffffffu, n);
    if ((threadIdx.x & 31) == 0 && n) atomicAdd(total, n);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct FftState {
    const SizeOps* row = nullptr;   // length W
    const SizeOps* col = nullptr;   // length H
    float2* tw_row = nullptr;
    float2* tw_col = nullptr;
    EncodeTiledFn encode = nullptr; // cuTensorMapEncodeTiled, resolved through the runtime (no -lcuda)
    // generation-2 column kernels without OTF registers fetch their OTF slice by TMA: one map per view
    std::vector<CUtensorMap> otf_maps, otf_b_maps;
};

// Tensor map of the spectrum buffer S = float [pairs * H][2 W] with a box of one column tile:
// 2 TC floats (TC complex columns) by box_h rows.
int make_col_tensor_map(mvd_handle* h, const FftState* st, float2* S, int pairs, CUtensorMap* map) {
    const bool v2 = st->col->generation == 2;
    // v1: S = float [pairs * H][2 W], box = one column tile;  v2 (tile-major S): float [pairs * W/16 * H][32]
    // (128-byte rows), box = one team's four columns (8 floats) by up to 256 tile rows
    const cuuint64_t dims[2] = {v2 ? (cuuint64_t)32 : (cuuint64_t)2 * h->W,
                                v2 ? (cuuint64_t)pairs * (h->W / 16) * h->H : (cuuint64_t)pairs * h->H};
    const cuuint64_t strides[1] = {v2 ? (cuuint64_t)128 : (cuuint64_t)h->W * sizeof(float2)};
    const cuuint32_t box[2] = {v2 ? (cuuint32_t)st->col->col_box_w : (cuuint32_t)(2 * st->col->col_tc), (cuuint32_t)st->col->col_box_h};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = st->encode(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, S, dims, strides, box, estr,
                                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                  CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        h->last_cuda = (int)cudaErrorInvalidValue;
        return MVD_ERR_CUDA;
    }
    return MVD_OK;
}

// Tensor map of one view's tile-major OTF, float [(W/16) * H][32], same box as the spectrum's map.
int make_otf_tensor_map(mvd_handle* h, const FftState* st, const float2* otf, CUtensorMap* map) {
    const cuuint64_t dims[2] = {32, (cuuint64_t)(h->W / 16) * h->H};
    const cuuint64_t strides[1] = {128};
    const cuuint32_t box[2] = {(cuuint32_t)st->col->col_box_w, (cuuint32_t)st->col->col_box_h};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = st->encode(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void*)otf, dims, strides, box, estr,
                                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                  CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        h->last_cuda = (int)cudaErrorInvalidValue;
        return MVD_ERR_CUDA;
    }
    return MVD_OK;
}

// Tensor map of one view's REAL tile-major OTF, float [(W/16) * H][16]: half the box width of the complex one.
int make_otf_real_tensor_map(mvd_handle* h, const FftState* st, const float* otf, CUtensorMap* map) {
    const cuuint64_t dims[2] = {16, (cuuint64_t)(h->W / 16) * h->H};
    const cuuint64_t strides[1] = {64};
    const cuuint32_t box[2] = {(cuuint32_t)st->col->col_box_w / 2, (cuuint32_t)st->col->col_box_h};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = st->encode(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void*)otf, dims, strides, box, estr,
                                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                  CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        h->last_cuda = (int)cudaErrorInvalidValue;
        return MVD_ERR_CUDA;
    }
    return MVD_OK;
}

FftState* state_of(const mvd_handle* h) { return static_cast<FftState*>(h->fft); }

}  // namespace

int fft_supported(int W, int H) {
    const SizeOps* r = find_row_ops(W, H);
    const SizeOps* c = find_col_ops(W, H);
    if (!r || !c) return 0;
    if (W % c->col_tc != 0) return 0;
    const size_t limit = 227u * 1024u;   // dynamic shared memory per CTA on sm_100
    if (r->row_smem > limit || c->col_smem > limit) return 0;
    return 1;
}

// 0: not supported, 1: generation-1 kernels, 2: generation-2 (team) kernels
int fft_generation(int W, int H) { return !fft_supported(W, H) ? 0 : use_v2(W, H) ? 2 : 1; }

int fft_pad_dims(int w_min, int h_min, int* Wp, int* Hp) {
    std::vector<int> lens;
    for (int n = 32; n <= 2048; ++n)
        if (find_ops_v1(n) || mvd_fft_ops_v2(n)) lens.push_back(n);
    // cost = padded area x the measured relative cost per voxel: generation-2 shapes 1 (2048-point columns 1.25: one team
    // per SM), shapes only the generation-1 kernels take 3.5 (30-42 against 110-150 GVoxel/s, profiles/r2_experiments.md)
    double best = 0.0;
    for (int w : lens) {
        if (w < w_min) continue;
        for (int hh : lens) {
            if (hh < h_min || !fft_supported(w, hh)) continue;
            const double cost = (double)w * hh * (use_v2(w, hh) ? (hh == 2048 || hh == 1536 ? 1.25 : 1.0) : 3.5);
            if (best == 0.0 || cost < best) { best = cost; *Wp = w; *Hp = hh; }
        }
    }
    return best > 0.0 ? 1 : 0;
}

void fft_teardown(mvd_handle* h) {
    FftState* st = state_of(h);
    if (!st) return;
    if (st->tw_row) cudaFree(st->tw_row);
    if (st->tw_col) cudaFree(st->tw_col);
    delete st;
    h->fft = nullptr;
}

int fft_setup(mvd_handle* h, const float* host_psfs, const float* host_xs) {
    if (!fft_supported(h->W, h->H)) return MVD_ERR_UNSUPPORTED;
    FftState st;
    st.row = find_row_ops(h->W, h->H);
    st.col = find_col_ops(h->W, h->H);
    MVD_TRY(h, st.row->prepare_rows());
    MVD_TRY(h, st.col->prepare_cols());
    {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        MVD_TRY(h, cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q));
        if (!fn || q != cudaDriverEntryPointSuccess) {
            h->last_cuda = (int)cudaErrorNotSupported;
            return MVD_ERR_CUDA;
        }
        st.encode = (EncodeTiledFn)fn;
    }

    auto upload = [&](const std::vector<float2>& v, float2** d) -> int {
        const size_t bytes = std::max<size_t>(v.size(), 1) * sizeof(float2);
        MVD_TRY(h, cudaMalloc((void**)d, bytes));
        if (!v.empty()) MVD_TRY(h, cudaMemcpy(*d, v.data(), v.size() * sizeof(float2), cudaMemcpyHostToDevice));
        return MVD_OK;
    };
    int rc = upload(make_twiddles(h->W, st.row->row), &st.tw_row);
    if (rc == MVD_OK) {
        if (st.col->col_tw_custom) {   // two-stage plan with unequal thread counts: [RA][RB], exp(-2 pi i t k / H) at [k][t]
            const int RA = st.col->col.radices[0], RB = st.col->col.radices[1];
            std::vector<float2> tw((size_t)RA * RB);
            for (int k = 0; k < RA; ++k)
                for (int t = 0; t < RB; ++t) {
                    const double ang = -2.0 * M_PI * (double)(k * t) / (double)h->H;
                    tw[(size_t)k * RB + t] = make_float2((float)cos(ang), (float)sin(ang));
                }
            rc = upload(tw, &st.tw_col);
        } else {
            rc = upload(make_twiddles(h->H, st.col->col), &st.tw_col);
        }
    }
    if (rc != MVD_OK) {
        if (st.tw_row) cudaFree(st.tw_row);
        if (st.tw_col) cudaFree(st.tw_col);
        return rc;
    }
    h->fft = new FftState(st);

    // optical transfer functions: O_v = FFT2(P_v) / (W H) for a1 and, when the caller supplied explicit
    // back-projectors X_v, B_v = FFT2(X_v) / (W H) for a3 (otherwise a3 uses conj O_v)
    const int W = h->W, H = h->H;
    const size_t npx = (size_t)W * H;
    const bool tile_major = st.row->generation == 2;
    // Real transfer functions: every PSF centro-symmetric (P[j][i] == P[K-1-j][K-1-i]) and a3 = correlation with P_v
    // (no explicit back-projector): O_v is real, a1 and a3 use the same array, stored as float (4 B per element
    // through the column kernels instead of 8, one packed multiply instead of a complex one).
    bool real_otf = st.col->col_real_otf && !host_xs;
    for (int v = 0; v < h->V && real_otf; ++v)
        for (int j = 0; j < h->K && real_otf; ++j)
            for (int i = 0; i < h->K; ++i)
                if (host_psfs[((size_t)v * h->K + j) * h->K + i] != host_psfs[((size_t)v * h->K + (h->K - 1 - j)) * h->K + (h->K - 1 - i)]) {
                    real_otf = false;
                    break;
                }
    auto build_otfs = [&](const float* host_k, int K, float2** dst) -> int {
        float* d_k = nullptr;
        double2* d_G = nullptr;
        if (real_otf) MVD_TRY(h, cudaMalloc((void**)&h->d_otf_real, sizeof(float) * npx * h->V));
        else MVD_TRY(h, cudaMalloc((void**)dst, sizeof(float2) * npx * h->V));
        MVD_TRY(h, cudaMalloc((void**)&d_k, sizeof(float) * (size_t)h->V * K * K));
        int r = mvd_check(h, cudaMalloc((void**)&d_G, sizeof(double2) * (size_t)K * W));
        if (r == MVD_OK)
            r = mvd_check(h, cudaMemcpy(d_k, host_k, sizeof(float) * (size_t)h->V * K * K, cudaMemcpyHostToDevice));
        for (int v = 0; v < h->V && r == MVD_OK; ++v) {
            const dim3 block(128), g1((W + 127) / 128, K), g2((W + 127) / 128, H);
            {
                LaunchScope ls(h, KC_SETUP, 0);
                otf_rows_kernel<<<g1, block>>>(d_k + (size_t)v * K * K, K, W, d_G);
            }
            {
                LaunchScope ls(h, KC_SETUP, 0);
                otf_cols_kernel<<<g2, block>>>(d_G, K, W, H, real_otf ? nullptr : *dst + (size_t)v * npx, tile_major,
                                               real_otf ? h->d_otf_real + (size_t)v * npx : nullptr);
            }
            r = mvd_check(h, cudaGetLastError());
        }
        if (r == MVD_OK) r = mvd_check(h, cudaDeviceSynchronize());
        if (d_k) cudaFree(d_k);
        if (d_G) cudaFree(d_G);
        return r;
    };
    rc = build_otfs(host_psfs, h->K, &h->d_otf);
    if (rc == MVD_OK && host_xs) rc = build_otfs(host_xs, h->KX, &h->d_otf_b);
    if (rc == MVD_OK && st.col->generation == 2 && st.col->col_box_h > 0 && !st.col->col_otf_regs) {
        FftState* fs = state_of(h);
        fs->otf_maps.resize(h->V);
        for (int v = 0; v < h->V && rc == MVD_OK; ++v)
            rc = real_otf ? make_otf_real_tensor_map(h, fs, h->d_otf_real + (size_t)v * npx, &fs->otf_maps[v])
                          : make_otf_tensor_map(h, fs, h->d_otf + (size_t)v * npx, &fs->otf_maps[v]);
        if (h->d_otf_b) {
            fs->otf_b_maps.resize(h->V);
            for (int v = 0; v < h->V && rc == MVD_OK; ++v)
                rc = make_otf_tensor_map(h, fs, h->d_otf_b + (size_t)v * npx, &fs->otf_b_maps[v]);
        }
    }
    // guard: the direct engine's coefficient arrays for the repair pass (PSFs too large for its two-plane kernel
    // leave the FFT engine without one: direct_repair_available), and the counter behind mvd_guard_flagged
    if (rc == MVD_OK) {
        const int rd = direct_setup(h, host_psfs, host_xs);
        if (rd != MVD_OK && rd != MVD_ERR_UNSUPPORTED) rc = rd;
        h->guard_rel = 1.0f / 8192.0f;
    }
    if (rc == MVD_OK) rc = mvd_check(h, cudaMalloc((void**)&h->d_guard_total, sizeof(unsigned)));
    if (rc == MVD_OK) rc = mvd_check(h, cudaMemset(h->d_guard_total, 0, sizeof(unsigned)));
    h->launches = 0;
    return rc;
}

// Guard words of a chunk of n planes: [pairs] max bits, [pairs] flags, [1] barrier of the repair kernel.
size_t fft_guard_bytes(int n_planes) { return sizeof(unsigned) * (2 * (size_t)((n_planes + 1) / 2) + 1); }

// Planes per internal pass: bound the two scratch buffers (8 B per voxel) to about 1 GiB.
int fft_default_chunk(const mvd_handle* h) {
    const size_t npx = (size_t)h->W * h->H;
    size_t c = ((size_t)1 << 30) / (npx * 8);
    c = std::max<size_t>(2, std::min<size_t>(c, 1024));   // <= 512 pairs: the repair kernel's list
    return (int)(c & ~(size_t)1);
}

int fft_run(mvd_handle* h, Workspace& ws, const PlaneIO& io, int n_planes, cudaStream_t stream) {
    const uint16_t* views = io.views;
    const ViewLayout lay = io.lay;
    FftState* st = state_of(h);
    if (!st) return MVD_ERR_INVALID;
    const int W = h->W, H = h->H;
    const int pairs = (n_planes + 1) / 2;
    const size_t bytes = sizeof(float2) * (size_t)pairs * H * W;
    if (io.weights && (((uintptr_t)io.weights & 15u) != 0 || (W & 3) != 0)) return MVD_ERR_INVALID;
    // the bulk copies of the row kernels need 16-byte aligned rows
    if (((uintptr_t)views & 15u) != 0 || ((lay.view * sizeof(uint16_t)) & 15u) != 0 ||
        ((lay.plane * sizeof(uint16_t)) & 15u) != 0 || ((lay.row * sizeof(uint16_t)) & 15u) != 0)
        return MVD_ERR_INVALID;
    int rc = ws_reserve(h, ws, bytes, bytes, fft_guard_bytes(n_planes));
    if (rc != MVD_OK) return rc;
    // Product form (PAPER.md:79 as printed; mvd_set_update_mode): every view's blur starts from psi^t's row spectrum,
    // saved in S0 and copied back into S before views 1 .. V-1, and the factors are multiplied into A = a copy of psi^t
    // (the update pass runs with its Z pointer on A), which the last view turns into psi^{t+1} -- together with its row
    // spectrum in S, exactly what the next iteration starts from.  Then Z and A swap roles.
    const bool product = h->update_mode == MVD_UPDATE_PRODUCT && h->T > 0;
    if (product && (rc = ws_reserve_product(h, ws, bytes, h->V > 1 ? bytes : 0)) != MVD_OK) return rc;
    if (pairs > 512) return MVD_ERR_INVALID;   // chunks are bounded by fft_default_chunk / mvd_set_chunk_planes
    MVD_TRY(h, cudaMemsetAsync(ws.g, 0, fft_guard_bytes(n_planes), stream));
    CUtensorMap tmap;
    memset(&tmap, 0, sizeof(tmap));
    if (st->col->col_box_h > 0) {
        rc = make_col_tensor_map(h, st, (float2*)ws.b, pairs, &tmap);
        if (rc != MVD_OK) return rc;
    }

    RowArgs a;
    a.Z = (float2*)ws.a;
    a.S = (float2*)ws.b;
    a.views = views;
    a.view_stride = lay.view;
    a.view_plane = lay.plane;
    a.view_row = lay.row;
    a.out = io.out;
    a.out16 = io.out16;
    a.weights = io.weights;
    a.w_view = io.w_view;
    a.n_planes = n_planes;
    a.H = H;
    a.V = h->V;
    a.v = 0;
    a.eps = h->eps;
    a.final = 0;
    a.total_rows = pairs * H;
    a.gmax = ws.g;
    a.gflag = ws.g + pairs;
    a.guard_rel = h->guard_rel;

    const int rp = st->row->row_threads / st->row->row.TPF;          // rows per CTA pass
    const int row_ctas = (a.total_rows + rp - 1) / rp;
    // v1: many short-lived CTAs; v2: persistent, two CTAs per SM
    const int row_grid = std::max(1, std::min(row_ctas, h->n_sm * (st->row->generation == 2 ? st->row->row_cps : 16)));
    const int row_grid_w = st->row->generation == 2 && st->row->row_cps_w > 0
                               ? std::max(1, std::min(row_ctas, h->n_sm * st->row->row_cps_w)) : row_grid;
    const int tiles = W / st->col->col_tc;
    dim3 col_grid;
    if (st->col->generation == 2) {
        // persistent 1D grid over (tile, pair) items, never more CTAs than fit at once (a second
        // wave would double the pass); a multiple of the tile count when CTAs keep OTF registers
        const long long items = (long long)tiles * pairs;
        long long g = (long long)h->n_sm * st->col->col_cps;
        if (st->col->col_otf_regs) g = std::max<long long>(tiles, g / tiles * tiles);
        col_grid = dim3((unsigned)std::max<long long>(1, std::min(g, items)));
    } else {
        const int per_tile = std::max(1, (h->n_sm * 8 + tiles - 1) / tiles);
        col_grid = dim3(tiles, std::min(pairs, per_tile));
    }
    const size_t npx = (size_t)W * H;

    {
        LaunchScope ls(h, KC_FFT_ROWS_FIRST, stream);
        a.final = h->T == 0;
        rc = mvd_check(h, st->row->rows(mvdfft::ROWS_FIRST, a, st->tw_row, row_grid, stream));
    }
    if (rc != MVD_OK) return rc;
    float2* Zcur = (float2*)ws.a;       // psi^t
    float2* Acc = (float2*)ws.c;        // product form: psi^t times the factors so far
    for (int t = 0; t < h->T; ++t) {
        if (product) {
            MVD_TRY(h, cudaMemcpyAsync(Acc, Zcur, bytes, cudaMemcpyDeviceToDevice, stream));
            if (h->V > 1) MVD_TRY(h, cudaMemcpyAsync(ws.d, ws.b, bytes, cudaMemcpyDeviceToDevice, stream));
        }
        for (int v = 0; v < h->V; ++v) {
            const bool real_otf = h->d_otf_real != nullptr;       // mode 2 of the column kernels; a1 and a3 alike
            const float2* otf = real_otf ? reinterpret_cast<const float2*>(h->d_otf_real + (size_t)v * npx) : h->d_otf + (size_t)v * npx;
            if (product && v > 0) MVD_TRY(h, cudaMemcpyAsync(ws.b, ws.d, bytes, cudaMemcpyDeviceToDevice, stream));
            a.Z = product ? Acc : Zcur;
            {
                LaunchScope ls(h, KC_FFT_COLS, stream);
                rc = mvd_check(h, st->col->cols(tmap, st->otf_maps.empty() ? tmap : st->otf_maps[v], a.S, otf, real_otf ? 2 : 0, pairs, W,
                                                st->tw_col, col_grid, stream));   // a1
            }
            if (rc != MVD_OK) return rc;
            {
                LaunchScope ls(h, KC_FFT_ROWS_RATIO, stream);
                a.v = v;
                a.final = 0;
                rc = mvd_check(h, st->row->rows(mvdfft::ROWS_RATIO, a, st->tw_row, row_grid, stream));   // a2
            }
            if (rc != MVD_OK) return rc;
            {
                LaunchScope ls(h, KC_FFT_COLS, stream);
                rc = h->d_otf_b      // a3: explicit back-projector B_v, or conj O_v (X = P_v^*)
                         ? mvd_check(h, st->col->cols(tmap, st->otf_b_maps.empty() ? tmap : st->otf_b_maps[v], a.S,
                                                      h->d_otf_b + (size_t)v * npx, 0, pairs, W, st->tw_col, col_grid, stream))
                         : mvd_check(h, st->col->cols(tmap, st->otf_maps.empty() ? tmap : st->otf_maps[v], a.S, otf, real_otf ? 2 : 1, pairs, W,
                                                      st->tw_col, col_grid, stream));
            }
            if (rc != MVD_OK) return rc;
            {
                LaunchScope ls(h, KC_FFT_ROWS_UPDATE, stream);
                a.final = (t == h->T - 1 && v == h->V - 1);
                rc = io.weights   // a4w: the weighted kernel keeps twice the landing zone, so fewer CTAs are resident
                         ? mvd_check(h, st->row->rows(mvdfft::ROWS_UPDATE_W, a, st->tw_row, row_grid_w, stream))
                         : mvd_check(h, st->row->rows(mvdfft::ROWS_UPDATE, a, st->tw_row, row_grid, stream));  // a4
            }
            if (rc != MVD_OK) return rc;
        }
        if (product) std::swap(Zcur, Acc);
    }
    if (product) {
        // the repair pass runs the product form too (psi^t and the estimate being built in two buffers): Z and the
        // product-form scratch are free by now.  Plans without a repair kernel only count the flagged pairs.
        if (direct_repair_available(h))
            return direct_repair_launch(h, io, io.out ? io.out : ws.b, ws.a, ws.g + pairs, ws.g + 2 * pairs, n_planes, stream, ws.c);
        LaunchScope ls(h, KC_GUARD_REPAIR, stream);
        guard_count_kernel<<<1, 256, 0, stream>>>(ws.g + pairs, pairs, h->d_guard_total);
        return mvd_check(h, cudaGetLastError());
    }
    // guard: pairs flagged by the ratio passes are recomputed with the direct engine's arithmetic (one empty
    // cooperative launch when nothing is flagged); Z is free by now and serves as its ratio scratch
    // (with uint16 output psi is iterated in S, which is free as well)
    if (h->T > 0 && direct_repair_available(h))
        return direct_repair_launch(h, io, io.out ? io.out : ws.b, ws.a, ws.g + pairs, ws.g + 2 * pairs, n_planes, stream);
    return MVD_OK;
}
