// mvd_internal.cuh -- shared declarations of libmvd's translation units (not part of the C ABI).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/mvd.h"

// Kernel classes for mvd_profile_read / bench.py's roofline line.
enum KernelClass {
    KC_INIT_MEAN = 0,        // a0: psi_0 = mean of the views (direct path)
    KC_DIRECT_BLUR_RATIO,    // a1+a2: b = psi (*) P_v, r = phi_v / max(b, eps)
    KC_DIRECT_BACK_UPDATE,   // a3+a4: q = r (*) P_v^*, psi *= q
    KC_FFT_ROWS_FIRST,       // a0 + forward row FFT of psi_0
    KC_FFT_COLS,             // column FFT . OTF . inverse column FFT (a1 / a3 middle part)
    KC_FFT_ROWS_RATIO,       // inverse row FFT -> b, a2 ratio, forward row FFT of r
    KC_FFT_ROWS_UPDATE,      // inverse row FFT -> q, a4 update, forward row FFT of the new psi
    KC_SETUP,                // mvd_create-time kernels (OTF construction)
    KC_GUARD_REPAIR,         // FFT engine's guard: flagged plane pairs recomputed with the direct engine's arithmetic
    KC_SMALL_RESIDENT,       // whole RL run of a small plane pair on chip, one launch
    KC_SEP_BLUR_RATIO,       // a1+a2 with a separable PSF: x pass, z pass, ratio
    KC_SEP_BACK_UPDATE       // a3+a4 with a separable PSF
};
static_assert(KC_SEP_BACK_UPDATE + 1 == MVD_N_KERNEL_CLASSES, "kernel class table and mvd.h disagree");

// One captured launch sequence (CUDA graph) and what it was captured for.  An entry is valid while the handle's
// graph_epoch is unchanged: every reallocation of scratch or slots and every setting that changes the launch sequence
// bumps the epoch.
struct GraphEntry {
    uint64_t key[8];
    uint64_t epoch;
    cudaGraphExec_t exec;
    long long launches;     // kernels in the graph (for mvd_launch_count)
    uint64_t last_use;
};

struct ProfRecord {
    int kc;
    cudaEvent_t e0, e1;
};

// Per-stream working memory.  Grown on demand, freed in mvd_destroy.
struct Workspace {
    float* a = nullptr;      // direct: r [chunk][H][W];   fft: Z (psi pairs, float2 [pairs][H][W])
    float* b = nullptr;      // direct: unused;            fft: S (spectrum, float2 [pairs][H][W])
    size_t a_bytes = 0, b_bytes = 0;
    unsigned* g = nullptr;   // fft: guard words of the chunk in flight: [pairs] max bits of psi_0, [pairs] flags, [1] barrier
    size_t g_bytes = 0;
    // padded plans (mvd_create_padded): the chunk's views embedded in zero planes of the engine's size, uint16
    // [V][n][H][W] (the padding is written once, when the buffer is allocated), and the engine's output [n][H][W]
    uint16_t* pin = nullptr;
    float* pout = nullptr;
    size_t pin_bytes = 0, pout_bytes = 0;
    float* pw = nullptr;     // ... and the chunk's per-view weights embedded the same way (zero in the padding), fp32 [V][n][H][W]
    size_t pw_bytes = 0;
    // product-form update (mvd_set_update_mode): the estimate being built (psi^t times the factors so far) and, on the
    // FFT engine, the row spectrum of psi^t that every view's blur starts from
    float* c = nullptr;
    float* d = nullptr;
    size_t c_bytes = 0, d_bytes = 0;
};

struct mvd_handle {
    int W = 0, H = 0, V = 0, K = 0, T = 0;   // W x H: the planes the engine works on
    // the caller's planes: uW x uH = W x H, or smaller for a padded plan: the caller's planes sit in the
    // corner of zero-filled W x H planes, W >= uW + K - 1 and H >= uH + K - 1, and the result is cropped
    int uW = 0, uH = 0;
    bool padded = false;
    float eps = 0.f;
    int path = MVD_PATH_DIRECT;
    int device = 0;
    int n_sm = 148;

    // direct path: per view two coefficient arrays, transposed and row-padded: G[v][which][K][Kp]
    // which = 0: blur (flipped PSF), 1: back-projection (PSF as given)
    float* d_coef = nullptr;
    int dK = 0;   // taps per axis of the direct engine's coefficient arrays: max(K, KX)
    int Kp = 0;   // padded number of PSF rows (multiple of the kernel's row chunk)
    int JC = 0;   // row chunk of the direct kernel chosen for K
    bool direct_pair = false;   // the two-plane FFMA2 kernel serves this plan (its float2 tile fits in shared memory)
    // separable fast path of the direct engine (mvd_sep.cu): every P_v is an outer product u_v w_v^T
    bool sep = false;
    float* d_sep = nullptr;     // [V][2 (a1, a3)][2 (z taps, x taps)][sepKp]
    int sepKp = 0;

    // fft path: optical transfer functions, float2 [V][H][W], pre-scaled by 1/(W*H)
    float2* d_otf = nullptr;
    float2* d_otf_b = nullptr;   // explicit back-projectors' transfer functions (nullptr: a3 uses conj d_otf)
    float* d_otf_real = nullptr; // real transfer functions (centro-symmetric PSFs on generation-2 column kernels): replaces d_otf
    int KX = 0;                  // size of the caller's back-projectors (0: Independent variant, X = P_v^*)
    void* fft = nullptr;   // FftState (mvd_fft.cu)
    // fft path, guard: plane pairs with a pixel phi_v > 0 whose blur is below guard_rel x max(psi_0)
    // are recomputed by direct_repair_launch; d_guard_total counts them over the handle's life
    float guard_rel = 0.f;
    unsigned* d_guard_total = nullptr;

    Workspace ws_main;
    // host pipeline (mvd_deconvolve_host): three slots, one stream each
    static constexpr int kSlots = 4;
    // slots (= streams) the host pipeline cycles through, 3 .. kSlots.  Algorithm 1 has three; with two batches computing at
    // a time a stream spends ~40 % of its cycle in its own copies, so three streams keep only ~1.9 batches computing.  A
    // fourth slot restores two (config 2: streamed / resident 0.845 -> 0.883; the other configs unchanged).
    int pipeline_slots = 4;
    cudaStream_t streams[kSlots] = {nullptr, nullptr, nullptr};
    Workspace ws_slot[kSlots];
    uint16_t* d_in[kSlots] = {nullptr, nullptr, nullptr};
    float* d_w[kSlots] = {nullptr, nullptr, nullptr};      // weights of the batch, allocated at the first weighted call
    size_t slot_w_planes = 0;
    float* d_out[kSlots] = {nullptr, nullptr, nullptr};
    size_t slot_planes = 0;

    // device-resident calls: planes are dealt in batches to this many internal streams, forked from and
    // joined to the caller's stream, so that one batch's kernel tails overlap the next batch's kernels
    int resident_streams = 2;   // measured: 2 beats 1 by 7-20 % and 3 by 3-10 % on configs 2-5
    cudaEvent_t ev_fork = nullptr, ev_join[kSlots] = {nullptr, nullptr, nullptr};
    // recorded on the caller's stream at the end of every device-resident call: the host pipeline's streams wait for
    // it, so that a later mvd_deconvolve_host never touches the slots' scratch while that work is still running
    cudaEvent_t ev_last = nullptr;
    bool have_last = false;

    int update_mode = 0;    // MVD_UPDATE_SEQUENTIAL / MVD_UPDATE_PRODUCT
    int chunk_planes = 0;   // 0 = default
    int batch_planes = 0;   // 0 = default

    // launch sequences replayed as CUDA graphs (mvd_api.cu: run_graphed): a batch of the host pipeline, or a whole
    // device-resident call of at most ~4000 launches on the same buffers as an earlier one
    std::vector<GraphEntry> graphs;
    uint64_t graph_epoch = 0, graph_clock = 0;
    bool use_graphs = true;

    int last_cuda = 0;
    long long launches = 0;
    bool profiling = false;
    std::vector<ProfRecord> prof;
    std::vector<cudaEvent_t> event_pool;
};

// Bracket a kernel launch: counts it and, when profiling, records events on `stream`.
struct LaunchScope {
    mvd_handle* h;
    cudaStream_t stream;
    cudaEvent_t e1 = nullptr;
    LaunchScope(mvd_handle* h_, int kc, cudaStream_t s);
    ~LaunchScope();
};

// Where plane p, image row y of view v starts in a uint16 view buffer (elements): v * view + p * plane + y * row.
// The ABI's default is view-major stacks of resliced planes {N H W, H W, W}; camera order (z-stacks of
// camera frames, Fig. 1a: planes orthogonal to the rotation axis are x-z planes, so plane
// p is camera line p of every frame) is {H N W, W, N W} -- reslicing is folded into the first read.
struct ViewLayout {
    size_t view, plane, row;
};

// What one call reads and writes, as the engines see it (device pointers; plane 0 = the first plane of the call
// or chunk).  weights: nullptr, or per-view per-pixel fp32 weights of step a4w (reading W1), dense [V][n][H][W]
// with w_view elements between views.  Exactly one of out (fp32) / out16 (uint16, round to nearest even,
// saturated at 65535) is set.
struct PlaneIO {
    const uint16_t* views = nullptr;
    ViewLayout lay{0, 0, 0};
    const float* weights = nullptr;
    size_t w_view = 0;
    float* out = nullptr;
    uint16_t* out16 = nullptr;
    PlaneIO at(int p0, size_t npx) const {     // the same, starting p0 planes further on
        PlaneIO r = *this;
        r.views = views + (size_t)p0 * lay.plane;
        if (weights) r.weights = weights + (size_t)p0 * npx;
        if (out) r.out = out + (size_t)p0 * npx;
        if (out16) r.out16 = out16 + (size_t)p0 * npx;
        return r;
    }
};

// Returns MVD_OK or records the CUDA error in h and returns MVD_ERR_CUDA / MVD_ERR_NOMEM.
int mvd_check(mvd_handle* h, cudaError_t e);
#define MVD_TRY(h, expr)                        \
    do {                                        \
        int rc__ = mvd_check((h), (expr));      \
        if (rc__ != MVD_OK) return rc__;        \
    } while (0)

int ws_reserve(mvd_handle* h, Workspace& ws, size_t a_bytes, size_t b_bytes, size_t g_bytes = 0);
int ws_reserve_product(mvd_handle* h, Workspace& ws, size_t c_bytes, size_t d_bytes);

// ---- direct path (mvd_direct.cu) ------------------------------------------------------------
int direct_choose_chunk(int K, int* JC, int* Kp);
int direct_setup(mvd_handle* h, const float* host_psfs, const float* host_xs);
size_t direct_scratch_bytes(const mvd_handle* h, int n_planes);
// views: view v of plane p at views + (v * view_stride + p * H * W); out: [n][H][W]
int direct_run(mvd_handle* h, Workspace& ws, const PlaneIO& io, int n_planes, cudaStream_t stream);

// ---- separable fast path (mvd_sep.cu) -----------------------------------------------------------
bool sep_psfs_separable(int n_views, const float* psfs, int K);   // host only
int sep_setup(mvd_handle* h, const float* host_psfs);              // sets h->sep when the plan qualifies
int sep_launch(int mode, const mvd_handle* h, int v, const float* src, const uint16_t* phi, float* dst, int n_planes,
               cudaStream_t st, size_t phi_plane, size_t phi_row, const float* wgt);

bool direct_small_available(const mvd_handle* h);
bool direct_repair_available(const mvd_handle* h);
// psi: fp32 [n][H][W] iteration buffer of the repair (io.out itself, or scratch when the output is uint16)
// acc: nullptr (sequential update) or fp32 [n][H][W] scratch for the product form (mvd_set_update_mode)
int direct_repair_launch(mvd_handle* h, const PlaneIO& io, float* psi, float* r_scratch,
                         const unsigned* flags, unsigned* barrier, int n_planes, cudaStream_t stream, float* acc = nullptr);

// ---- fft path (mvd_fft.cu) --------------------------------------------------------------------
int fft_supported(int W, int H);
int fft_generation(int W, int H);   // 0: not supported, 1: generation-1 kernels, 2: generation-2 (team) kernels
// smallest supported W x H (by area) with W >= w_min and H >= h_min; 0 if there is none
int fft_pad_dims(int w_min, int h_min, int* W, int* H);
int fft_setup(mvd_handle* h, const float* host_psfs, const float* host_xs);
int fft_run(mvd_handle* h, Workspace& ws, const PlaneIO& io, int n_planes, cudaStream_t stream);
int fft_default_chunk(const mvd_handle* h);
size_t fft_guard_bytes(int n_planes);
void fft_teardown(mvd_handle* h);
