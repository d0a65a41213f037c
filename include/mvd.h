/*
 * mvd.h -- C ABI of libmvd: plane-wise multi-view Richardson-Lucy deconvolution on one B200.
 *
 * The operation (arXiv 1503.07998, Schmid & Huisken, "Real-time multi-view deconvolution"):
 *   PAPER.md:79      (Supp. Note 1)  psi^{t+1} = psi^t  prod_v  ( phi_v / (psi^t * P_v) ) * P_v^*
 *   PAPER.md:100-104 (Supp. Note 2 s.1) "Independent" back-projector X = P_v^*
 *   PAPER.md:118     P_v^* is the flipped PSF of view v
 *   PAPER.md:31      the 3D transfer function is approximated by a 2D PSF, so every plane orthogonal
 *                    to the rotation axis (an x-z plane) is an independent 2D problem
 *   PAPER.md:87-89   phi_v is uint16 camera data, the estimate psi is float
 *   PAPER.md:126-152 (Supp. Note 2 s.3, Algorithm 1) three CUDA streams overlap H2D, the RL steps and D2H
 *
 * Per plane, with the readings of DESIGN.md (the paper is silent on most of them; BASELINE.json's
 * north_star fixes them): psi_0 = mean_v phi_v; then for t = 0..iterations-1, for v = 0..n_views-1 IN TURN
 *   b   = psi (*) P_v                      periodic convolution   b(x) = sum_u P_v(u) psi(x - u)
 *   r   = phi_v / max(b, eps)
 *   q   = r (*) P_v^*                      periodic correlation   q(x) = sum_u P_v(u) r(x + u)
 *   psi = psi . q
 * PSF array index (j, i) <-> offset u = (j - c, i - c), c = (psf_size - 1) / 2, j along z (rows), i along x.
 *
 * Layouts (x fastest everywhere):
 *   psfs   float    [n_views][psf_size][psf_size]
 *   views  uint16_t [n_views][n_planes][plane_h][plane_w]      ("view-major": each view is one stack)
 *   out    float    [n_planes][plane_h][plane_w]
 *
 * All functions return MVD_OK (0) or a negative code; nothing throws, aborts or prints.  The library
 * never falls back to the CPU: without a CUDA device every compute call fails with MVD_ERR_CUDA.
 */
#ifndef MVD_H_
#define MVD_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define MVD_API __attribute__((visibility("default")))
#else
#define MVD_API
#endif

typedef struct mvd_handle mvd_handle; /* opaque; owned by the library; one device, not thread-safe */

enum {
    MVD_OK = 0,
    MVD_ERR_INVALID = -1,     /* null pointer, non-positive size, even psf_size, bad eps, bad PSF value */
    MVD_ERR_UNSUPPORTED = -2, /* a forced path cannot handle this shape (e.g. FFT on a non-smooth size)  */
    MVD_ERR_CUDA = -3,        /* a CUDA call failed; mvd_last_cuda_error() has the cudaError_t           */
    MVD_ERR_NOMEM = -4,       /* device or pinned-staging allocation failed                              */
    MVD_ERR_BUSY = -5,        /* reserved                                                                */
    MVD_ERR_IO = -6,          /* mvd_deconvolve_files: a file could not be opened, is too short, or a read / write failed */
    MVD_ERR_TOO_LARGE = -7    /* mvd_deconvolve_planes_noalloc: n_planes * plane_w * plane_h exceeds MVD_NOALLOC_MAX_VOXELS */
};

/* Convolution engine used for steps a1 and a3 (both engines fuse a2 and a4 into their kernels). */
enum {
    MVD_PATH_AUTO = 0,   /* chosen in mvd_create from the measured crossover: the FFT engine on every shape its
                            fast kernels take; on the other supported shapes whichever engine is estimated faster for this K  */
    MVD_PATH_DIRECT = 1, /* shared-memory halo tiles + register-blocked FP32 FMA; any shape               */
    MVD_PATH_FFT = 2     /* hand-written batched 2D FFT with the pointwise steps fused into the passes;
                            plane_w and plane_h must be supported transform lengths (32 ... 2048) within the kernel's
                            shared-memory limit (see mvd_path_supported)                                  */
};

/*
 * mvd_create -- build a plan for planes of plane_w x plane_h pixels seen by n_views views.
 *   psfs        HOST pointer, float [n_views][psf_size][psf_size]; copied, may be freed on return.
 *               Used as given (not renormalised); values must be finite and >= 0.
 *   psf_size    odd, >= 1.  psf_size > plane_w or plane_h is allowed (taps alias around the plane).
 *   iterations  >= 0; 0 returns the mean of the views (the count is the user's choice).
 *   eps         division guard of step a2, finite and > 0 (north_star: 1e-6).
 *   out         receives the handle.
 * The path is MVD_PATH_AUTO unless the environment variable MVD_FORCE_PATH is "direct" or "fft"
 * (measurement only).  Errors: MVD_ERR_INVALID, MVD_ERR_UNSUPPORTED (forced path), MVD_ERR_CUDA, MVD_ERR_NOMEM.
 */
MVD_API int mvd_create(int plane_w, int plane_h, int n_views, const float* psfs, int psf_size,
               int iterations, float eps, mvd_handle** out);

/* Same, with the path given explicitly (MVD_PATH_*); MVD_FORCE_PATH is ignored. */
MVD_API int mvd_create_path(int plane_w, int plane_h, int n_views, const float* psfs, int psf_size,
                    int iterations, float eps, int path, mvd_handle** out);

/*
 * mvd_create_padded -- the paper's own boundary (Supp. Table 1 caption: the transformed sizes are "the
 * sum of the actual data size and the size of PSF").  The caller's planes stay plane_w x plane_h; inside the library
 * every plane of every view is embedded in a ZERO-filled plane at least psf_size - 1 pixels larger in x and z
 * (READING PD1 of DESIGN.md: the paper does not say what the padding holds), the periodic iteration of mvd_create runs
 * on the padded planes and the result is cropped.  Because psi_0 and r are zero in the padding and the update is
 * multiplicative, the result is the RL iteration with zero boundary conditions on the caller's plane, whatever the
 * padded size is.  The FFT engine pads to the next supported transform lengths (so ANY plane_w, plane_h up to
 * 2048 - psf_size + 1 runs on it), the direct engine to exactly plane + psf_size - 1; mvd_get_engine_plane tells.
 *   path   MVD_PATH_AUTO (FFT whenever a padded size exists) / MVD_PATH_DIRECT / MVD_PATH_FFT.
 * Layouts, ownership and errors as for mvd_create.  Calls on a padded handle take dense or row-strided views (planes a
 * whole number of rows apart) and per-view weights (embedded like the views, zero in the padding); camera-order host
 * stacks return MVD_ERR_UNSUPPORTED.
 * Cost: one zero-fill + embed copy of the views and one crop copy of the result per chunk (2 V + 8 bytes per padded
 * pixel against 42 V T for the iterations), plus the iterations on the larger planes.
 */
MVD_API int mvd_create_padded(int plane_w, int plane_h, int n_views, const float* psfs, int psf_size,
                              int iterations, float eps, int path, mvd_handle** out);

/* The planes the engine of this handle works on: plane_w x plane_h of mvd_create, the padded size of mvd_create_padded. */
MVD_API int mvd_get_engine_plane(const mvd_handle* h, int* w, int* hh);

/*
 * Other back-projectors (Supp. Note 2 s.1: "the implemented variants all used the
 * following formula, but replaced X").  Step a3 becomes the TRUE periodic convolution with X_v,
 *   q = r (*) X_v,   q(x) = sum_u X_v(u) r(x - u),   index (j, i) <-> u = (j - cx, i - cx), cx = (bp_size - 1) / 2;
 * X_v = flipped P_v is the Independent variant that mvd_create builds.
 *   backprojectors  HOST, float [n_views][bp_size][bp_size]; copied; finite (any sign); bp_size odd, may
 *                   differ from psf_size.  Used as given (not renormalised).
 *   path            MVD_PATH_AUTO / DIRECT / FFT as in mvd_create_path.
 * Everything else as mvd_create.  Errors: MVD_ERR_INVALID (NULL, even bp_size, non-finite value), ...
 */
MVD_API int mvd_create_backprojectors(int plane_w, int plane_h, int n_views, const float* psfs, int psf_size,
                              const float* backprojectors, int bp_size, int iterations, float eps,
                              int path, mvd_handle** out);

/*
 * mvd_build_backprojectors -- the paper's variants written out on the host (fp64, no device needed):
 *   MVD_BP_INDEPENDENT         X_v = P_v^*
 *   MVD_BP_EFFICIENT_BAYESIAN  X_v = P_v^* . prod_{w != v} (P_v^* * P_w * P_w^*)
 *   MVD_BP_OPTIMIZATION1       X_v = P_v^* . prod_{w != v} (P_v^* * P_w)
 * under the readings of DESIGN.md section 2 (B1-B4; the printed formulas define no operator): "*" is the
 * full convolution of the small kernels, "." and the product sign are pointwise products over a common
 * centre (so X_v lives on P_v^*'s psf_size x psf_size support), W_v is every other view, and the two
 * compound kernels are normalised to sum 1.  Optimization II is not recoverable from the
 * text and is not offered.
 *   psfs  HOST float [n_views][psf_size][psf_size], finite, >= 0;   out  HOST float, same shape.
 */
enum { MVD_BP_INDEPENDENT = 0, MVD_BP_EFFICIENT_BAYESIAN = 1, MVD_BP_OPTIMIZATION1 = 2 };
MVD_API int mvd_build_backprojectors(int variant, int n_views, const float* psfs, int psf_size, float* out);

/*
 * mvd_deconvolve_planes -- steps a0..a5 on n_planes device-resident planes.
 *   dev_views_u16  DEVICE, uint16 [n_views][n_planes][plane_h][plane_w]; read-only.
 *   dev_out_f32    DEVICE, float  [n_planes][plane_h][plane_w]; fully overwritten; must not alias the input.
 *   stream         a cudaStream_t (NULL = legacy default stream).  The call ENQUEUES and returns; it does
 *                  not synchronise -- except that scratch is per handle and grown on demand: a call that needs
 *                  more than is reserved allocates first (see mvd_reserve).  Calls on one handle must all be
 *                  ordered on one stream; a later mvd_deconvolve_host* on the handle waits for them by itself.
 *                  Launch-bound calls (small stacks: at most ~4000 short launches) on the same buffers as an earlier
 *                  call are replayed as one CUDA graph captured on `stream` the first time; a `stream` that the caller
 *                  is capturing himself is never captured again.
 * n_planes == 0 is a no-op.  Errors: MVD_ERR_INVALID, MVD_ERR_CUDA, MVD_ERR_NOMEM.
 */
MVD_API int mvd_deconvolve_planes(mvd_handle* h, const uint16_t* dev_views_u16, float* dev_out_f32,
                          int n_planes, void* stream);

/*
 * mvd_deconvolve_host -- the same result for host-resident stacks, streamed through the GPU in batches
 * of planes on CUDA streams (four by default, the paper's three with mvd_set_pipeline_streams) so that H2D copies, the RL iterations and D2H copies of different
 * batches overlap (Algorithm 1, with pinned host buffers standing in for disk IO).
 *   host_views_u16  HOST (pinned for overlap; pageable memory works but serialises), same layout as above.
 *   host_out_f32    HOST, float [n_planes][plane_h][plane_w].
 * Blocks until host_out_f32 is complete.  Bit-identical to mvd_deconvolve_planes on the same data.
 */
MVD_API int mvd_deconvolve_host(mvd_handle* h, const uint16_t* host_views_u16, float* host_out_f32,
                        int n_planes);

/*
 * Reslicing folded into the first read (Fig. 1a: the acquired stacks
 * are resliced into planes orthogonal to the rotation axis).  Plane p, image row y, pixel x of view v is
 * read at  dev_views_u16[v * view_stride + p * plane_stride + y * row_stride + x]  (strides in uint16
 * elements, each a multiple of 8 for the FFT engine; row_stride >= plane_w).  The default layout of
 * mvd_deconvolve_planes is {n_planes * H * W, H * W, W}; a view acquired as a z-stack of camera frames,
 * uint16 [plane_h (z)][n_planes (camera lines)][plane_w], is {H * N * W, W, N * W}.  Output as above.
 */
MVD_API int mvd_deconvolve_planes_strided(mvd_handle* h, const uint16_t* dev_views_u16, size_t view_stride,
                                  size_t plane_stride, size_t row_stride, float* dev_out_f32,
                                  int n_planes, void* stream);

/*
 * mvd_deconvolve_host with the input in camera order: host_frames_u16 is HOST (pinned) uint16
 * [n_views][plane_h][n_planes][plane_w]; batches are gathered by one 2D copy per view and read in place.
 * Same output, bit-identical to mvd_deconvolve_host on the resliced stack.
 */
MVD_API int mvd_deconvolve_host_camera(mvd_handle* h, const uint16_t* host_frames_u16, float* host_out_f32,
                               int n_planes);

/*
 * The general form of both calls: one request structure instead of one entry point per combination.
 *   views          as in mvd_deconvolve_planes (DEVICE) / mvd_deconvolve_host (HOST, pinned for overlap).
 *   view_stride, plane_stride, row_stride
 *                  all 0: dense uint16 [n_views][n_planes][plane_h][plane_w]; otherwise the strided layout of
 *                  mvd_deconvolve_planes_strided (device calls only).
 *   weights        NULL, or float [n_views][n_planes][plane_h][plane_w] in the same memory space as `views`:
 *                  per-view, per-pixel weights in [0, 1] (PAPER.md:88 lists "weights, float, 4 v bytes/pixel" and
 *                  never defines them; READING W1 of DESIGN.md section 2): step a4 becomes
 *                      psi <- psi . (w_v q + (1 - w_v)),
 *                  so w_v = 1 is the unweighted update bit for bit and w_v = 0 leaves the pixel untouched by view
 *                  v (a registered view that does not cover it).  Values outside [0, 1] are not checked.
 *   out, out_type  MVD_OUT_F32: float [n_planes][plane_h][plane_w] (as above);
 *                  MVD_OUT_U16: uint16_t, same shape: psi rounded to nearest (ties to even) and saturated at
 *                  65535 in the final store (the data are uint16) -- halves the output and its D2H copy.
 *   camera_order   mvd_deconvolve_host_ex only: non-zero = `views` is [n_views][plane_h][n_planes][plane_w] as in
 *                  mvd_deconvolve_host_camera (weights and output stay plane-major).
 * Everything else (asynchrony, ownership, errors) as for mvd_deconvolve_planes / mvd_deconvolve_host.
 */
enum { MVD_OUT_F32 = 0, MVD_OUT_U16 = 1 };
typedef struct mvd_io {
    const uint16_t* views;
    size_t view_stride, plane_stride, row_stride;
    const float* weights;
    void* out;
    int out_type;
    int camera_order;
} mvd_io;
MVD_API int mvd_deconvolve_planes_ex(mvd_handle* h, const mvd_io* io, int n_planes, void* stream);
MVD_API int mvd_deconvolve_host_ex(mvd_handle* h, const mvd_io* io, int n_planes);

/* Shorthands: per-view weights and uint16 output. */
MVD_API int mvd_deconvolve_planes_weighted(mvd_handle* h, const uint16_t* dev_views_u16, const float* dev_weights_f32,
                                           float* dev_out_f32, int n_planes, void* stream);
MVD_API int mvd_deconvolve_host_weighted(mvd_handle* h, const uint16_t* host_views_u16, const float* host_weights_f32,
                                         float* host_out_f32, int n_planes);
MVD_API int mvd_deconvolve_planes_u16(mvd_handle* h, const uint16_t* dev_views_u16, uint16_t* dev_out_u16,
                                      int n_planes, void* stream);
MVD_API int mvd_deconvolve_host_u16(mvd_handle* h, const uint16_t* host_views_u16, uint16_t* host_out_u16, int n_planes);

/*
 * mvd_deconvolve_files -- the paper's whole workflow (Algorithm 1): loading from and saving to disk
 * overlap the GPU pipeline.  view_paths[v] names a raw little-endian uint16 file holding view v as
 * [n_planes][plane_h][plane_w] (the first n_planes planes of a longer file are used); out_path is created / truncated
 * and receives [n_planes][plane_h][plane_w] as float (MVD_OUT_F32) or uint16 (MVD_OUT_U16).  Slabs of planes (a whole
 * number of pipeline batches, ~256 MiB of input) cycle through three pinned buffer sets: a reader thread loads slab
 * k + 1 and a writer thread saves slab k - 1 while slab k runs through mvd_deconvolve_host_ex.  Blocks until the output
 * file is complete; the bytes written are those mvd_deconvolve_host produces.  Errors: MVD_ERR_INVALID, MVD_ERR_IO,
 * MVD_ERR_NOMEM (pinned buffers), and everything mvd_deconvolve_host returns.
 */
MVD_API int mvd_deconvolve_files(mvd_handle* h, const char* const* view_paths, const char* out_path, int n_planes,
                                 int out_type);

/*
 * mvd_deconvolve_planes_noalloc -- mvd_deconvolve_planes for callers that cannot allocate (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc): the call allocates NOTHING -- no cudaMalloc, cudaFree
 * or allocating library routine, whatever was or was not reserved.  It runs the direct engine's tiled kernels (steps
 * a0..a5) with their ratio scratch r in a fixed device array inside the library instead of the handle's
 * workspace:
 *   - limit: n_planes * plane_w * plane_h <= MVD_NOALLOC_MAX_VOXELS (4 Mi voxels = 16 MiB, held by every GPU that
 *     loads libmvd.so until the process exits); larger requests return MVD_ERR_TOO_LARGE and enqueue nothing;
 *   - the handle must run the direct engine (mvd_create_path(.., MVD_PATH_DIRECT, ..)), sequential update mode, not
 *     padded: otherwise MVD_ERR_UNSUPPORTED; the handle's device must be the current device (else MVD_ERR_INVALID);
 *   - dev_views_u16 / dev_out_f32 / stream exactly as for mvd_deconvolve_planes (dense layout, fp32 output); the result
 *     is the direct engine's (for separable PSFs and planes that fit on chip mvd_deconvolve_planes picks other kernels of
 *     that engine: same result within the parity tolerance, otherwise bit for bit);
 *   - the first call on a device resolves the array's address (cudaGetSymbolAddress): make it outside stream capture;
 *   - ALL calls (of all handles) share the one array: calls that overlap on the GPU -- different streams with no
 *     ordering between them -- race on it.  Calls ordered on one stream are safe; the array needs no clearing.
 */
enum { MVD_NOALLOC_MAX_VOXELS = 4194304 };
MVD_API int mvd_deconvolve_planes_noalloc(mvd_handle* h, const uint16_t* dev_views_u16, float* dev_out_f32,
                                          int n_planes, void* stream);

/*
 * mvd_reserve -- size everything a later call on up to max_planes planes needs (scratch of the engine, the
 * internal streams and events, the pipeline's device slots) now.  After it, mvd_deconvolve_planes* with
 * n_planes <= max_planes only enqueues: no allocation, no synchronisation, so the call can be captured into a
 * CUDA graph (stream capture on `stream`).  Without it the first call (and any call that needs more scratch
 * than an earlier one) allocates, which synchronises the device.  Errors: MVD_ERR_INVALID, MVD_ERR_NOMEM.
 */
MVD_API int mvd_reserve(mvd_handle* h, int max_planes);

/* Planes per batch that mvd_deconvolve_host / the forked device-resident path use for a stack of n_planes
 * (the default policy, or mvd_set_batch_planes); batches start at multiples of it. */
MVD_API int mvd_get_batch_planes(const mvd_handle* h, int n_planes);

/*
 * Guard of the FFT engine.  Step a2 divides by the blur b = psi (*) P_v; where b is smaller than the
 * round-off of an fp32 transform (about 1e-6 of the plane's maximum) and phi_v > 0 there, the quotient is noise of
 * the order phi / eps, and the next transform spreads it over the whole plane pair.  (This needs data that say
 * "signal" where the estimate says "nothing": a view zero-filled where the others are not, photons on an exactly
 * zero background.)  The FFT engine therefore flags every plane pair in which some pixel has phi_v > 0 and
 * b < 2^-13 max(psi_0), and recomputes the flagged pairs from scratch with the direct engine's arithmetic, in the
 * same call and on the same stream; the result is the direct engine's, bit for bit.  mvd_guard_flagged returns how
 * many plane pairs this handle has handed over so far (blocks until the handle's work is done).
 */
MVD_API long long mvd_guard_flagged(mvd_handle* h);

/* Frees the plan, its scratch, its streams and staging buffers.  NULL is a no-op. */
MVD_API void mvd_destroy(mvd_handle* h);

/* Static, never-NULL description of a return code. */
MVD_API const char* mvd_strerror(int code);

/* The raw cudaError_t behind the last MVD_ERR_CUDA / MVD_ERR_NOMEM of this handle (0 if none). */
MVD_API int mvd_last_cuda_error(const mvd_handle* h);

/* MVD_PATH_DIRECT or MVD_PATH_FFT: what this handle runs. */
MVD_API int mvd_get_path(const mvd_handle* h);

/* 1 if `path` can run planes of this shape, else 0 (no device needed). */
MVD_API int mvd_path_supported(int path, int plane_w, int plane_h, int psf_size);

/*
 * mvd_set_update_mode -- which form of the multi-view update the handle's later calls run.
 *   MVD_UPDATE_SEQUENTIAL (default)  north_star's reading (A1 of DESIGN.md): for every view in turn, each view's factor is
 *                                    multiplied in before the next view's blur.
 *   MVD_UPDATE_PRODUCT               the update exactly as PAPER.md:79 prints it:
 *                                        psi^{t+1} = psi^t  prod_v  ( phi_v / (psi^t * P_v) ) * P_v^*,
 *                                    every view's factor from the SAME psi^t (the "simultaneous" form).  Both engines run it
 *                                    with the kernels of the sequential form: the factors are multiplied into a copy of psi^t
 *                                    that becomes psi^{t+1} after the last view (FFT engine: every view's blur restarts
 *                                    from a saved copy of psi^t's row spectrum; 8 (1 + 2 / V) extra bytes per unit).  The FFT
 *                                    engine's guard repairs flagged plane pairs with the direct engine's arithmetic in this
 *                                    mode as well (plans whose PSF is too large for the repair kernel only count them:
 *                                    mvd_guard_flagged).
 * Call it before mvd_reserve.  Errors: MVD_ERR_INVALID.
 */
enum { MVD_UPDATE_SEQUENTIAL = 0, MVD_UPDATE_PRODUCT = 1 };
MVD_API int mvd_set_update_mode(mvd_handle* h, int mode);

/*
 * Tuning knobs (measurement; defaults are chosen in mvd_create).
 *   mvd_set_chunk_planes  planes processed per internal pass of mvd_deconvolve_planes (0 = default)
 *   mvd_set_batch_planes  planes per pipeline batch of mvd_deconvolve_host (0 = default)
 *   mvd_set_pipeline_streams  3 or 4 (default 4): streams = batch slots that mvd_deconvolve_host* cycles through.  Algorithm 1
 *                          has three; with two batches computing at a time a stream spends ~40 % of its cycle in
 *                         its own H2D / D2H copies, so a fourth keeps two batches computing (config 2: +4 %); bit-identical
 *   mvd_set_resident_streams  1..3: mvd_deconvolve_planes deals batches of planes (the pipeline's batch size)
 *                         to this many internal streams forked from / joined to the caller's stream, so that
 *                         kernel tails of one batch overlap the next batch; results are bit-identical
 */
MVD_API int mvd_set_pipeline_streams(mvd_handle* h, int n);
MVD_API int mvd_set_resident_streams(mvd_handle* h, int n);
MVD_API int mvd_set_chunk_planes(mvd_handle* h, int planes);
MVD_API int mvd_set_batch_planes(mvd_handle* h, int planes);

/*
 * Instrumentation for bench.py's roofline line.
 *   mvd_launch_count      kernels launched by this handle since creation (or since the last reset).
 *   mvd_profile_enable    when on, every kernel launch is bracketed by CUDA events on the launching stream.
 *   mvd_profile_read      synchronises the recorded events and returns, per kernel class k in
 *                         [0, MVD_N_KERNEL_CLASSES), the summed device time ms[k] and launch count n[k]
 *                         since the last read; both arrays are HOST, length MVD_N_KERNEL_CLASSES.
 *   mvd_kernel_class_name static name of class k (NULL if out of range).
 */
enum { MVD_N_KERNEL_CLASSES = 12 };
MVD_API long long mvd_launch_count(const mvd_handle* h);
MVD_API void mvd_launch_count_reset(mvd_handle* h);
MVD_API int mvd_profile_enable(mvd_handle* h, int on);
MVD_API int mvd_profile_read(mvd_handle* h, float* ms, long long* n);
MVD_API const char* mvd_kernel_class_name(int k);

/*
 * FP32 FMA peak of the current device, measured with a register-only FFMA micro-kernel: *tflops
 * (2 flop per FMA) and the SM clock in MHz seen while it ran.  Denominator of the direct engine's
 * roofline fraction (the driver-measured peaks file has no FP32 figure).
 */
MVD_API int mvd_measure_fp32_peak(double* tflops, double* sm_mhz);

/* Library version string, e.g. "mvd 0.1 sm_100a". */
MVD_API const char* mvd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MVD_H_ */
