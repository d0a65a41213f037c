// mvd_api.cu -- the C ABI of libmvd (include/mvd.h): plan creation, the device-resident entry
// point, and the three-stream host pipeline (Algorithm 1).
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <new>
#include <vector>

#include "mvd_internal.cuh"

// ---------------------------------------------------------------------------------------------
// helpers
// ---------------------------------------------------------------------------------------------
int mvd_check(mvd_handle* h, cudaError_t e) {
    if (e == cudaSuccess) return MVD_OK;
    if (h) h->last_cuda = (int)e;
    (void)cudaGetLastError();   // clear the sticky-less error state
    return e == cudaErrorMemoryAllocation ? MVD_ERR_NOMEM : MVD_ERR_CUDA;
}

LaunchScope::LaunchScope(mvd_handle* h_, int kc, cudaStream_t s) : h(h_), stream(s) {
    h->launches++;
    if (!h->profiling) return;
    cudaEvent_t ev[2] = {nullptr, nullptr};
    for (int k = 0; k < 2; ++k) {
        if (!h->event_pool.empty()) {
            ev[k] = h->event_pool.back();
            h->event_pool.pop_back();
        } else if (cudaEventCreate(&ev[k]) != cudaSuccess) {
            ev[k] = nullptr;
        }
    }
    if (!ev[0] || !ev[1]) return;
    cudaEventRecord(ev[0], stream);
    e1 = ev[1];
    h->prof.push_back(ProfRecord{kc, ev[0], ev[1]});
}

LaunchScope::~LaunchScope() {
    if (e1) cudaEventRecord(e1, stream);
}

static int grow(mvd_handle* h, float** p, size_t* have, size_t want) {
    if (want <= *have) return MVD_OK;
    if (h) h->graph_epoch++;      // captured launch sequences hold the old pointer
    if (*p) {
        // the buffer may still be in use by work enqueued earlier on this handle's stream
        MVD_TRY(h, cudaDeviceSynchronize());
        MVD_TRY(h, cudaFree(*p));
        *p = nullptr;
        *have = 0;
    }
    MVD_TRY(h, cudaMalloc((void**)p, want));
    *have = want;
    return MVD_OK;
}

int ws_reserve(mvd_handle* h, Workspace& ws, size_t a_bytes, size_t b_bytes, size_t g_bytes) {
    int rc = grow(h, &ws.a, &ws.a_bytes, a_bytes);
    if (rc == MVD_OK) rc = grow(h, &ws.b, &ws.b_bytes, b_bytes);
    if (rc == MVD_OK) rc = grow(h, reinterpret_cast<float**>(&ws.g), &ws.g_bytes, g_bytes);
    return rc;
}

int ws_reserve_product(mvd_handle* h, Workspace& ws, size_t c_bytes, size_t d_bytes) {
    int rc = grow(h, &ws.c, &ws.c_bytes, c_bytes);
    if (rc == MVD_OK) rc = grow(h, &ws.d, &ws.d_bytes, d_bytes);
    return rc;
}

static void ws_free(Workspace& ws) {
    if (ws.a) cudaFree(ws.a);
    if (ws.b) cudaFree(ws.b);
    if (ws.g) cudaFree(ws.g);
    if (ws.pin) cudaFree(ws.pin);
    if (ws.pout) cudaFree(ws.pout);
    if (ws.pw) cudaFree(ws.pw);
    if (ws.c) cudaFree(ws.c);
    if (ws.d) cudaFree(ws.d);
    ws = Workspace();
}

// Replay `body`'s launch sequence as a CUDA graph: captured the first time a key is seen (stream capture on `st`;
// everything body enqueues, including work forked to the internal streams, becomes one graph), launched with one call
// afterwards.  Falls back to running body directly when the stream is already being captured by the caller, while
// profiling, or when capture fails.  body must only enqueue (everything it needs is reserved beforehand).
template <class F>
static int run_graphed(mvd_handle* h, const uint64_t (&key)[8], cudaStream_t st, F&& body) {
    if (!h->use_graphs || h->profiling) return body();
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) {
        (void)cudaGetLastError();
        return body();
    }
    for (size_t i = 0; i < h->graphs.size();) {       // drop what an epoch change invalidated
        if (h->graphs[i].epoch != h->graph_epoch) {
            cudaGraphExecDestroy(h->graphs[i].exec);
            h->graphs[i] = h->graphs.back();
            h->graphs.pop_back();
        } else {
            ++i;
        }
    }
    for (auto& e : h->graphs)
        if (!memcmp(e.key, key, sizeof key)) {
            e.last_use = ++h->graph_clock;
            h->launches += e.launches;
            return mvd_check(h, cudaGraphLaunch(e.exec, st));
        }
    const uint64_t epoch0 = h->graph_epoch;
    const long long launches0 = h->launches;
    if (cudaStreamBeginCapture(st, cudaStreamCaptureModeRelaxed) != cudaSuccess) {
        (void)cudaGetLastError();
        return body();
    }
    const int rc = body();
    cudaGraph_t g = nullptr;
    const cudaError_t ee = cudaStreamEndCapture(st, &g);
    cudaGraphExec_t exec = nullptr;
    if (h->graph_epoch != epoch0 && rc == MVD_OK && ee == cudaSuccess) {
        // body had to allocate (first use of some scratch): nothing ran, the pointers are new -- run it plainly now,
        // the next call captures
        if (g) cudaGraphDestroy(g);
        h->launches = launches0;
        return body();
    }
    if (rc != MVD_OK || ee != cudaSuccess || !g || cudaGraphInstantiate(&exec, g, 0) != cudaSuccess) {
        if (g) cudaGraphDestroy(g);
        (void)cudaGetLastError();
        h->launches = launches0;
        h->use_graphs = false;        // this plan's sequence cannot be captured: plain launches from now on
        return body();
    }
    cudaGraphDestroy(g);
    // bounded: evict the least recently used.  One host-pipeline call alone needs up to 4 slots x 4 batch sizes (ramp, full,
    // remainder) = 16 entries; a cache of that size thrashed as soon as a device-resident capture joined them.
    if (h->graphs.size() >= 64) {
        size_t lru = 0;
        for (size_t i = 1; i < h->graphs.size(); ++i)
            if (h->graphs[i].last_use < h->graphs[lru].last_use) lru = i;
        cudaGraphExecDestroy(h->graphs[lru].exec);
        h->graphs[lru] = h->graphs.back();
        h->graphs.pop_back();
    }
    GraphEntry e;
    memcpy(e.key, key, sizeof key);
    e.epoch = epoch0;
    e.exec = exec;
    e.launches = h->launches - launches0;
    e.last_use = ++h->graph_clock;
    h->graphs.push_back(e);
    return mvd_check(h, cudaGraphLaunch(exec, st));
}

// ---------------------------------------------------------------------------------------------
// plan
// ---------------------------------------------------------------------------------------------
int mvd_path_supported(int path, int plane_w, int plane_h, int psf_size) {
    if (plane_w < 1 || plane_h < 1 || psf_size < 1 || (psf_size % 2) == 0) return 0;
    if (path == MVD_PATH_DIRECT) {
        int JC, Kp;
        direct_choose_chunk(psf_size, &JC, &Kp);
        const size_t smem = sizeof(float) * ((size_t)psf_size * Kp + (size_t)(64 + Kp - 1) * (psf_size + 64 - 1));
        return smem <= 227u * 1024u ? 1 : 0;
    }
    if (path == MVD_PATH_FFT) return fft_supported(plane_w, plane_h);
    if (path == MVD_PATH_AUTO)
        return mvd_path_supported(MVD_PATH_DIRECT, plane_w, plane_h, psf_size) ||
               mvd_path_supported(MVD_PATH_FFT, plane_w, plane_h, psf_size);
    return 0;
}

// Measured crossover.  The FFT engine moves a fixed number of bytes per voxel-view-iteration whatever K
// is: ~120 GVoxel/s on shapes its generation-2 kernels take (where it wins at EVERY K, even K = 3), ~31 GVoxel/s on
// shapes only generation 1 takes.  The direct engine does 4 K^2 flop per unit (88 ... 5.5 GVoxel/s for K = 3 ... 51), or
// 8 K with separable PSFs (79 / 63 GVoxel/s at K = 21 / 41).  So on generation-1 shapes the direct engine is chosen when its
// estimate is better -- except for planes small enough for launch overheads to decide (below 256 x 256: config 1's 8 planes
// of 64 x 64 take 0.22 ms on the FFT engine's replayed launches against 0.50 ms for the direct engine's on-chip kernel).
static int choose_path(int W, int H, int K, bool separable) {
    const bool fft_ok = mvd_path_supported(MVD_PATH_FFT, W, H, K) != 0;
    const bool dir_ok = mvd_path_supported(MVD_PATH_DIRECT, W, H, K) != 0;
    if (fft_ok && dir_ok && fft_generation(W, H) == 1 && (long long)W * H >= 256 * 256) {
        const double fft_rate = 31.0;
        const double direct_rate = separable && K >= 3 && K <= 65 ? std::min(85.0, 95.0 - 0.8 * K)
                                   : K <= 9 ? 75.0 : K <= 13 ? 50.0 : 13000.0 / ((double)K * K);
        if (direct_rate > 1.1 * fft_rate) return MVD_PATH_DIRECT;
    }
    if (fft_ok) return MVD_PATH_FFT;
    if (dir_ok) return MVD_PATH_DIRECT;
    return -1;
}

static int create_impl(int plane_w, int plane_h, int n_views, const float* psfs, int psf_size,
                       const float* xs, int bp_size, int iterations, float eps, int path, mvd_handle** out,
                       bool padded = false) {
    if (!out) return MVD_ERR_INVALID;
    *out = nullptr;
    if (xs) {
        if (bp_size < 1 || (bp_size % 2) == 0 || n_views < 1) return MVD_ERR_INVALID;
        const size_t nx = (size_t)n_views * bp_size * bp_size;
        for (size_t k = 0; k < nx; ++k)
            if (!isfinite(xs[k])) return MVD_ERR_INVALID;
    }
    const int k_eff = xs && bp_size > psf_size ? bp_size : psf_size;   // taps the direct engine works with
    if (!psfs || plane_w < 1 || plane_h < 1 || n_views < 1 || n_views > 255 || iterations < 0)
        return MVD_ERR_INVALID;
    if (psf_size < 1 || (psf_size % 2) == 0) return MVD_ERR_INVALID;
    if (!(eps > 0.f) || !isfinite(eps)) return MVD_ERR_INVALID;
    if ((long long)plane_w * plane_h > (1LL << 30)) return MVD_ERR_INVALID;
    const size_t ncoef = (size_t)n_views * psf_size * psf_size;
    for (size_t k = 0; k < ncoef; ++k)
        if (!isfinite(psfs[k]) || psfs[k] < 0.f) return MVD_ERR_INVALID;
    if (path != MVD_PATH_AUTO && path != MVD_PATH_DIRECT && path != MVD_PATH_FFT) return MVD_ERR_INVALID;
    // Padded plan: the engine works on zero-filled planes at least K - 1 pixels larger -- the next
    // supported transform lengths for the FFT engine, exactly K - 1 more for the direct engine.
    int eng_w = plane_w, eng_h = plane_h;
    if (padded) {
        const int w_min = plane_w + k_eff - 1, h_min = plane_h + k_eff - 1;
        int fw = 0, fh = 0;
        const bool fft_ok = path != MVD_PATH_DIRECT && fft_pad_dims(w_min, h_min, &fw, &fh);
        if (fft_ok) { path = MVD_PATH_FFT; eng_w = fw; eng_h = fh; }
        else if (path == MVD_PATH_FFT) return MVD_ERR_UNSUPPORTED;
        else { path = MVD_PATH_DIRECT; eng_w = w_min; eng_h = h_min; }
        if ((long long)eng_w * eng_h > (1LL << 30) || !mvd_path_supported(path, eng_w, eng_h, k_eff)) return MVD_ERR_UNSUPPORTED;
    } else if (path == MVD_PATH_AUTO) {
        path = choose_path(plane_w, plane_h, k_eff, !xs && sep_psfs_separable(n_views, psfs, psf_size));
        if (path < 0) return MVD_ERR_UNSUPPORTED;
    } else if (!mvd_path_supported(path, plane_w, plane_h, k_eff)) {
        return MVD_ERR_UNSUPPORTED;
    }

    mvd_handle* h = new (std::nothrow) mvd_handle();
    if (!h) return MVD_ERR_NOMEM;
    h->W = eng_w; h->H = eng_h; h->uW = plane_w; h->uH = plane_h; h->padded = padded;
    h->V = n_views; h->K = psf_size; h->T = iterations;
    h->eps = eps; h->path = path;
    h->KX = xs ? bp_size : 0;
    int rc = mvd_check(h, cudaGetDevice(&h->device));
    if (rc == MVD_OK) rc = mvd_check(h, cudaDeviceGetAttribute(&h->n_sm, cudaDevAttrMultiProcessorCount, h->device));
    if (rc == MVD_OK) rc = path == MVD_PATH_FFT ? fft_setup(h, psfs, xs) : direct_setup(h, psfs, xs);
    if (rc == MVD_OK && path == MVD_PATH_DIRECT) rc = sep_setup(h, psfs);
    if (rc != MVD_OK) {
        // keep the cuda error visible to the caller through the return code only
        mvd_destroy(h);
        return rc;
    }
    *out = h;
    return MVD_OK;
}

int mvd_create_path(int plane_w, int plane_h, int n_views, const float* psfs, int psf_size,
                    int iterations, float eps, int path, mvd_handle** out) {
    return create_impl(plane_w, plane_h, n_views, psfs, psf_size, nullptr, 0, iterations, eps, path, out);
}

int mvd_create_padded(int plane_w, int plane_h, int n_views, const float* psfs, int psf_size,
                      int iterations, float eps, int path, mvd_handle** out) {
    return create_impl(plane_w, plane_h, n_views, psfs, psf_size, nullptr, 0, iterations, eps, path, out, true);
}

int mvd_get_engine_plane(const mvd_handle* h, int* w, int* hh) {
    if (!h || !w || !hh) return MVD_ERR_INVALID;
    *w = h->W;
    *hh = h->H;
    return MVD_OK;
}

int mvd_create_backprojectors(int plane_w, int plane_h, int n_views, const float* psfs, int psf_size,
                              const float* backprojectors, int bp_size, int iterations, float eps,
                              int path, mvd_handle** out) {
    if (!backprojectors) {
        if (out) *out = nullptr;
        return MVD_ERR_INVALID;
    }
    return create_impl(plane_w, plane_h, n_views, psfs, psf_size, backprojectors, bp_size, iterations, eps, path, out);
}

// Back-projectors of Supp. Note 2 section 1 under readings B1-B4 of DESIGN.md:
//   X_v = P_v^* . prod_{w != v} F_vw  (pointwise, on P_v^*'s K x K support), normalised to sum 1, with
//   F_vw = P_v^* * P_w * P_w^* (Efficient Bayesian) or P_v^* * P_w (Optimization I), "*" the full convolution.
int mvd_build_backprojectors(int variant, int n_views, const float* psfs, int psf_size, float* out) {
    if (!psfs || !out || n_views < 1 || psf_size < 1 || (psf_size % 2) == 0) return MVD_ERR_INVALID;
    if (variant != MVD_BP_INDEPENDENT && variant != MVD_BP_EFFICIENT_BAYESIAN && variant != MVD_BP_OPTIMIZATION1)
        return MVD_ERR_INVALID;
    const int K = psf_size, c = (K - 1) / 2, G = 2 * K - 1;
    const size_t kk = (size_t)K * K;
    for (size_t k = 0; k < kk * n_views; ++k)
        if (!isfinite(psfs[k]) || psfs[k] < 0.f) return MVD_ERR_INVALID;
    auto P = [&](int v, int j, int i) -> double {       // P_v at array index (j, i), 0 outside
        return (j < 0 || j >= K || i < 0 || i >= K) ? 0.0 : (double)psfs[v * kk + (size_t)j * K + i];
    };
    auto Pf = [&](int v, int j, int i) -> double { return P(v, K - 1 - j, K - 1 - i); };   // P_v^*
    std::vector<double> g((size_t)G * G), x(kk);
    for (int v = 0; v < n_views; ++v) {
        for (int j = 0; j < K; ++j)
            for (int i = 0; i < K; ++i) x[(size_t)j * K + i] = Pf(v, j, i);
        if (variant != MVD_BP_INDEPENDENT) {
            for (int w = 0; w < n_views; ++w) {
                if (w == v) continue;
                // g = P_v^* * P_w on (2K-1)^2, index (a, b) <-> offset (a - 2c, b - 2c)
                for (int a = 0; a < G; ++a)
                    for (int b = 0; b < G; ++b) {
                        double s = 0.0;
                        for (int j = 0; j < K; ++j)
                            for (int i = 0; i < K; ++i) s += Pf(v, j, i) * P(w, a - j, b - i);
                        g[(size_t)a * G + b] = s;
                    }
                for (int j = 0; j < K; ++j)
                    for (int i = 0; i < K; ++i) {
                        double f;
                        if (variant == MVD_BP_OPTIMIZATION1) {
                            f = g[(size_t)(j + c) * G + (i + c)];          // offset (j - c, i - c)
                        } else {                                           // (g * P_w^*) at offset (j - c, i - c)
                            f = 0.0;
                            for (int a = 0; a < G; ++a)
                                for (int b = 0; b < G; ++b)
                                    f += g[(size_t)a * G + b] * Pf(w, j + 2 * c - a, i + 2 * c - b);
                        }
                        x[(size_t)j * K + i] *= f;
                    }
            }
            double sum = 0.0;
            for (size_t k = 0; k < kk; ++k) sum += x[k];
            if (!(sum > 0.0)) return MVD_ERR_INVALID;
            for (size_t k = 0; k < kk; ++k) x[k] /= sum;
        }
        for (size_t k = 0; k < kk; ++k) out[v * kk + k] = (float)x[k];
    }
    return MVD_OK;
}

int mvd_create(int plane_w, int plane_h, int n_views, const float* psfs, int psf_size,
               int iterations, float eps, mvd_handle** out) {
    int path = MVD_PATH_AUTO;
    const char* f = getenv("MVD_FORCE_PATH");
    if (f && !strcmp(f, "direct")) path = MVD_PATH_DIRECT;
    else if (f && !strcmp(f, "fft")) path = MVD_PATH_FFT;
    return mvd_create_path(plane_w, plane_h, n_views, psfs, psf_size, iterations, eps, path, out);
}

void mvd_destroy(mvd_handle* h) {
    if (!h) return;
    cudaDeviceSynchronize();
    for (auto& r : h->prof) { cudaEventDestroy(r.e0); cudaEventDestroy(r.e1); }
    for (auto& e : h->event_pool) cudaEventDestroy(e);
    for (auto& g : h->graphs) cudaGraphExecDestroy(g.exec);
    ws_free(h->ws_main);
    for (int s = 0; s < mvd_handle::kSlots; ++s) {
        ws_free(h->ws_slot[s]);
        if (h->d_in[s]) cudaFree(h->d_in[s]);
        if (h->d_out[s]) cudaFree(h->d_out[s]);
        if (h->d_w[s]) cudaFree(h->d_w[s]);
        if (h->streams[s]) cudaStreamDestroy(h->streams[s]);
        if (h->ev_join[s]) cudaEventDestroy(h->ev_join[s]);
    }
    if (h->ev_fork) cudaEventDestroy(h->ev_fork);
    if (h->ev_last) cudaEventDestroy(h->ev_last);
    if (h->d_coef) cudaFree(h->d_coef);
    if (h->d_sep) cudaFree(h->d_sep);
    if (h->d_guard_total) cudaFree(h->d_guard_total);
    if (h->d_otf) cudaFree(h->d_otf);
    if (h->d_otf_b) cudaFree(h->d_otf_b);
    if (h->d_otf_real) cudaFree(h->d_otf_real);
    fft_teardown(h);
    (void)cudaGetLastError();
    delete h;
}

// ---------------------------------------------------------------------------------------------
// compute
// ---------------------------------------------------------------------------------------------
// The FFT engine packs planes (2m, 2m+1) into one complex plane; chunks and batches start on even
// planes so that the pairing -- and with it every output bit -- does not depend on the chunking.
static int even_up(int n) { return n + (n & 1); }

static int default_chunk(const mvd_handle* h) {
    if (h->chunk_planes > 0) return h->path == MVD_PATH_FFT ? even_up(std::min(h->chunk_planes, 1024)) : h->chunk_planes;
    if (h->path == MVD_PATH_FFT) return fft_default_chunk(h);
    // direct: bound the scratch (one fp32 plane per plane) to ~1 GiB
    const size_t npx = (size_t)h->W * h->H;
    size_t c = ((size_t)1 << 30) / (npx * sizeof(float));
    return (int)std::max<size_t>(1, std::min<size_t>(c, 1 << 20));
}

// Padded plans: staging for chunks of n planes.  The input staging is zeroed when it is allocated and only its
// uW x uH corners are ever rewritten, so the padding stays zero.
static int pad_reserve(mvd_handle* h, Workspace& ws, int n) {
    if (!h->padded) return MVD_OK;
    const size_t npx = (size_t)h->W * h->H;
    const size_t in_b = sizeof(uint16_t) * npx * n * h->V, out_b = sizeof(float) * npx * n;
    if (in_b > ws.pin_bytes) {
        if (ws.pin) { MVD_TRY(h, cudaDeviceSynchronize()); MVD_TRY(h, cudaFree(ws.pin)); ws.pin = nullptr; ws.pin_bytes = 0; h->graph_epoch++; }
        h->graph_epoch++;
        MVD_TRY(h, cudaMalloc((void**)&ws.pin, in_b));
        ws.pin_bytes = in_b;
    }
    // the layout [V][n][H][W] depends on n: the corners move, so the whole buffer is cleared for every new n
    if (out_b > ws.pout_bytes) {
        if (ws.pout) { MVD_TRY(h, cudaDeviceSynchronize()); MVD_TRY(h, cudaFree(ws.pout)); ws.pout = nullptr; ws.pout_bytes = 0; h->graph_epoch++; }
        h->graph_epoch++;
        MVD_TRY(h, cudaMalloc((void**)&ws.pout, out_b));
        ws.pout_bytes = out_b;
    }
    return MVD_OK;
}

// One chunk of a padded plan: embed, run the engine on the padded planes, crop (reading PD1).
static int run_padded_chunk(mvd_handle* h, Workspace& ws, const PlaneIO& sub, int n, cudaStream_t stream) {
    if (sub.lay.row < (size_t)h->uW || sub.lay.plane % sub.lay.row != 0 || sub.lay.plane / sub.lay.row < (size_t)h->uH)
        return MVD_ERR_UNSUPPORTED;   // one pitched 3D copy per view: planes must be whole numbers of rows apart
    const size_t npx = (size_t)h->W * h->H;
    int rc = pad_reserve(h, ws, n);
    if (rc != MVD_OK) return rc;
    // Rows beyond uW and planes' rows beyond uH hold zeros: cleared here because the corner positions depend on n
    // (chunks of one call share n except the last) -- 2 V bytes per padded pixel, ~2 % of a 10-iteration step.
    MVD_TRY(h, cudaMemsetAsync(ws.pin, 0, sizeof(uint16_t) * npx * n * h->V, stream));
    for (int v = 0; v < h->V; ++v) {
        cudaMemcpy3DParms c = {};
        c.srcPtr = make_cudaPitchedPtr(const_cast<uint16_t*>(sub.views + (size_t)v * sub.lay.view), sub.lay.row * sizeof(uint16_t),
                                       h->uW * sizeof(uint16_t), sub.lay.plane / sub.lay.row);
        c.dstPtr = make_cudaPitchedPtr(ws.pin + (size_t)v * n * npx, h->W * sizeof(uint16_t), h->W * sizeof(uint16_t), h->H);
        c.extent = make_cudaExtent(h->uW * sizeof(uint16_t), h->uH, n);
        c.kind = cudaMemcpyDeviceToDevice;
        MVD_TRY(h, cudaMemcpy3DAsync(&c, stream));
    }
    PlaneIO pio;
    if (sub.weights) {
        // weights embedded like the views; ZERO in the padding (psi is zero there whatever the weight is, but the weight
        // must be finite: 0 . NaN would not be 0).  Allocated at the first weighted call of this workspace.
        rc = grow(h, &ws.pw, &ws.pw_bytes, sizeof(float) * npx * n * h->V);
        if (rc != MVD_OK) return rc;
        MVD_TRY(h, cudaMemsetAsync(ws.pw, 0, sizeof(float) * npx * n * h->V, stream));
        const size_t unpx = (size_t)h->uW * h->uH;
        for (int v = 0; v < h->V; ++v) {
            cudaMemcpy3DParms c = {};
            c.srcPtr = make_cudaPitchedPtr(const_cast<float*>(sub.weights + (size_t)v * sub.w_view), h->uW * sizeof(float),
                                           h->uW * sizeof(float), h->uH);
            c.dstPtr = make_cudaPitchedPtr(ws.pw + (size_t)v * n * npx, h->W * sizeof(float), h->W * sizeof(float), h->H);
            c.extent = make_cudaExtent(h->uW * sizeof(float), h->uH, n);
            c.kind = cudaMemcpyDeviceToDevice;
            MVD_TRY(h, cudaMemcpy3DAsync(&c, stream));
        }
        (void)unpx;
        pio.weights = ws.pw;
        pio.w_view = (size_t)n * npx;
    }
    pio.views = ws.pin;
    pio.lay = ViewLayout{(size_t)n * npx, npx, (size_t)h->W};
    if (sub.out16) pio.out16 = reinterpret_cast<uint16_t*>(ws.pout);
    else pio.out = ws.pout;
    rc = h->path == MVD_PATH_FFT ? fft_run(h, ws, pio, n, stream) : direct_run(h, ws, pio, n, stream);
    if (rc != MVD_OK) return rc;
    const size_t elem = sub.out16 ? sizeof(uint16_t) : sizeof(float);
    cudaMemcpy3DParms c = {};
    c.srcPtr = make_cudaPitchedPtr(ws.pout, h->W * elem, h->W * elem, h->H);
    c.dstPtr = make_cudaPitchedPtr(sub.out16 ? (void*)sub.out16 : (void*)sub.out, h->uW * elem, h->uW * elem, h->uH);
    c.extent = make_cudaExtent(h->uW * elem, h->uH, n);
    c.kind = cudaMemcpyDeviceToDevice;
    MVD_TRY(h, cudaMemcpy3DAsync(&c, stream));
    return MVD_OK;
}

// All T iterations on planes [0, n) of `io`, in chunks (each chunk runs to completion).
static int run_core(mvd_handle* h, Workspace& ws, const PlaneIO& io, int n_planes, cudaStream_t stream) {
    const size_t npx = (size_t)h->uW * h->uH;
    const int chunk = default_chunk(h);
    for (int p0 = 0; p0 < n_planes; p0 += chunk) {
        const int n = std::min(chunk, n_planes - p0);
        const PlaneIO sub = io.at(p0, npx);
        int rc = h->padded ? run_padded_chunk(h, ws, sub, n, stream)
                           : h->path == MVD_PATH_FFT ? fft_run(h, ws, sub, n, stream) : direct_run(h, ws, sub, n, stream);
        if (rc != MVD_OK) return rc;
    }
    return MVD_OK;
}

static int default_batch(const mvd_handle* h, int n_planes, int min_batches = 16);

// Streams and events of the host pipeline / the forked device-resident batches, created once.
static int ensure_streams(mvd_handle* h) {
    if (!h->ev_fork) MVD_TRY(h, cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming));
    if (!h->ev_last) MVD_TRY(h, cudaEventCreateWithFlags(&h->ev_last, cudaEventDisableTiming));
    for (int s = 0; s < mvd_handle::kSlots; ++s) {
        if (!h->streams[s]) MVD_TRY(h, cudaStreamCreateWithFlags(&h->streams[s], cudaStreamNonBlocking));
        if (!h->ev_join[s]) MVD_TRY(h, cudaEventCreateWithFlags(&h->ev_join[s], cudaEventDisableTiming));
    }
    return MVD_OK;
}

// Scratch of one workspace that runs n planes at a time (FFT: Z and S, 8 B per voxel each; direct: r).
static void scratch_bytes(const mvd_handle* h, int n, size_t* a, size_t* b, size_t* g) {
    const size_t npx = (size_t)h->W * h->H;
    if (h->path == MVD_PATH_FFT) {
        *a = *b = sizeof(float2) * (size_t)((n + 1) / 2) * npx;
        *g = fft_guard_bytes(n);
    } else {
        *a = h->T > 0 ? sizeof(float) * (size_t)n * npx : 0;
        *b = *g = 0;
    }
}

// Pipeline slots (uint16 in, fp32 out) for batches of B planes.
static int reserve_slots(mvd_handle* h, int B) {
    if ((size_t)B <= h->slot_planes) return MVD_OK;
    const size_t npx = (size_t)h->uW * h->uH;
    MVD_TRY(h, cudaDeviceSynchronize());
    for (int s = 0; s < mvd_handle::kSlots; ++s) {
        if (h->d_in[s]) { cudaFree(h->d_in[s]); h->d_in[s] = nullptr; }
        if (h->d_out[s]) { cudaFree(h->d_out[s]); h->d_out[s] = nullptr; }
    }
    h->slot_planes = 0;
    h->graph_epoch++;
    for (int s = 0; s < mvd_handle::kSlots; ++s) {
        MVD_TRY(h, cudaMalloc((void**)&h->d_in[s], sizeof(uint16_t) * npx * B * h->V));
        MVD_TRY(h, cudaMalloc((void**)&h->d_out[s], sizeof(float) * npx * B));
    }
    h->slot_planes = (size_t)B;
    return MVD_OK;
}

int mvd_reserve(mvd_handle* h, int max_planes) {
    if (!h || max_planes < 1) return MVD_ERR_INVALID;
    int rc = ensure_streams(h);
    if (rc != MVD_OK) return rc;
    const int B = std::max(default_batch(h, max_planes), default_batch(h, max_planes, 4)), chunk = default_chunk(h);
    size_t a, b, g;
    scratch_bytes(h, std::min(chunk, max_planes), &a, &b, &g);
    if ((rc = ws_reserve(h, h->ws_main, a, b, g)) != MVD_OK) return rc;
    if ((rc = pad_reserve(h, h->ws_main, std::min(chunk, max_planes))) != MVD_OK) return rc;
    if (h->update_mode == MVD_UPDATE_PRODUCT) {
        if ((rc = ws_reserve_product(h, h->ws_main, a, h->path == MVD_PATH_FFT ? b : 0)) != MVD_OK) return rc;
        size_t a2, b2, g2;
        scratch_bytes(h, std::min(chunk, B), &a2, &b2, &g2);
        for (int s = 0; s < mvd_handle::kSlots; ++s)
            if ((rc = ws_reserve_product(h, h->ws_slot[s], a2, h->path == MVD_PATH_FFT ? b2 : 0)) != MVD_OK) return rc;
    }
    scratch_bytes(h, std::min(chunk, B), &a, &b, &g);
    for (int s = 0; s < mvd_handle::kSlots; ++s) {
        if ((rc = ws_reserve(h, h->ws_slot[s], a, b, g)) != MVD_OK) return rc;
        if ((rc = pad_reserve(h, h->ws_slot[s], std::min(chunk, B))) != MVD_OK) return rc;
    }
    return reserve_slots(h, B);
}

int mvd_get_batch_planes(const mvd_handle* h, int n_planes) {
    if (!h || n_planes < 1) return MVD_ERR_INVALID;
    return default_batch(h, n_planes);
}

// Device-resident work: one stream, or batches dealt round-robin to internal streams that fork from and
// join the caller's stream (planes are independent; results do not depend on the split).
static int run_resident(mvd_handle* h, const PlaneIO& io, int n_planes, cudaStream_t stream) {
    const size_t npx = (size_t)h->uW * h->uH;
    const int B = default_batch(h, n_planes, 4);
    const int ns = std::min(h->resident_streams, mvd_handle::kSlots);
    if (ns <= 1 || h->profiling || n_planes < 2 * B) return run_core(h, h->ws_main, io, n_planes, stream);
    int rc = ensure_streams(h);
    {
        size_t a, b, g;
        scratch_bytes(h, std::min(default_chunk(h), B), &a, &b, &g);
        for (int s = 0; s < ns && rc == MVD_OK; ++s) rc = ws_reserve(h, h->ws_slot[s], a, b, g);
    }
    if (rc != MVD_OK) return rc;
    MVD_TRY(h, cudaEventRecord(h->ev_fork, stream));
    for (int s = 0; s < ns; ++s) MVD_TRY(h, cudaStreamWaitEvent(h->streams[s], h->ev_fork, 0));
    int k = 0;
    for (int p0 = 0; p0 < n_planes && rc == MVD_OK; p0 += B, ++k) {
        const int s = k % ns;
        rc = run_core(h, h->ws_slot[s], io.at(p0, npx), std::min(B, n_planes - p0), h->streams[s]);
    }
    for (int s = 0; s < ns; ++s) {   // join even after an error so that the caller's stream stays ordered
        int rj = mvd_check(h, cudaEventRecord(h->ev_join[s], h->streams[s]));
        if (rj == MVD_OK) rj = mvd_check(h, cudaStreamWaitEvent(stream, h->ev_join[s], 0));
        if (rc == MVD_OK) rc = rj;
    }
    return rc;
}

// mvd_io -> PlaneIO for n_planes device-resident planes; MVD_ERR_INVALID on a malformed request
static int io_from(const mvd_handle* h, const mvd_io* io, int n_planes, PlaneIO* out) {
    if (!io || !io->views || !io->out) return MVD_ERR_INVALID;
    if (io->out_type != MVD_OUT_F32 && io->out_type != MVD_OUT_U16) return MVD_ERR_INVALID;
    const size_t npx = (size_t)h->uW * h->uH;
    PlaneIO p;
    p.views = io->views;
    if (io->view_stride == 0 && io->plane_stride == 0 && io->row_stride == 0) {
        p.lay = ViewLayout{(size_t)n_planes * npx, npx, (size_t)h->uW};
    } else {
        if (io->row_stride < (size_t)h->uW || io->plane_stride < 1 || (h->V > 1 && io->view_stride < 1)) return MVD_ERR_INVALID;
        p.lay = ViewLayout{io->view_stride, io->plane_stride, io->row_stride};
    }
    p.weights = io->weights;
    p.w_view = (size_t)n_planes * npx;
    if (io->out_type == MVD_OUT_U16) p.out16 = static_cast<uint16_t*>(io->out);
    else p.out = static_cast<float*>(io->out);
    *out = p;
    return MVD_OK;
}

// Scratch of a device-resident call, sized before anything is enqueued (so that the call can be captured).
static int reserve_resident(mvd_handle* h, int n_planes) {
    const int B = default_batch(h, n_planes, 4), chunk = default_chunk(h);
    const int ns = std::min(h->resident_streams, mvd_handle::kSlots);
    const bool forked = !(ns <= 1 || h->profiling || n_planes < 2 * B);
    const bool product = h->update_mode == MVD_UPDATE_PRODUCT;
    size_t a, b, g;
    int rc = MVD_OK;
    if (forked) {
        rc = ensure_streams(h);
        const int n = std::min(chunk, B);
        scratch_bytes(h, n, &a, &b, &g);
        for (int s = 0; s < ns && rc == MVD_OK; ++s) {
            rc = ws_reserve(h, h->ws_slot[s], a, b, g);
            if (rc == MVD_OK) rc = pad_reserve(h, h->ws_slot[s], n);
            if (rc == MVD_OK && product) rc = ws_reserve_product(h, h->ws_slot[s], a, h->path == MVD_PATH_FFT ? b : 0);
        }
    } else {
        const int n = std::min(chunk, n_planes);
        scratch_bytes(h, n, &a, &b, &g);
        rc = ws_reserve(h, h->ws_main, a, b, g);
        if (rc == MVD_OK) rc = pad_reserve(h, h->ws_main, n);
        if (rc == MVD_OK && product) rc = ws_reserve_product(h, h->ws_main, a, h->path == MVD_PATH_FFT ? b : 0);
    }
    return rc;
}

int mvd_deconvolve_planes_ex(mvd_handle* h, const mvd_io* io, int n_planes, void* stream) {
    if (!h || n_planes < 0) return MVD_ERR_INVALID;
    if (n_planes == 0) return MVD_OK;
    PlaneIO p;
    int rc = io_from(h, io, n_planes, &p);
    if (rc != MVD_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    // Launch-bound calls (small planes, few planes: up to ~4000 launches of a few microseconds) are replayed as one
    // CUDA graph when the same buffers come again -- the typical loop over time points.  Larger calls gain nothing.
    const long long est = (long long)((n_planes + default_batch(h, n_planes, 4) - 1) / default_batch(h, n_planes, 4)) *
                          (4LL * h->T * h->V + 3);
    const size_t mvox = (size_t)h->W * h->H * (size_t)std::min(n_planes, default_batch(h, n_planes, 4));
    auto mark_last = [&](int r) {     // order a later host-pipeline call after this one (not while the caller captures)
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (r == MVD_OK && ensure_streams(h) == MVD_OK && cudaStreamIsCapturing(st, &cs) == cudaSuccess &&
            cs == cudaStreamCaptureStatusNone && cudaEventRecord(h->ev_last, st) == cudaSuccess)
            h->have_last = true;
        (void)cudaGetLastError();
        return r;
    };
    if (est > 4096 || mvox > ((size_t)24 << 20) || h->path != MVD_PATH_FFT) return mark_last(run_resident(h, p, n_planes, st));
    // the direct engine's row-chunk scratch `b` of a uint16 call etc. is covered by ws_reserve inside; for the graph
    // everything is sized now
    if ((rc = reserve_resident(h, n_planes)) != MVD_OK) return rc;
    const uint64_t key[8] = {1u, (uint64_t)(uintptr_t)p.views, (uint64_t)p.lay.view, (uint64_t)p.lay.plane ^ ((uint64_t)p.lay.row << 32),
                             (uint64_t)(uintptr_t)p.weights, (uint64_t)(uintptr_t)(p.out ? (void*)p.out : (void*)p.out16),
                             (uint64_t)(p.out16 ? 1 : 0), (uint64_t)n_planes};
    return mark_last(run_graphed(h, key, st, [&] { return run_resident(h, p, n_planes, st); }));
}

int mvd_deconvolve_planes(mvd_handle* h, const uint16_t* dev_views_u16, float* dev_out_f32,
                          int n_planes, void* stream) {
    const mvd_io io = {dev_views_u16, 0, 0, 0, nullptr, dev_out_f32, MVD_OUT_F32, 0};
    return mvd_deconvolve_planes_ex(h, &io, n_planes, stream);
}

int mvd_deconvolve_planes_strided(mvd_handle* h, const uint16_t* dev_views_u16, size_t view_stride,
                                  size_t plane_stride, size_t row_stride, float* dev_out_f32,
                                  int n_planes, void* stream) {
    if (view_stride == 0 && plane_stride == 0 && row_stride == 0) return MVD_ERR_INVALID;
    const mvd_io io = {dev_views_u16, view_stride, plane_stride, row_stride, nullptr, dev_out_f32, MVD_OUT_F32, 0};
    return mvd_deconvolve_planes_ex(h, &io, n_planes, stream);
}

int mvd_deconvolve_planes_weighted(mvd_handle* h, const uint16_t* dev_views_u16, const float* dev_weights_f32,
                                   float* dev_out_f32, int n_planes, void* stream) {
    if (!dev_weights_f32) return MVD_ERR_INVALID;
    const mvd_io io = {dev_views_u16, 0, 0, 0, dev_weights_f32, dev_out_f32, MVD_OUT_F32, 0};
    return mvd_deconvolve_planes_ex(h, &io, n_planes, stream);
}

int mvd_deconvolve_planes_u16(mvd_handle* h, const uint16_t* dev_views_u16, uint16_t* dev_out_u16,
                              int n_planes, void* stream) {
    const mvd_io io = {dev_views_u16, 0, 0, 0, nullptr, dev_out_u16, MVD_OUT_U16, 0};
    return mvd_deconvolve_planes_ex(h, &io, n_planes, stream);
}

// min_batches: 16 for the host pipeline (its fill and drain -- one H2D and one D2H that overlap nothing -- stay a few
// percent), 4 for device-resident stacks (two batches per internal stream; measured on config 2: 134 vs 128 GVoxel/s)
static int default_batch(const mvd_handle* h, int n_planes, int min_batches) {
    if (h->batch_planes > 0)
        return h->path == MVD_PATH_FFT ? even_up(h->batch_planes) : std::min(h->batch_planes, n_planes);
    // ~64 MiB of uint16 input per batch
    const size_t per_plane = (size_t)h->uW * h->uH * sizeof(uint16_t) * h->V;
    size_t b = std::max<size_t>(1, ((size_t)64 << 20) / per_plane);
    if (h->path == MVD_PATH_FFT) {
        // FFT engine (device-resident stacks and the host pipeline alike): two batches are in flight, each cycling its Z and S (8 B per
        // plane-pixel together) through all T x V passes.  When two such working sets fit the 126 MB L2 with at
        // least five planes per batch the passes run largely from L2 (measured: configs 2 / 3 / 5 best
        // at 64 / 8-16 / 4-6 planes); when they cannot (config 4: 13 MB per plane), long launches win instead
        // (~32 Mvoxel per batch: 99 vs 95 GVoxel/s at 10 planes).
        const size_t npx = (size_t)h->W * h->H;
        const size_t fit = (size_t)100e6 / (16 * npx);
        b = fit >= 5 ? fit : std::max<size_t>(1, ((size_t)32 << 20) / npx);
    }
    b = std::min<size_t>(b, std::max(1, n_planes / min_batches));
    // ... but never batches so small that a launch has nothing to chew on: at least ~2 Mvoxel
    // (config 1's 8 planes of 64 x 64 stay one batch)
    const size_t floor_planes = (((size_t)2 << 20) + (size_t)h->uW * h->uH - 1) / ((size_t)h->uW * h->uH);
    b = std::max(b, floor_planes);
    b = std::max<size_t>(1, std::min<size_t>(b, (size_t)n_planes));
    return h->path == MVD_PATH_FFT ? even_up((int)b) : (int)b;
}

// camera_order: the host stack is [V][H][n_planes][W] (z-stacks of camera frames; plane p = camera line p
// of every frame).  A batch of B planes is then H row-blocks of B*W contiguous uint16 per view: one
// cudaMemcpy2DAsync, landing as [V][H][B][W]; the kernels read it in place with ViewLayout{H B W, W, B W}.
int mvd_deconvolve_host_ex(mvd_handle* h, const mvd_io* io, int n_planes) {
    if (!h || n_planes < 0) return MVD_ERR_INVALID;
    if (n_planes == 0) return MVD_OK;
    if (!io || !io->views || !io->out) return MVD_ERR_INVALID;
    if (io->out_type != MVD_OUT_F32 && io->out_type != MVD_OUT_U16) return MVD_ERR_INVALID;
    if (io->view_stride || io->plane_stride || io->row_stride) return MVD_ERR_INVALID;   // host stacks are dense
    const bool camera_order = io->camera_order != 0, u16 = io->out_type == MVD_OUT_U16;
    if (h->padded && camera_order) return MVD_ERR_UNSUPPORTED;
    const uint16_t* host_views_u16 = io->views;
    const float* host_w = io->weights;
    const size_t npx = (size_t)h->uW * h->uH;
    const size_t out_elem = u16 ? sizeof(uint16_t) : sizeof(float);
    const int B = default_batch(h, n_planes);

    {   // everything the batches need is sized before the first copy is enqueued: nothing below allocates
        int rc0 = ensure_streams(h);
        if (rc0 == MVD_OK) rc0 = reserve_slots(h, B);
        if (rc0 == MVD_OK && host_w && (size_t)B > h->slot_w_planes) {
            rc0 = mvd_check(h, cudaDeviceSynchronize());
            for (int s = 0; s < mvd_handle::kSlots; ++s) {
                if (h->d_w[s]) { cudaFree(h->d_w[s]); h->d_w[s] = nullptr; }
            }
            h->slot_w_planes = 0;
            h->graph_epoch++;
            for (int s = 0; s < mvd_handle::kSlots && rc0 == MVD_OK; ++s)
                rc0 = mvd_check(h, cudaMalloc((void**)&h->d_w[s], sizeof(float) * npx * B * h->V));
            if (rc0 == MVD_OK) h->slot_w_planes = (size_t)B;
        }
        size_t a, b, g;
        scratch_bytes(h, std::min(default_chunk(h), B), &a, &b, &g);
        for (int s = 0; s < mvd_handle::kSlots && rc0 == MVD_OK; ++s) {
            rc0 = ws_reserve(h, h->ws_slot[s], a, b, g);
            if (rc0 == MVD_OK) rc0 = pad_reserve(h, h->ws_slot[s], std::min(default_chunk(h), B));
            if (rc0 == MVD_OK && h->update_mode == MVD_UPDATE_PRODUCT)
                rc0 = ws_reserve_product(h, h->ws_slot[s], a, h->path == MVD_PATH_FFT ? b : 0);
        }
        if (rc0 != MVD_OK) return rc0;
    }

    // Algorithm 1 with batches of planes instead of single planes and pinned
    // host memory instead of disk: batch k goes to stream k mod 3; within a stream H2D, the RL
    // steps and D2H are ordered, across streams they overlap.  Nothing blocks until the end.
    // Batch sizes: B, with a ramp B/4, B/2 at both ends of a long stack so that the first H2D copy and the
    // last D2H copy -- the only ones that overlap no compute -- are short.
    // Every batch except the very last holds an EVEN number of planes: the FFT engine pairs planes (2m, 2m+1)
    // counted from the start of its batch, so a batch that started on an odd plane would pair differently
    // from mvd_deconvolve_planes and the output bits would differ.  An odd stack is split as if it had one
    // plane less and the last plane joins the last batch (or forms a batch of its own when that one is full).
    std::vector<int> sizes;
    {
        std::vector<int> ramp;
        const int n_even = n_planes & ~1;
        if (h->batch_planes == 0 && n_even >= 8 * B && B >= 8) ramp = {(B / 4 + 1) & ~1, (B / 2 + 1) & ~1};
        int left = n_even;
        for (int r : ramp) { sizes.push_back(r); left -= r; }
        int tail = 0;
        for (int r : ramp) tail += r;
        while (left - tail > 0) { const int n = std::min(B, left - tail); sizes.push_back(n); left -= n; }
        for (auto it = ramp.rbegin(); it != ramp.rend(); ++it) sizes.push_back(*it);
        if (n_planes & 1) {
            if (!sizes.empty() && sizes.back() < B) sizes.back() += 1;
            else sizes.push_back(1);
        }
    }
    const int P = h->pipeline_slots;
    const int used = std::min<int>(P, (int)sizes.size());      // streams this call touches (small stacks: one)
    if (h->have_last) {     // device-resident work enqueued earlier on this handle shares the slots' scratch
        for (int s = 0; s < used; ++s) MVD_TRY(h, cudaStreamWaitEvent(h->streams[s], h->ev_last, 0));
        h->have_last = false;   // ... and everything enqueued here is complete when this call returns
    }
    int rc = MVD_OK;
    int k = 0, p0 = 0;
    for (size_t bi = 0; bi < sizes.size() && rc == MVD_OK; p0 += sizes[bi], ++bi, ++k) {
        const int s = k % P;
        const int n = sizes[bi];
        cudaStream_t st = h->streams[s];
        PlaneIO p;
        p.views = h->d_in[s];
        if (camera_order) {
            p.lay = ViewLayout{(size_t)h->uH * B * h->uW, (size_t)h->uW, (size_t)B * h->uW};
            for (int v = 0; v < h->V && rc == MVD_OK; ++v)
                rc = mvd_check(h, cudaMemcpy2DAsync(h->d_in[s] + (size_t)v * p.lay.view, sizeof(uint16_t) * B * h->uW,
                                                   host_views_u16 + ((size_t)v * h->uH * n_planes + p0) * h->uW,
                                                   sizeof(uint16_t) * (size_t)n_planes * h->uW,
                                                   sizeof(uint16_t) * (size_t)n * h->uW, (size_t)h->uH,
                                                   cudaMemcpyHostToDevice, st));
        } else {
            p.lay = ViewLayout{(size_t)B * npx, npx, (size_t)h->uW};
            for (int v = 0; v < h->V && rc == MVD_OK; ++v)
                rc = mvd_check(h, cudaMemcpyAsync(h->d_in[s] + (size_t)v * B * npx,
                                                 host_views_u16 + ((size_t)v * n_planes + p0) * npx,
                                                 sizeof(uint16_t) * npx * n, cudaMemcpyHostToDevice, st));
        }
        if (host_w) {
            p.weights = h->d_w[s];
            p.w_view = (size_t)B * npx;
            for (int v = 0; v < h->V && rc == MVD_OK; ++v)
                rc = mvd_check(h, cudaMemcpyAsync(h->d_w[s] + (size_t)v * B * npx,
                                                 host_w + ((size_t)v * n_planes + p0) * npx,
                                                 sizeof(float) * npx * n, cudaMemcpyHostToDevice, st));
        }
        if (u16) p.out16 = reinterpret_cast<uint16_t*>(h->d_out[s]);
        else p.out = h->d_out[s];
        // at most two batches compute at a time (measured: two concurrent batches fill each other's kernel
        // tails, a third only adds contention), while the copies of all three streams overlap freely
        if (rc == MVD_OK && k >= 2) rc = mvd_check(h, cudaStreamWaitEvent(st, h->ev_join[(k - 2) % P], 0));
        if (rc == MVD_OK) {     // the batch's launch sequence depends on the slot and the batch size only: replayed as a graph
            const uint64_t key[8] = {2u, (uint64_t)s, (uint64_t)n, (uint64_t)B, (uint64_t)(u16 ? 1 : 0) | (host_w ? 2u : 0u) | (camera_order ? 4u : 0u),
                                     0, 0, 0};
            rc = run_graphed(h, key, st, [&] { return run_core(h, h->ws_slot[s], p, n, st); });
        }
        if (rc == MVD_OK) rc = mvd_check(h, cudaEventRecord(h->ev_join[s], st));
        if (rc == MVD_OK)
            rc = mvd_check(h, cudaMemcpyAsync(static_cast<char*>(io->out) + (size_t)p0 * npx * out_elem, h->d_out[s],
                                             out_elem * npx * n, cudaMemcpyDeviceToHost, st));
    }
    for (int s = 0; s < used; ++s) {
        int rs = mvd_check(h, cudaStreamSynchronize(h->streams[s]));
        if (rc == MVD_OK) rc = rs;
    }
    return rc;
}

int mvd_deconvolve_host(mvd_handle* h, const uint16_t* host_views_u16, float* host_out_f32,
                        int n_planes) {
    const mvd_io io = {host_views_u16, 0, 0, 0, nullptr, host_out_f32, MVD_OUT_F32, 0};
    return mvd_deconvolve_host_ex(h, &io, n_planes);
}

int mvd_deconvolve_host_camera(mvd_handle* h, const uint16_t* host_frames_u16, float* host_out_f32,
                               int n_planes) {
    const mvd_io io = {host_frames_u16, 0, 0, 0, nullptr, host_out_f32, MVD_OUT_F32, 1};
    return mvd_deconvolve_host_ex(h, &io, n_planes);
}

int mvd_deconvolve_host_weighted(mvd_handle* h, const uint16_t* host_views_u16, const float* host_weights_f32,
                                 float* host_out_f32, int n_planes) {
    if (!host_weights_f32) return MVD_ERR_INVALID;
    const mvd_io io = {host_views_u16, 0, 0, 0, host_weights_f32, host_out_f32, MVD_OUT_F32, 0};
    return mvd_deconvolve_host_ex(h, &io, n_planes);
}

int mvd_deconvolve_host_u16(mvd_handle* h, const uint16_t* host_views_u16, uint16_t* host_out_u16, int n_planes) {
    const mvd_io io = {host_views_u16, 0, 0, 0, nullptr, host_out_u16, MVD_OUT_U16, 0};
    return mvd_deconvolve_host_ex(h, &io, n_planes);
}

// ---------------------------------------------------------------------------------------------
// small accessors
// ---------------------------------------------------------------------------------------------
const char* mvd_strerror(int code) {
    switch (code) {
        case MVD_OK: return "ok";
        case MVD_ERR_INVALID: return "invalid argument";
        case MVD_ERR_UNSUPPORTED: return "shape not supported by the requested path";
        case MVD_ERR_CUDA: return "CUDA error (see mvd_last_cuda_error)";
        case MVD_ERR_NOMEM: return "out of device or pinned memory";
        case MVD_ERR_BUSY: return "handle busy";
        case MVD_ERR_IO: return "file could not be opened, is too short, or a read / write failed";
        case MVD_ERR_TOO_LARGE: return "request exceeds MVD_NOALLOC_MAX_VOXELS, the fixed scratch of mvd_deconvolve_planes_noalloc";
        default: return "unknown mvd error code";
    }
}

int mvd_last_cuda_error(const mvd_handle* h) { return h ? h->last_cuda : 0; }

long long mvd_guard_flagged(mvd_handle* h) {
    if (!h) return MVD_ERR_INVALID;
    if (!h->d_guard_total) return 0;
    unsigned n = 0;
    if (mvd_check(h, cudaDeviceSynchronize()) != MVD_OK) return MVD_ERR_CUDA;
    if (mvd_check(h, cudaMemcpy(&n, h->d_guard_total, sizeof n, cudaMemcpyDeviceToHost)) != MVD_OK) return MVD_ERR_CUDA;
    return (long long)n;
}
int mvd_get_path(const mvd_handle* h) { return h ? h->path : MVD_ERR_INVALID; }

int mvd_set_update_mode(mvd_handle* h, int mode) {
    if (!h || (mode != MVD_UPDATE_SEQUENTIAL && mode != MVD_UPDATE_PRODUCT)) return MVD_ERR_INVALID;
    h->update_mode = mode;
    h->graph_epoch++;
    return MVD_OK;
}

int mvd_set_chunk_planes(mvd_handle* h, int planes) {
    if (!h || planes < 0) return MVD_ERR_INVALID;
    h->chunk_planes = planes;
    h->graph_epoch++;
    return MVD_OK;
}

int mvd_set_resident_streams(mvd_handle* h, int n) {
    if (!h || n < 1 || n > 3) return MVD_ERR_INVALID;
    h->resident_streams = n;
    h->graph_epoch++;
    return MVD_OK;
}

int mvd_set_pipeline_streams(mvd_handle* h, int n) {
    if (!h || n < 3 || n > mvd_handle::kSlots) return MVD_ERR_INVALID;
    h->pipeline_slots = n;
    h->graph_epoch++;
    return MVD_OK;
}

int mvd_set_batch_planes(mvd_handle* h, int planes) {
    if (!h || planes < 0) return MVD_ERR_INVALID;
    h->batch_planes = planes;
    h->graph_epoch++;
    return MVD_OK;
}

long long mvd_launch_count(const mvd_handle* h) { return h ? h->launches : 0; }
void mvd_launch_count_reset(mvd_handle* h) { if (h) h->launches = 0; }

int mvd_profile_enable(mvd_handle* h, int on) {
    if (!h) return MVD_ERR_INVALID;
    h->profiling = on != 0;
    return MVD_OK;
}

int mvd_profile_read(mvd_handle* h, float* ms, long long* n) {
    if (!h || !ms || !n) return MVD_ERR_INVALID;
    for (int k = 0; k < MVD_N_KERNEL_CLASSES; ++k) { ms[k] = 0.f; n[k] = 0; }
    int rc = MVD_OK;
    for (auto& r : h->prof) {
        float t = 0.f;
        cudaError_t e = cudaEventSynchronize(r.e1);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&t, r.e0, r.e1);
        if (e != cudaSuccess) rc = mvd_check(h, e);
        else if (r.kc >= 0 && r.kc < MVD_N_KERNEL_CLASSES) { ms[r.kc] += t; n[r.kc]++; }
        h->event_pool.push_back(r.e0);
        h->event_pool.push_back(r.e1);
    }
    h->prof.clear();
    return rc;
}

const char* mvd_kernel_class_name(int k) {
    static const char* names[MVD_N_KERNEL_CLASSES] = {
        "init_mean", "direct_blur_ratio", "direct_backproject_update", "fft_rows_first",
        "fft_cols_otf", "fft_rows_ratio", "fft_rows_update", "setup", "guard_repair", "small_resident",
        "sep_blur_ratio", "sep_backproject_update"};
    return (k >= 0 && k < MVD_N_KERNEL_CLASSES) ? names[k] : nullptr;
}

const char* mvd_version(void) { return "mvd 0.1 sm_100a"; }
