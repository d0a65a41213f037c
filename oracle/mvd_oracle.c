/*
 * mvd_oracle.c -- TEST INFRASTRUCTURE.  Plain, slow, fp64 CPU oracle for the plane-wise multi-view
 * Richardson-Lucy iteration of arXiv 1503.07998 (Schmid & Huisken, "Real-time multi-view
 * deconvolution").  It exists to judge the CUDA path; nothing in the product path may import, call,
 * link or execute it (only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs do).  It shares no code with paper_1503_07998_b200/csrc.
 *
 * What it computes (the algorithm step by step, in the paper's notation):
 *
 *   PAPER.md:79  (Supp. Note 1)   psi^{t+1} = psi^t  prod_v  ( phi_v / (psi^t * P_v) ) * P_v^*
 *   PAPER.md:100-104 (Note 2 s.1) "Independent" variant, X = P_v^*
 *   PAPER.md:118                  P_v^* is the flipped PSF of view v
 *   PAPER.md:31                   2D PSF, every plane orthogonal to the rotation axis independent
 *   PAPER.md:87-89                phi_v is uint16, the estimate psi is floating point
 *   PAPER.md:143-145 (Alg. 1)     nIterations RL steps per plane
 *
 * Readings where the paper is silent or ambiguous:
 *   A1 the views are applied SEQUENTIALLY: each view's factor is multiplied into psi before the next
 *      view's blur is formed (BASELINE.json north_star); A2 the ratio is (phi/(psi*P)) and only then
 *      convolved with P^*; A3 "psi * P" is true convolution b(x) = sum_u P(u) psi(x-u), and "* P^*"
 *      is correlation q(x) = sum_u P(u) r(x+u), array index (j,i) <-> offset (j-c, i-c),
 *      c = (K-1)/2, K odd; A4 views in index order 0..V-1, every iteration; A5 periodic boundary on
 *      the plane as given; A6 r = phi / max(b, eps); A7 psi_0 = mean of the views; A8 no weights.
 *
 * Two implementations of the same arithmetic:
 *   *_literal : modular indexing, one pixel at a time -- the definition written out.
 *   default   : the same sums in the same (j, i) order, but read from a wrap-padded copy so the
 *               inner loop is a row axpy (about 14x faster).  Per-pixel summation order is
 *               unchanged; tests assert the two are BIT-IDENTICAL.
 * Compile with -ffp-contract=off so no FMA contraction changes rounding between the two.
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): P1 centred delta, P2 off-centre delta
 * closed form, P3 constants, P4 non-negativity, P5 dense-matrix brute force, P6 sum conservation,
 * P7 I-divergence monotone, P8 numpy-FFT cross-check of both convolutions, P9 duplicated view,
 * P10 shift equivariance, P11 zero iterations; explicit back-projectors (mvd_oracle_x): PX1 X = flip(P)
 * reduces to the Independent variant, PX2 dense-matrix brute force with an asymmetric X of another
 * size, PX3 centred-delta X closed form; per-view weights (mvd_oracle_w): PW1 w = 1 is the unweighted run bit for
 * bit, PW2 a view with w = 0 is never applied, PW3 constants stay fixed, PW4 dense-matrix brute force with random
 * weights.  Parity unpinned: READING W1 (what the paper's "weights" buffer, does) -- its arithmetic is
 * pinned, its meaning is not fixed by anything the paper prints.
 */
#include <math.h>
#include <pthread.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

static int pmod(int a, int m) {            /* mathematical (non-negative) modulus */
    int r = a % m;
    return r < 0 ? r + m : r;
}

/* ---------------------------------------------------------------------------------------------
 * Literal definitions (SURVEY 8(c) pseudo-code, lines a1 and a3)
 * ------------------------------------------------------------------------------------------- */

/* a1: b(y,x) = sum_{j,i} P[j][i] * psi((y-(j-c)) mod H, (x-(i-c)) mod W)      [psi * P_v, PAPER.md:79] */
void mvd_oracle_blur_literal(const double* psi, const float* P, int K, int W, int H, double* b) {
    const int c = (K - 1) / 2;
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            double s = 0.0;
            for (int j = 0; j < K; ++j)
                for (int i = 0; i < K; ++i)
                    s += (double)P[j * K + i] * psi[(size_t)pmod(y - (j - c), H) * W + pmod(x - (i - c), W)];
            b[(size_t)y * W + x] = s;
        }
}

/* a3: q(y,x) = sum_{j,i} P[j][i] * r((y+(j-c)) mod H, (x+(i-c)) mod W)        [r * P_v^*, PAPER.md:79,:118] */
void mvd_oracle_backproject_literal(const double* r, const float* P, int K, int W, int H, double* q) {
    const int c = (K - 1) / 2;
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            double s = 0.0;
            for (int j = 0; j < K; ++j)
                for (int i = 0; i < K; ++i)
                    s += (double)P[j * K + i] * r[(size_t)pmod(y + (j - c), H) * W + pmod(x + (i - c), W)];
            q[(size_t)y * W + x] = s;
        }
}

/* ---------------------------------------------------------------------------------------------
 * Same sums from a wrap-padded copy: pad[yy][xx] = src[(yy-c) mod H][(xx-c) mod W],
 * yy in [0, H+K-1), xx in [0, W+K-1).
 * ------------------------------------------------------------------------------------------- */
static void wrap_pad(const double* src, int K, int W, int H, double* pad) {
    const int c = (K - 1) / 2, PW = W + K - 1, PH = H + K - 1;
    for (int yy = 0; yy < PH; ++yy) {
        const double* row = src + (size_t)pmod(yy - c, H) * W;
        double* prow = pad + (size_t)yy * PW;
        for (int xx = 0; xx < PW; ++xx) prow[xx] = row[pmod(xx - c, W)];
    }
}

/* a1 from the padded copy: psi[y-(j-c)][x-(i-c)] = pad[y-j+2c][x-i+2c] */
static void blur_padded(const double* pad, const float* P, int K, int W, int H, double* b) {
    const int PW = W + K - 1, c2 = K - 1;
    for (int y = 0; y < H; ++y) {
        double* out = b + (size_t)y * W;
        for (int x = 0; x < W; ++x) out[x] = 0.0;
        for (int j = 0; j < K; ++j) {
            const double* prow = pad + (size_t)(y - j + c2) * PW;
            for (int i = 0; i < K; ++i) {
                const double w = (double)P[j * K + i];
                const double* in = prow + (c2 - i);
                for (int x = 0; x < W; ++x) out[x] += w * in[x];
            }
        }
    }
}

/* a3 from the padded copy: r[y+(j-c)][x+(i-c)] = pad[y+j][x+i] */
static void backproject_padded(const double* pad, const float* P, int K, int W, int H, double* q) {
    const int PW = W + K - 1;
    for (int y = 0; y < H; ++y) {
        double* out = q + (size_t)y * W;
        for (int x = 0; x < W; ++x) out[x] = 0.0;
        for (int j = 0; j < K; ++j) {
            const double* prow = pad + (size_t)(y + j) * PW;
            for (int i = 0; i < K; ++i) {
                const double w = (double)P[j * K + i];
                const double* in = prow + i;
                for (int x = 0; x < W; ++x) out[x] += w * in[x];
            }
        }
    }
}

void mvd_oracle_blur(const double* psi, const float* P, int K, int W, int H, double* b) {
    double* pad = (double*)malloc(sizeof(double) * (size_t)(W + K - 1) * (H + K - 1));
    wrap_pad(psi, K, W, H, pad);
    blur_padded(pad, P, K, W, H, b);
    free(pad);
}

void mvd_oracle_backproject(const double* r, const float* P, int K, int W, int H, double* q) {
    double* pad = (double*)malloc(sizeof(double) * (size_t)(W + K - 1) * (H + K - 1));
    wrap_pad(r, K, W, H, pad);
    backproject_padded(pad, P, K, W, H, q);
    free(pad);
}

/* ---------------------------------------------------------------------------------------------
 * One plane: a0 .. a5 of SURVEY 8(a).  `views` points at view 0 of this plane; view v of the same
 * plane is `view_stride` uint16 elements further on.  trace (nullable) receives psi after every
 * view update: [T*V][H][W].
 * ------------------------------------------------------------------------------------------- */
/* xs (nullable): explicit back-projectors X_v, float [V][KX][KX] ("the implemented
 * variants all used the following formula, but replaced X"): step a3 becomes the TRUE periodic
 * convolution q = r * X_v, q(x) = sum_u X_v(u) r(x - u), index (j,i) <-> u = (j-cx, i-cx).
 * xs == NULL is the "Independent" variant X = P_v^* (correlation with P_v). */
/* weights (nullable): per-view, per-pixel weights w_v in [0, 1], float, same layout as the views
 * (PAPER.md:88 lists "weights, float, 4 v bytes/pixel" and never says what they do; READING W1, DESIGN.md
 * section 2, parity unpinned): the weight blends view v's multiplicative correction with the identity,
 *     a4w   psi <- psi . (w_v q + (1 - w_v)),
 * so w_v = 1 is the unweighted update (bit for bit: 1 q + 0) and w_v = 0 leaves the pixel untouched by view v
 * (a registered view that does not cover it).  a0 (the mean of the views) and a1-a3 are unchanged. */
static void rl_plane(int W, int H, int V, const float* psfs, int K, int T, double eps,
                     const uint16_t* views, size_t view_stride, double* psi, double* trace,
                     int literal, const float* xs, int KX, const float* weights, size_t w_view_stride) {
    const size_t npx = (size_t)W * H;
    double* b = (double*)malloc(sizeof(double) * npx);
    double* r = (double*)malloc(sizeof(double) * npx);
    double* q = (double*)malloc(sizeof(double) * npx);

    /* a0: psi_0 = mean of the views (A7) */
    for (size_t p = 0; p < npx; ++p) {
        double s = 0.0;
        for (int v = 0; v < V; ++v) s += (double)views[(size_t)v * view_stride + p];
        psi[p] = s / (double)V;
    }
    for (int t = 0; t < T; ++t) {                 /* a5: nIterations RL steps */
        for (int v = 0; v < V; ++v) {             /* A4: index order; A1: sequential */
            const float* P = psfs + (size_t)v * K * K;
            const uint16_t* phi = views + (size_t)v * view_stride;
            if (literal) mvd_oracle_blur_literal(psi, P, K, W, H, b);            /* a1 */
            else         mvd_oracle_blur(psi, P, K, W, H, b);
            for (size_t p = 0; p < npx; ++p) {                                   /* a2 (A6) */
                const double den = b[p] > eps ? b[p] : eps;
                r[p] = (double)phi[p] / den;
            }
            if (xs) {                                                            /* a3 with X_v given */
                const float* X = xs + (size_t)v * KX * KX;
                if (literal) mvd_oracle_blur_literal(r, X, KX, W, H, q);
                else         mvd_oracle_blur(r, X, KX, W, H, q);
            } else if (literal) mvd_oracle_backproject_literal(r, P, K, W, H, q); /* a3, X = P_v^* */
            else         mvd_oracle_backproject(r, P, K, W, H, q);
            if (weights) {                                                       /* a4w (reading W1) */
                const float* w = weights + (size_t)v * w_view_stride;
                for (size_t p = 0; p < npx; ++p)
                    psi[p] = psi[p] * ((double)w[p] * q[p] + (1.0 - (double)w[p]));
            } else {
                for (size_t p = 0; p < npx; ++p) psi[p] = psi[p] * q[p];         /* a4 */
            }
            if (trace) memcpy(trace + ((size_t)t * V + v) * npx, psi, sizeof(double) * npx);
        }
    }
    free(b); free(r); free(q);
}

/* ---------------------------------------------------------------------------------------------
 * Public entry points (C linkage, loaded through ctypes by oracle/mvd_oracle.py).
 * Layouts as include/mvd.h: psfs float [V][K][K]; views uint16 [V][N][H][W]; out double [N][H][W].
 * ------------------------------------------------------------------------------------------- */
static int check_args(int W, int H, int V, const float* psfs, int K, int T, double eps,
                      const uint16_t* views, double* out, int N) {
    if (!psfs || !views || !out) return -1;
    if (W < 1 || H < 1 || V < 1 || N < 1 || T < 0) return -1;
    if (K < 1 || (K % 2) == 0) return -1;
    if (!(eps > 0.0) || !isfinite(eps)) return -1;
    return 0;
}

typedef struct {
    int W, H, V, K, T, N, literal;
    double eps;
    const float* xs;
    int KX;
    const float* weights;
    const float* psfs;
    const uint16_t* views;
    double* out;
    int p_begin, p_end;
} job_t;

static void* worker(void* arg) {
    job_t* j = (job_t*)arg;
    const size_t npx = (size_t)j->W * j->H;
    for (int p = j->p_begin; p < j->p_end; ++p)
        rl_plane(j->W, j->H, j->V, j->psfs, j->K, j->T, j->eps, j->views + (size_t)p * npx,
                 (size_t)j->N * npx, j->out + (size_t)p * npx, NULL, j->literal, j->xs, j->KX,
                 j->weights ? j->weights + (size_t)p * npx : NULL, (size_t)j->N * npx);
    return NULL;
}

static int run(int W, int H, int V, const float* psfs, int K, int T, double eps,
               const uint16_t* views, double* out, int N, int n_threads, int literal,
               const float* xs, int KX, const float* weights) {
    int rc = check_args(W, H, V, psfs, K, T, eps, views, out, N);
    if (rc) return rc;
    if (xs && (KX < 1 || (KX % 2) == 0)) return -1;
    if (n_threads < 1) n_threads = 1;
    if (n_threads > N) n_threads = N;           /* parallel over planes only */
    job_t* jobs = (job_t*)calloc((size_t)n_threads, sizeof(job_t));
    pthread_t* th = (pthread_t*)calloc((size_t)n_threads, sizeof(pthread_t));
    for (int k = 0; k < n_threads; ++k) {
        job_t j = {W, H, V, K, T, N, literal, eps, xs, KX, weights, psfs, views, out,
                   (int)((long long)N * k / n_threads), (int)((long long)N * (k + 1) / n_threads)};
        jobs[k] = j;
    }
    for (int k = 1; k < n_threads; ++k) pthread_create(&th[k], NULL, worker, &jobs[k]);
    worker(&jobs[0]);
    for (int k = 1; k < n_threads; ++k) pthread_join(th[k], NULL);
    free(jobs); free(th);
    return 0;
}

int mvd_oracle(int W, int H, int V, const float* psfs, int K, int T, double eps,
               const uint16_t* views, double* out, int N, int n_threads) {
    return run(W, H, V, psfs, K, T, eps, views, out, N, n_threads, 0, NULL, 0, NULL);
}

/* The same iteration with the back-projectors X_v given explicitly: xs float [V][KX][KX], KX odd. */
int mvd_oracle_x(int W, int H, int V, const float* psfs, int K, const float* xs, int KX, int T,
                 double eps, const uint16_t* views, double* out, int N, int n_threads, int literal) {
    if (!xs) return -1;
    return run(W, H, V, psfs, K, T, eps, views, out, N, n_threads, literal, xs, KX, NULL);
}

/* The same iteration with per-view weights (reading W1 above): weights float [V][N][H][W], finite, in [0, 1];
 * xs (nullable) as in mvd_oracle_x. */
int mvd_oracle_w(int W, int H, int V, const float* psfs, int K, const float* xs, int KX, int T, double eps,
                 const uint16_t* views, const float* weights, double* out, int N, int n_threads, int literal) {
    if (!weights) return -1;
    const size_t nw = (size_t)V * N * H * W;
    for (size_t k = 0; k < nw; ++k)
        if (!(weights[k] >= 0.f && weights[k] <= 1.f)) return -1;
    return run(W, H, V, psfs, K, T, eps, views, out, N, n_threads, literal, xs, KX, weights);
}

int mvd_oracle_literal(int W, int H, int V, const float* psfs, int K, int T, double eps,
                       const uint16_t* views, double* out, int N, int n_threads) {
    return run(W, H, V, psfs, K, T, eps, views, out, N, n_threads, 1, NULL, 0, NULL);
}

/* One plane (views [V][H][W]); trace [T*V][H][W] = psi after every view update; out [H][W]. */
int mvd_oracle_trace(int W, int H, int V, const float* psfs, int K, int T, double eps,
                     const uint16_t* views, double* out, double* trace) {
    int rc = check_args(W, H, V, psfs, K, T, eps, views, out, 1);
    if (rc) return rc;
    rl_plane(W, H, V, psfs, K, T, eps, views, (size_t)W * H, out, trace, 0, NULL, 0, NULL, 0);
    return 0;
}
