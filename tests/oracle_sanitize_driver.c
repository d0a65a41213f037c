/* Driver for tests/test_oracle_sanitized.py: every public entry point of oracle/mvd_oracle.c on tiny seeded inputs, built
 * with -fsanitize=address,undefined.  Shapes include a PSF wider than the plane (wrap-around more
 * than once), odd sizes and more threads than planes.  Prints one checksum per call; exits non-zero on a bad return
 * code or when the literal and the padded formulations of the same iteration disagree. */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

void mvd_oracle_blur_literal(const double*, const float*, int, int, int, double*);
void mvd_oracle_backproject_literal(const double*, const float*, int, int, int, double*);
void mvd_oracle_blur(const double*, const float*, int, int, int, double*);
void mvd_oracle_backproject(const double*, const float*, int, int, int, double*);
int mvd_oracle(int, int, int, const float*, int, int, double, const uint16_t*, double*, int, int);
int mvd_oracle_x(int, int, int, const float*, int, const float*, int, int, double, const uint16_t*, double*, int, int, int);
int mvd_oracle_w(int, int, int, const float*, int, const float*, int, int, double, const uint16_t*, const float*, double*,
                 int, int, int);
int mvd_oracle_literal(int, int, int, const float*, int, int, double, const uint16_t*, double*, int, int);
int mvd_oracle_trace(int, int, int, const float*, int, int, double, const uint16_t*, double*, double*);

static uint32_t s = 12345u;
static double rnd(void) { s = s * 1664525u + 1013904223u; return (s >> 8) / 16777216.0; }

static double sum(const double* a, size_t n) { double t = 0; for (size_t k = 0; k < n; ++k) t += a[k]; return t; }
static double maxdiff(const double* a, const double* b, size_t n) {
    double m = 0;
    for (size_t k = 0; k < n; ++k) { double d = fabs(a[k] - b[k]) / (fabs(b[k]) + 1e-300); if (d > m) m = d; }
    return m;
}

static int one(int W, int H, int V, int K, int KX, int T, int N, int threads) {
    const size_t npx = (size_t)W * H;
    float* psfs = malloc(sizeof(float) * V * K * K);
    float* xs = malloc(sizeof(float) * V * KX * KX);
    float* wts = malloc(sizeof(float) * V * N * npx);
    uint16_t* views = malloc(sizeof(uint16_t) * V * N * npx);
    double* o1 = malloc(sizeof(double) * N * npx);
    double* o2 = malloc(sizeof(double) * N * npx);
    double* tr = malloc(sizeof(double) * (T ? T : 1) * V * npx);
    for (int v = 0; v < V; ++v) {
        double t = 0;
        for (int k = 0; k < K * K; ++k) t += (psfs[v * K * K + k] = (float)rnd());
        for (int k = 0; k < K * K; ++k) psfs[v * K * K + k] /= (float)t;
        t = 0;
        for (int k = 0; k < KX * KX; ++k) t += (xs[v * KX * KX + k] = (float)rnd());
        for (int k = 0; k < KX * KX; ++k) xs[v * KX * KX + k] /= (float)t;
    }
    for (size_t k = 0; k < (size_t)V * N * npx; ++k) { views[k] = (uint16_t)(rnd() * 4000.0); wts[k] = (float)rnd(); }
    int bad = 0;
    bad |= mvd_oracle(W, H, V, psfs, K, T, 1e-6, views, o1, N, threads);
    bad |= mvd_oracle_literal(W, H, V, psfs, K, T, 1e-6, views, o2, N, threads);
    if (maxdiff(o1, o2, N * npx) > 1e-10) { fprintf(stderr, "literal != padded (plain)\n"); bad = 1; }
    printf("plain   %dx%d V%d K%d T%d N%d: %.12g\n", W, H, V, K, T, N, sum(o1, N * npx));
    bad |= mvd_oracle_x(W, H, V, psfs, K, xs, KX, T, 1e-6, views, o1, N, threads, 0);
    bad |= mvd_oracle_x(W, H, V, psfs, K, xs, KX, T, 1e-6, views, o2, N, threads, 1);
    if (maxdiff(o1, o2, N * npx) > 1e-10) { fprintf(stderr, "literal != padded (x)\n"); bad = 1; }
    printf("x       KX%d: %.12g\n", KX, sum(o1, N * npx));
    bad |= mvd_oracle_w(W, H, V, psfs, K, NULL, 0, T, 1e-6, views, wts, o1, N, threads, 0);
    bad |= mvd_oracle_w(W, H, V, psfs, K, xs, KX, T, 1e-6, views, wts, o2, N, threads, 1);
    printf("weights: %.12g %.12g\n", sum(o1, N * npx), sum(o2, N * npx));
    bad |= mvd_oracle_trace(W, H, V, psfs, K, T, 1e-6, views, o1, tr);
    if (T > 0 && maxdiff(o1, tr + ((size_t)T * V - 1) * npx, npx) != 0.0) { fprintf(stderr, "trace end != out\n"); bad = 1; }
    printf("trace  : %.12g\n", sum(o1, npx));
    mvd_oracle_blur(o1, psfs, K, W, H, o2);
    mvd_oracle_blur_literal(o1, psfs, K, W, H, tr);
    if (maxdiff(o2, tr, npx) > 1e-12) { fprintf(stderr, "blur literal != padded\n"); bad = 1; }
    mvd_oracle_backproject(o1, psfs, K, W, H, o2);
    mvd_oracle_backproject_literal(o1, psfs, K, W, H, tr);
    if (maxdiff(o2, tr, npx) > 1e-12) { fprintf(stderr, "backproject literal != padded\n"); bad = 1; }
    free(psfs); free(xs); free(wts); free(views); free(o1); free(o2); free(tr);
    return bad;
}

int main(void) {
    int bad = 0;
    bad |= one(16, 12, 2, 5, 3, 2, 3, 2);
    bad |= one(7, 5, 3, 9, 11, 1, 2, 8);      /* PSF and back-projector wider than the plane; threads > planes */
    bad |= one(1, 1, 1, 3, 1, 3, 1, 1);       /* one voxel */
    bad |= one(33, 9, 4, 1, 1, 0, 5, 3);      /* T = 0: the mean of the views */
    /* argument checks return -1 and touch nothing */
    double o;
    uint16_t v = 1;
    float p = 1.f;
    if (mvd_oracle(1, 1, 1, &p, 2, 1, 1e-6, &v, &o, 1, 1) != -1) bad = 1;       /* even K */
    if (mvd_oracle(1, 1, 1, &p, 1, 1, 0.0, &v, &o, 1, 1) != -1) bad = 1;        /* eps = 0 */
    if (mvd_oracle(1, 1, 1, NULL, 1, 1, 1e-6, &v, &o, 1, 1) != -1) bad = 1;
    return bad ? 1 : 0;
}
