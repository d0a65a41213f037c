// mvd_fft_kernels.cuh -- hand-written batched FFT convolution kernels of libmvd's FFT engine (sm_100a).
//
// Two planes are packed into one complex plane, z = psi_a + i psi_b.  Convolution with a REAL kernel
// is linear and real, so  z (*) P = (psi_a (*) P) + i (psi_b (*) P):  one complex 2D FFT serves two
// planes, no real-FFT post-processing, no Hermitian bookkeeping.  With X = FFT2(z) and the optical
// transfer function O_v = FFT2(P_v embedded with its centre at the origin) / (W H):
//     a1  b = IFFT2(X . O_v)              (periodic convolution,  PAPER.md:79  "psi * P_v")
//     a3  q = IFFT2(FFT2(r) . conj O_v)   (periodic correlation,  PAPER.md:79, :118  "* P_v^*", P real)
// The 2D transforms are split into row passes (x, contiguous) and column passes (z, strided), and the
// pointwise steps are fused into them:
//     rows_first   a0: psi_0 = mean_v phi_v -> Z;  row FFT -> S
//     cols         column FFT, . O_v (or conj O_v), inverse column FFT          S -> S   (twice per view update)
//     rows_ratio   inverse row FFT -> b;  a2: r = phi_v / max(b, eps);  row FFT  S -> S
//     rows_update  inverse row FFT -> q;  a4: psi <- psi . q  (Z, or the output after the last update);
//                  row FFT of the new psi -> S
//
// One FFT of length N = R0 R1 ... is a Stockham autosort: every thread keeps E elements in registers,
// element e of thread t being position t + TPF e (TPF = N / E threads per FFT) -- the layout every
// stage reads, and the layout the last stage leaves its results in, so global loads, the pointwise
// steps and global stores all use it directly and only S-1 exchanges per FFT go through shared memory.
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace mvdfft {

// ---------------------------------------------------------------------------------------------
// TMA (cp.async.bulk) + mbarrier plumbing: inputs of the next work item stream into shared memory
// while the current one is transformed
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!done);
}
// 1D bulk copy global -> shared (16-byte aligned, size a multiple of 16); SASS UBLKCP
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// 2D tiled tensor copy global -> shared; SASS UTMALDG
__device__ __forceinline__ void tma_2d_g2s(void* dst, const CUtensorMap* map, int x, int y, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(x), "r"(y), "r"(smem_u32(bar)) : "memory");
}
__host__ __device__ constexpr size_t align_up(size_t n, size_t a) { return (n + a - 1) / a * a; }

// ---------------------------------------------------------------------------------------------
// complex arithmetic on packed f32x2 (SASS FADD2 / FMUL2 / FFMA2 on sm_100a)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ float2 add2(float2 a, float2 b) {
    float2 r;
    asm("{ .reg .b64 ra, rb, rc; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; add.rn.f32x2 rc, ra, rb; "
        "mov.b64 {%0,%1}, rc; }" : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 sub2(float2 a, float2 b) {
    float2 r;
    asm("{ .reg .b64 ra, rb, rc; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; sub.rn.f32x2 rc, ra, rb; "
        "mov.b64 {%0,%1}, rc; }" : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 mul2(float2 a, float2 b) {
    float2 r;
    asm("{ .reg .b64 ra, rb, rc; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; mul.rn.f32x2 rc, ra, rb; "
        "mov.b64 {%0,%1}, rc; }" : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) {
    float2 r;
    asm("{ .reg .b64 ra, rb, rc, rd; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; mov.b64 rc, {%6,%7}; "
        "fma.rn.f32x2 rd, ra, rb, rc; mov.b64 {%0,%1}, rd; }"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
    return r;
}
__device__ __forceinline__ float2 scale2(float2 a, float s) { return mul2(a, make_float2(s, s)); }
// a * w = a w.x + (i a) w.y: the two halves of w enter as broadcast scalars and i a = (-a.y, a.x) as a swapped, half-negated
// view of a -- operand modifiers of FFMA2 / FMUL2 in SASS, so a twiddle loaded from shared memory needs no extra
// instruction to build (-w.y, w.x)
__device__ __forceinline__ float2 cmul(float2 a, float2 w) {
    return fma2(a, make_float2(w.x, w.x), mul2(make_float2(-a.y, a.x), make_float2(w.y, w.y)));
}
// a * conj(w) = a w.x + (-i a) w.y
__device__ __forceinline__ float2 cmulc(float2 a, float2 w) {
    return fma2(a, make_float2(w.x, w.x), mul2(make_float2(a.y, -a.x), make_float2(w.y, w.y)));
}
// x / d for d in [eps, 2^126): reciprocal on the special-function unit and one multiply (2 ulp), without the range
// handling __fdividef carries for huge denominators
__device__ __forceinline__ float div_approx(float x, float d) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(d));
    return x * r;
}
// a * (-i) for the forward transform (DIR < 0), a * (+i) for the inverse
template <int DIR>
__device__ __forceinline__ float2 rot90(float2 a) {
    return DIR < 0 ? make_float2(a.y, -a.x) : make_float2(-a.y, a.x);
}

// ---------------------------------------------------------------------------------------------
// in-register DFTs, natural order in and out: v[q] <- sum_m v[m] exp(DIR 2 pi i m q / R)
// ---------------------------------------------------------------------------------------------
template <int R, int DIR>
struct Bfly;

template <int DIR>
struct Bfly<2, DIR> {
    static __device__ __forceinline__ void run(float2* v) {
        const float2 a = v[0];
        v[0] = add2(a, v[1]);
        v[1] = sub2(a, v[1]);
    }
};

template <int DIR>
struct Bfly<3, DIR> {
    static __device__ __forceinline__ void run(float2* v) {
        const float2 t1 = add2(v[1], v[2]);
        const float2 m = fma2(t1, make_float2(-0.5f, -0.5f), v[0]);
        const float2 s = rot90<DIR>(scale2(sub2(v[1], v[2]), 0.86602540378443864676f));
        v[0] = add2(v[0], t1);
        v[1] = add2(m, s);
        v[2] = sub2(m, s);
    }
};

template <int DIR>
struct Bfly<4, DIR> {
    static __device__ __forceinline__ void run(float2* v) {
        const float2 a0 = add2(v[0], v[2]), a1 = sub2(v[0], v[2]);
        const float2 a2 = add2(v[1], v[3]), a3 = rot90<DIR>(sub2(v[1], v[3]));
        v[0] = add2(a0, a2);
        v[2] = sub2(a0, a2);
        v[1] = add2(a1, a3);
        v[3] = sub2(a1, a3);
    }
};

template <int DIR>
struct Bfly<5, DIR> {
    static __device__ __forceinline__ void run(float2* v) {
        constexpr float c1 = 0.30901699437494742410f, c2 = -0.80901699437494742410f;   // cos 72, cos 144
        constexpr float s1 = 0.95105651629515357212f, s2 = 0.58778525229247312917f;    // sin 72, sin 144
        const float2 a1 = add2(v[1], v[4]), a2 = add2(v[2], v[3]);
        const float2 b1 = sub2(v[1], v[4]), b2 = sub2(v[2], v[3]);
        const float2 x0 = v[0];
        v[0] = add2(x0, add2(a1, a2));
        const float2 e1 = fma2(a2, make_float2(c2, c2), fma2(a1, make_float2(c1, c1), x0));
        const float2 e2 = fma2(a2, make_float2(c1, c1), fma2(a1, make_float2(c2, c2), x0));
        const float2 d1 = rot90<DIR>(fma2(b2, make_float2(s2, s2), scale2(b1, s1)));
        const float2 d2 = rot90<DIR>(fma2(b2, make_float2(-s1, -s1), scale2(b1, s2)));
        v[1] = add2(e1, d1);
        v[4] = sub2(e1, d1);
        v[2] = add2(e2, d2);
        v[3] = sub2(e2, d2);
    }
};

// a * exp(DIR i pi / 4) and a * exp(DIR 3 i pi / 4)
template <int DIR>
__device__ __forceinline__ float2 rot45(float2 a) {
    constexpr float h = 0.70710678118654752440f;
    return scale2(add2(a, rot90<DIR>(a)), h);
}
template <int DIR>
__device__ __forceinline__ float2 rot135(float2 a) {
    constexpr float h = 0.70710678118654752440f;
    return scale2(sub2(rot90<DIR>(a), a), h);
}

template <int DIR>
struct Bfly<8, DIR> {
    static __device__ __forceinline__ void run(float2* v) {
        // radix-2 split (decimation in frequency), then two radix-4 transforms
        float2 a[4], b[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            a[k] = add2(v[k], v[k + 4]);
            b[k] = sub2(v[k], v[k + 4]);
        }
        b[1] = rot45<DIR>(b[1]);
        b[2] = rot90<DIR>(b[2]);
        b[3] = rot135<DIR>(b[3]);
        Bfly<4, DIR>::run(a);
        Bfly<4, DIR>::run(b);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            v[2 * q] = a[q];
            v[2 * q + 1] = b[q];
        }
    }
};

template <int DIR>
struct Bfly<16, DIR> {
    static __device__ __forceinline__ void run(float2* v) {
        // 16 = 4 x 4: n = n1 + 4 n2, f = f2 + 4 f1
        constexpr float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f;   // cos, sin of pi/8
        constexpr float h = 0.70710678118654752440f;
        float2 a[4][4];
#pragma unroll
        for (int n1 = 0; n1 < 4; ++n1) {
            float2 t[4] = {v[n1], v[n1 + 4], v[n1 + 8], v[n1 + 12]};
            Bfly<4, DIR>::run(t);
#pragma unroll
            for (int f2 = 0; f2 < 4; ++f2) a[n1][f2] = t[f2];
        }
        // twiddles w16^(n1 f2), w16 = exp(DIR 2 pi i / 16)
        const float sg = DIR < 0 ? -1.f : 1.f;
        const float2 w1 = make_float2(c1, sg * s1), w2 = make_float2(h, sg * h), w3 = make_float2(s1, sg * c1);
        const float2 w6 = make_float2(-h, sg * h), w9 = make_float2(-c1, -sg * s1);
        a[1][1] = cmul(a[1][1], w1);
        a[1][2] = cmul(a[1][2], w2);
        a[1][3] = cmul(a[1][3], w3);
        a[2][1] = cmul(a[2][1], w2);
        a[2][2] = rot90<DIR>(a[2][2]);
        a[2][3] = cmul(a[2][3], w6);
        a[3][1] = cmul(a[3][1], w3);
        a[3][2] = cmul(a[3][2], w6);
        a[3][3] = cmul(a[3][3], w9);
#pragma unroll
        for (int f2 = 0; f2 < 4; ++f2) {
            float2 t[4] = {a[0][f2], a[1][f2], a[2][f2], a[3][f2]};
            Bfly<4, DIR>::run(t);
#pragma unroll
            for (int f1 = 0; f1 < 4; ++f1) v[f2 + 4 * f1] = t[f1];
        }
    }
};

// cos / sin of 2 pi k / 32 as compile-time constants (k any integer)
__host__ __device__ constexpr float cos32(int k) {
    constexpr float C[9] = {1.0f, 0.98078528040323044913f, 0.92387953251128675613f, 0.83146961230254523708f,
                            0.70710678118654752440f, 0.55557023301960222474f, 0.38268343236508977173f,
                            0.19509032201612826785f, 0.0f};
    k = ((k % 32) + 32) % 32;
    if (k > 16) k = 32 - k;
    return k > 8 ? -C[16 - k] : C[k];
}
__host__ __device__ constexpr float sin32(int k) { return cos32(k - 8); }

template <int DIR>
struct Bfly<32, DIR> {
    static __device__ __forceinline__ void run(float2* v) {
        // 32 = 8 x 4: n = n1 + 4 n2 (n1 < 4, n2 < 8), f = f2 + 8 f1 (f2 < 8, f1 < 4)
        float2 a[4][8];
#pragma unroll
        for (int n1 = 0; n1 < 4; ++n1) {
            float2 t[8];
#pragma unroll
            for (int n2 = 0; n2 < 8; ++n2) t[n2] = v[n1 + 4 * n2];
            Bfly<8, DIR>::run(t);
#pragma unroll
            for (int f2 = 0; f2 < 8; ++f2) a[n1][f2] = t[f2];
        }
        // twiddles w32^(n1 f2), w32 = exp(DIR 2 pi i / 32)
#pragma unroll
        for (int n1 = 1; n1 < 4; ++n1) {
#pragma unroll
            for (int f2 = 1; f2 < 8; ++f2) {
                const int k = n1 * f2;
                if (k == 8) a[n1][f2] = rot90<DIR>(a[n1][f2]);
                else if (k == 4) a[n1][f2] = rot45<DIR>(a[n1][f2]);
                else if (k == 12) a[n1][f2] = rot135<DIR>(a[n1][f2]);
                else a[n1][f2] = cmul(a[n1][f2], make_float2(cos32(k), (DIR < 0 ? -1.f : 1.f) * sin32(k)));
            }
        }
#pragma unroll
        for (int f2 = 0; f2 < 8; ++f2) {
            float2 t[4] = {a[0][f2], a[1][f2], a[2][f2], a[3][f2]};
            Bfly<4, DIR>::run(t);
#pragma unroll
            for (int f1 = 0; f1 < 4; ++f1) v[f2 + 8 * f1] = t[f1];
        }
    }
};

// cos / sin of 2 pi k / 40 as compile-time constants (k any integer)
__host__ __device__ constexpr float cos40(int k) {
    constexpr float C[11] = {1.0f, 0.98768834059513777035f, 0.95105651629515357212f, 0.89100652418836786236f,
                             0.80901699437494742410f, 0.70710678118654752440f, 0.58778525229247312917f,
                             0.45399049973954679156f, 0.30901699437494742410f, 0.15643446504023086901f, 0.0f};
    k = ((k % 40) + 40) % 40;
    if (k > 20) k = 40 - k;
    return k > 10 ? -C[20 - k] : C[k];
}
__host__ __device__ constexpr float sin40(int k) { return cos40(k - 10); }

// Composite butterfly of length RA * 5 (RA = 4 or 8): n = n1 + 5 n2 (n1 < 5, n2 < RA), f = f2 + RA f1;
// RA-point transforms over n2, twiddles w^(n1 f2) with w = exp(DIR 2 pi i / (5 RA)), 5-point transforms over n1.
template <int RA, int DIR>
struct BflyTimes5 {
    static __device__ __forceinline__ void run(float2* v) {
        constexpr int N = 5 * RA, Q = 40 / N;   // w_N^k = w_40^(Q k)
        float2 a[5][RA];
#pragma unroll
        for (int n1 = 0; n1 < 5; ++n1) {
            float2 t[RA];
#pragma unroll
            for (int n2 = 0; n2 < RA; ++n2) t[n2] = v[n1 + 5 * n2];
            Bfly<RA, DIR>::run(t);
#pragma unroll
            for (int f2 = 0; f2 < RA; ++f2) a[n1][f2] = t[f2];
        }
#pragma unroll
        for (int n1 = 1; n1 < 5; ++n1) {
#pragma unroll
            for (int f2 = 1; f2 < RA; ++f2) {
                const int k = Q * n1 * f2;
                if (k % 40 == 10) a[n1][f2] = rot90<DIR>(a[n1][f2]);
                else if (k % 40 == 5) a[n1][f2] = rot45<DIR>(a[n1][f2]);
                else if (k % 40 == 15) a[n1][f2] = rot135<DIR>(a[n1][f2]);
                else a[n1][f2] = cmul(a[n1][f2], make_float2(cos40(k), (DIR < 0 ? -1.f : 1.f) * sin40(k)));
            }
        }
#pragma unroll
        for (int f2 = 0; f2 < RA; ++f2) {
            float2 t[5] = {a[0][f2], a[1][f2], a[2][f2], a[3][f2], a[4][f2]};
            Bfly<5, DIR>::run(t);
#pragma unroll
            for (int f1 = 0; f1 < 5; ++f1) v[f2 + RA * f1] = t[f1];
        }
    }
};
template <int DIR>
struct Bfly<20, DIR> : BflyTimes5<4, DIR> {};
template <int DIR>
struct Bfly<40, DIR> : BflyTimes5<8, DIR> {};

// cos / sin of 2 pi k / 24 as compile-time constants (k any integer)
__host__ __device__ constexpr float cos24(int k) {
    constexpr float C[7] = {1.0f, 0.96592582628906828675f, 0.86602540378443864676f, 0.70710678118654752440f, 0.5f,
                            0.25881904510252076235f, 0.0f};
    k = ((k % 24) + 24) % 24;
    if (k > 12) k = 24 - k;
    return k > 6 ? -C[12 - k] : C[k];
}
__host__ __device__ constexpr float sin24(int k) { return cos24(k - 6); }

// 24 = 8 x 3: n = n1 + 3 n2 (n1 < 3, n2 < 8), f = f2 + 8 f1; 8-point transforms over n2, twiddles w24^(n1 f2), 3-point
// transforms over n1
template <int DIR>
struct Bfly<24, DIR> {
    static __device__ __forceinline__ void run(float2* v) {
        float2 a[3][8];
#pragma unroll
        for (int n1 = 0; n1 < 3; ++n1) {
            float2 t[8];
#pragma unroll
            for (int n2 = 0; n2 < 8; ++n2) t[n2] = v[n1 + 3 * n2];
            Bfly<8, DIR>::run(t);
#pragma unroll
            for (int f2 = 0; f2 < 8; ++f2) a[n1][f2] = t[f2];
        }
#pragma unroll
        for (int n1 = 1; n1 < 3; ++n1) {
#pragma unroll
            for (int f2 = 1; f2 < 8; ++f2) {
                const int k = n1 * f2;
                if (k % 24 == 6) a[n1][f2] = rot90<DIR>(a[n1][f2]);
                else if (k % 24 == 3) a[n1][f2] = rot45<DIR>(a[n1][f2]);
                else if (k % 24 == 9) a[n1][f2] = rot135<DIR>(a[n1][f2]);
                else a[n1][f2] = cmul(a[n1][f2], make_float2(cos24(k), (DIR < 0 ? -1.f : 1.f) * sin24(k)));
            }
        }
#pragma unroll
        for (int f2 = 0; f2 < 8; ++f2) {
            float2 t[3] = {a[0][f2], a[1][f2], a[2][f2]};
            Bfly<3, DIR>::run(t);
#pragma unroll
            for (int f1 = 0; f1 < 3; ++f1) v[f2 + 8 * f1] = t[f1];
        }
    }
};

// cos / sin of 2 pi k / 25 as compile-time constants (k any integer)
__host__ __device__ constexpr float cos25(int k) {
    constexpr float C[13] = {1.0f, 0.96858316112863107605f, 0.87630668004386358394f, 0.72896862742141155245f,
                             0.53582679497899654564f, 0.30901699437494745126f, 0.06279051952931352654f,
                             -0.18738131458572460097f, -0.42577929156507271502f, -0.63742398974868974548f,
                             -0.80901699437494734024f, -0.92977648588825134723f, -0.99211470131447776488f};
    k = ((k % 25) + 25) % 25;
    return C[k > 12 ? 25 - k : k];
}
__host__ __device__ constexpr float sin25(int k) {
    constexpr float S[13] = {0.0f, 0.24868988716485479484f, 0.48175367410171532345f, 0.68454710592868861507f,
                             0.84432792550201507531f, 0.95105651629515353118f, 0.99802672842827155897f,
                             0.98228725072868872115f, 0.90482705246601946580f, 0.77051324277578925326f,
                             0.58778525229247324813f, 0.36812455268467814129f, 0.12533323356430453588f};
    k = ((k % 25) + 25) % 25;
    return k > 12 ? -S[25 - k] : S[k];
}
// 25 = 5 x 5: n = n1 + 5 n2, f = f2 + 5 f1; 5-point transforms over n2, twiddles w25^(n1 f2), 5-point transforms over n1
template <int DIR>
struct Bfly<25, DIR> {
    static __device__ __forceinline__ void run(float2* v) {
        float2 a[5][5];
#pragma unroll
        for (int n1 = 0; n1 < 5; ++n1) {
            float2 t[5] = {v[n1], v[n1 + 5], v[n1 + 10], v[n1 + 15], v[n1 + 20]};
            Bfly<5, DIR>::run(t);
#pragma unroll
            for (int f2 = 0; f2 < 5; ++f2) a[n1][f2] = t[f2];
        }
#pragma unroll
        for (int n1 = 1; n1 < 5; ++n1) {
#pragma unroll
            for (int f2 = 1; f2 < 5; ++f2)
                a[n1][f2] = cmul(a[n1][f2], make_float2(cos25(n1 * f2), (DIR < 0 ? -1.f : 1.f) * sin25(n1 * f2)));
        }
#pragma unroll
        for (int f2 = 0; f2 < 5; ++f2) {
            float2 t[5] = {a[0][f2], a[1][f2], a[2][f2], a[3][f2], a[4][f2]};
            Bfly<5, DIR>::run(t);
#pragma unroll
            for (int f1 = 0; f1 < 5; ++f1) v[f2 + 5 * f1] = t[f1];
        }
    }
};

// ---------------------------------------------------------------------------------------------
// plans
// ---------------------------------------------------------------------------------------------
template <int N_, int E_, int R0, int R1 = 1, int R2 = 1, int R3 = 1, int R4 = 1>
struct Plan {
    static constexpr int N = N_, E = E_, TPF = N_ / E_;
    static constexpr int S = 1 + (R1 > 1) + (R2 > 1) + (R3 > 1) + (R4 > 1);
    static constexpr int PAD_DIV = R0;   // row layout: pos -> pos + pos / R0 (conflict-free strided stores)
    static constexpr int NPAD = N_ + N_ / R0;
    __host__ __device__ static constexpr int radix(int s) {
        return s == 0 ? R0 : s == 1 ? R1 : s == 2 ? R2 : s == 3 ? R3 : R4;
    }
    __host__ __device__ static constexpr int ns(int s) {   // product of the radices before stage s
        int p = 1;
        for (int k = 0; k < s; ++k) p *= radix(k);
        return p;
    }
    static_assert(R0 * R1 * R2 * R3 * R4 == N_, "radices must multiply to N");
    static_assert(N_ % E_ == 0 && E_ % R0 == 0 && E_ % R1 == 0 && E_ % R2 == 0 && E_ % R3 == 0 && E_ % R4 == 0,
                  "every radix must divide the per-thread element count");
};

// A plan whose last stage is a radix-2 over elements of the same thread (N = R0 R1 2 with E = R1, TPF = 64):
// the exchange in front of it goes through warp shuffles when the kernel maps logical thread t of an FFT to
// lane ((t >> 5) << 4 | t & 15) of warp (t >> 4) & 1 (fft_stage).
template <class P>
struct ShflTail : P {
    static constexpr bool kShflTail = true;
    static_assert(P::S >= 2 && P::radix(P::S - 1) == 2 && P::radix(P::S - 2) == P::E && P::TPF == 64,
                  "shuffle exchange: one radix-E butterfly per thread in front of a final radix-2 stage, two warps per FFT");
};
template <class P, class = void>
struct ShflTailOf { static constexpr bool value = false; };
template <class P>
struct ShflTailOf<P, decltype((void)P::kShflTail)> { static constexpr bool value = P::kShflTail; };
template <class P>
__host__ __device__ constexpr bool shfl_tail() { return ShflTailOf<P>::value; }

// Row layout: one FFT per TPF threads, exchange region of NPAD float2 per FFT, padded against the
// stride-R0 stores of stage 0.
template <class P>
struct RowAddr {
    int base;
    __device__ __forceinline__ int operator()(int pos) const { return base + pos + pos / P::PAD_DIV; }
};
// Column layout: TC FFTs side by side, position-major: [pos][TC].  With TC = 16 a half-warp touches
// one 128-byte line; narrower tiles shift every group of R0 positions by one slot so that the
// stride-R0 stores of stage 0 from two neighbouring threads land in different bank halves.
template <class P, int TC>
struct ColAddr {
    static constexpr int NPOS = TC < 16 ? P::NPAD : P::N;
    int c;
    __device__ __forceinline__ int operator()(int pos) const {
        return (TC < 16 ? pos + pos / P::PAD_DIV : pos) * TC + c;
    }
};

// Who has to meet at an exchange: the whole CTA (v1 kernels: an FFT's threads are spread over all
// warps), or only the team of NTH threads that owns the FFTs in one exchange region (v2 kernels:
// __syncwarp for teams inside a warp, a named barrier for teams of whole warps).
struct CtaSync {
    __device__ __forceinline__ void operator()() const { __syncthreads(); }
};
template <int NTH>
struct TeamSync {
    int id;   // team index within the CTA (named barrier id - 1); unused for NTH <= 32
    __device__ __forceinline__ void operator()() const {
        if constexpr (NTH <= 32) __syncwarp();
        else asm volatile("bar.sync %0, %1;" ::"r"(id + 1), "n"(NTH) : "memory");
    }
};

// tw: shared memory, [(s-1) * E + e][TPF] for stages s >= 1: exp(-2 pi i m k / (Ns R)) of the element
template <class P, int s, int DIR, class Addr, class Sync>
__device__ __forceinline__ void fft_stage(float2 (&x)[P::E], float2* buf, const float2* tw, int t, const Addr& addr,
                                          const Sync& sync) {
    constexpr int R = P::radix(s), NB = P::E / R, NS = P::ns(s), TPF = P::TPF;
    constexpr bool last = (s == P::S - 1);
    constexpr bool shfl = shfl_tail<P>() && s == P::S - 2;
#pragma unroll
    for (int u = 0; u < NB; ++u) {
        float2 v[R];
#pragma unroll
        for (int m = 0; m < R; ++m) v[m] = x[u + m * NB];
        if (s > 0) {
#pragma unroll
            for (int m = 1; m < R; ++m) {
                const float2 w = tw[((s - 1) * P::E + u + m * NB) * TPF + t];
                v[m] = DIR < 0 ? cmul(v[m], w) : cmulc(v[m], w);
            }
        }
        Bfly<R, DIR>::run(v);
        if (last) {
#pragma unroll
            for (int m = 0; m < R; ++m) x[u + m * NB] = v[m];
        } else if constexpr (shfl) {
            // The exchange in front of a final radix-2 stage only swaps half of the data between threads t and
            // t ^ (N / 2 / R) (here 32): position (t / 32) 1024 + t % 32 + 32 m goes to thread t % 32 + 32 (m & 1),
            // element 16 (t / 32) + m / 2.  The row kernels map those two threads to lanes l and l ^ 16 of one
            // warp (ShflTail), so the exchange is 16 shuffles and no shared memory or barrier.
            const bool hi = (t >> 5) & 1;
#pragma unroll
            for (int i = 0; i < R / 2; ++i) {
                const float2 send = hi ? v[2 * i] : v[2 * i + 1];
                float2 recv;
                recv.x = __shfl_xor_sync(0xffffffffu, send.x, 16);
                recv.y = __shfl_xor_sync(0xffffffffu, send.y, 16);
                x[i] = hi ? recv : v[2 * i];
                x[R / 2 + i] = hi ? v[2 * i + 1] : recv;
            }
        } else {
            const int j = t + u * TPF;
            const int k = j % NS;
            const int base = (j - k) * R + k;
#pragma unroll
            for (int m = 0; m < R; ++m) buf[addr(base + m * NS)] = v[m];
        }
    }
    if (!last && !shfl) {
        sync();
#pragma unroll
        for (int e = 0; e < P::E; ++e) x[e] = buf[addr(t + TPF * e)];
        sync();
    }
}

template <class P, int DIR, class Addr, class Sync = CtaSync>
__device__ __forceinline__ void fft_run(float2 (&x)[P::E], float2* buf, const float2* tw, int t, const Addr& addr,
                                        const Sync& sync = Sync()) {
    fft_stage<P, 0, DIR>(x, buf, tw, t, addr, sync);
    if constexpr (P::S > 1) fft_stage<P, 1, DIR>(x, buf, tw, t, addr, sync);
    if constexpr (P::S > 2) fft_stage<P, 2, DIR>(x, buf, tw, t, addr, sync);
    if constexpr (P::S > 3) fft_stage<P, 3, DIR>(x, buf, tw, t, addr, sync);
    if constexpr (P::S > 4) fft_stage<P, 4, DIR>(x, buf, tw, t, addr, sync);
}

// fft_run in two parts: every stage that exchanges through shared memory, then the last stage, which
// works on registers only -- the exchange region is free from the end of the head onwards.
template <class P, int DIR, class Addr, class Sync>
__device__ __forceinline__ void fft_run_head(float2 (&x)[P::E], float2* buf, const float2* tw, int t, const Addr& addr,
                                             const Sync& sync) {
    if constexpr (P::S > 1) fft_stage<P, 0, DIR>(x, buf, tw, t, addr, sync);
    if constexpr (P::S > 2) fft_stage<P, 1, DIR>(x, buf, tw, t, addr, sync);
    if constexpr (P::S > 3) fft_stage<P, 2, DIR>(x, buf, tw, t, addr, sync);
    if constexpr (P::S > 4) fft_stage<P, 3, DIR>(x, buf, tw, t, addr, sync);
}
template <class P, int DIR, class Addr, class Sync>
__device__ __forceinline__ void fft_run_tail(float2 (&x)[P::E], float2* buf, const float2* tw, int t, const Addr& addr,
                                             const Sync& sync) {
    fft_stage<P, P::S - 1, DIR>(x, buf, tw, t, addr, sync);
}

// ---------------------------------------------------------------------------------------------
// kernels
// ---------------------------------------------------------------------------------------------
// ROWS_UPDATE_W: ROWS_UPDATE with per-view weights (a4w: psi <- psi . (w q + 1 - w), reading W1); the generation-2
// kernel gives every team a second landing zone for the two weight rows, generation 1 reads them directly
enum RowMode { ROWS_FIRST = 0, ROWS_RATIO = 1, ROWS_UPDATE = 2, ROWS_UPDATE_W = 3 };

// final store as uint16: round to nearest even, saturate at 65535; negative round-off and NaN -> 0
__device__ __forceinline__ uint16_t to_u16(float x) { return (uint16_t)__float2uint_rn(fminf(x, 65535.f)); }

struct RowArgs {
    float2* S;               // [pairs][H][W] spectrum (row pass in / out)
    float2* Z;               // [pairs][H][W] psi pairs
    const uint16_t* views;   // view 0 of plane 0 of this chunk
    size_t view_stride;      // elements between views
    size_t view_plane, view_row;   // elements between planes / image rows of a view (ViewLayout)
    float* out;              // [n_planes][H][W]; written when `final` (nullptr when out16 is set)
    uint16_t* out16;         // the same as uint16 (nullptr when out is set)
    const float* weights;    // nullptr, or the weights of view 0 of plane 0 of this chunk, dense [V][n][H][W]
    size_t w_view;           // elements between the weight stacks of two views
    int n_planes, H, V, v;   // v: the view of this update (ROWS_RATIO, ROWS_UPDATE*)
    float eps;
    int final;               // ROWS_UPDATE: last update -> write `out`, skip the forward FFT
                             // ROWS_FIRST : iterations == 0 -> write `out` only
    int total_rows;          // pairs * H
    // guard: ROWS_FIRST records max(psi_0) of every pair (float bits; psi_0 >= 0), ROWS_RATIO flags
    // the pairs in which some pixel has phi_v > 0 and blur < guard_rel * that maximum
    unsigned* gmax;          // [pairs]
    unsigned* gflag;         // [pairs]
    float guard_rel;
};

// ROWS_FIRST: fold this thread's maximum of psi_0 into the pair's word.  The plain read is only a filter
// (a stale value costs an extra atomic, never a wrong result).
__device__ __forceinline__ void guard_note_max(unsigned* gmax, int pair, float m) {
    const unsigned bits = __float_as_uint(m);
    if (bits > *(volatile unsigned*)(gmax + pair)) atomicMax(gmax + pair, bits);
}

template <class P, int MODE, int NT>
__global__ void __launch_bounds__(NT) fft_rows_kernel(RowArgs a, const float2* __restrict__ tw_g) {
    constexpr int E = P::E, TPF = P::TPF, W = P::N, RP = NT / TPF;
    static_assert(NT % TPF == 0 && RP >= 1, "block must hold whole FFTs");
    extern __shared__ float2 smem_rows[];
    float2* tw = smem_rows;                                   // [(S-1) E][TPF]
    float2* buf = smem_rows + (P::S - 1) * E * TPF;           // [RP][NPAD]
    for (int k = threadIdx.x; k < (P::S - 1) * E * TPF; k += NT) tw[k] = tw_g[k];
    __syncthreads();
    const int r = threadIdx.x / TPF, t = threadIdx.x % TPF;
    const RowAddr<P> addr{r * P::NPAD};
    const size_t npx = (size_t)a.H * W;

    for (int row0 = blockIdx.x * RP; row0 < a.total_rows; row0 += gridDim.x * RP) {
        const int row = row0 + r;
        const bool valid = row < a.total_rows;
        const int pair = valid ? row / a.H : 0, y = valid ? row % a.H : 0;
        const int pa = 2 * pair, pb = 2 * pair + 1;
        const bool has_b = pb < a.n_planes;
        const size_t rowoff = (size_t)row * W;          // into S / Z
        const size_t pxa = (size_t)pa * npx + (size_t)y * W, pxb = pxa + npx;   // into out
        const size_t vxa = (size_t)pa * a.view_plane + (size_t)y * a.view_row, vxb = vxa + a.view_plane;   // into views
        float2 x[E];

        if (MODE == ROWS_FIRST) {
            float gm = 0.f;
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const int pos = t + TPF * e;
                float sa = 0.f, sb = 0.f;
                if (valid)
                    for (int v = 0; v < a.V; ++v) {
                        const uint16_t* vp = a.views + (size_t)v * a.view_stride;
                        sa += (float)__ldg(vp + vxa + pos);
                        if (has_b) sb += (float)__ldg(vp + vxb + pos);
                    }
                x[e] = make_float2(sa / (float)a.V, sb / (float)a.V);       // a0
                gm = fmaxf(gm, fmaxf(x[e].x, x[e].y));
                if (valid) {
                    if (a.final) {
                        if (a.out16) {
                            a.out16[pxa + pos] = to_u16(x[e].x);
                            if (has_b) a.out16[pxb + pos] = to_u16(x[e].y);
                        } else {
                            a.out[pxa + pos] = x[e].x;
                            if (has_b) a.out[pxb + pos] = x[e].y;
                        }
                    } else {
                        a.Z[rowoff + pos] = x[e];
                    }
                }
            }
            if (a.final) continue;   // uniform over the block
            if (valid) guard_note_max(a.gmax, pair, gm);
        } else {
            uint32_t ph[E];          // phi_a | phi_b << 16, fetched before the inverse transform
            if (MODE == ROWS_RATIO) {
                const uint16_t* vp = a.views + (size_t)a.v * a.view_stride;
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    const int pos = t + TPF * e;
                    uint32_t lo = 0, hi = 0;
                    if (valid) {
                        lo = __ldg(vp + vxa + pos);
                        if (has_b) hi = __ldg(vp + vxb + pos);
                    }
                    ph[e] = lo | (hi << 16);
                }
            }
#pragma unroll
            for (int e = 0; e < E; ++e) x[e] = valid ? a.S[rowoff + t + TPF * e] : make_float2(0.f, 0.f);
            fft_run<P, +1>(x, buf, tw, t, addr);
            if (MODE == ROWS_RATIO) {
#pragma unroll
                for (int e = 0; e < E; ++e) {                                 // a2
                    x[e].x = (float)(ph[e] & 0xffffu) / fmaxf(x[e].x, a.eps);
                    x[e].y = (float)(ph[e] >> 16) / fmaxf(x[e].y, a.eps);
                }
            } else {
#pragma unroll
                for (int e = 0; e < E; ++e) {                                 // a4
                    const int pos = t + TPF * e;
                    const float2 z = valid ? a.Z[rowoff + pos] : make_float2(0.f, 0.f);
                    x[e] = make_float2(z.x * x[e].x, z.y * x[e].y);
                    if (valid) {
                        if (a.final) {
                            if (a.out16) {
                                a.out16[pxa + pos] = to_u16(x[e].x);
                                if (has_b) a.out16[pxb + pos] = to_u16(x[e].y);
                            } else {
                                a.out[pxa + pos] = x[e].x;
                                if (has_b) a.out[pxb + pos] = x[e].y;
                            }
                        } else {
                            a.Z[rowoff + pos] = x[e];
                        }
                    }
                }
                if (a.final) continue;
            }
        }
        fft_run<P, -1>(x, buf, tw, t, addr);
        if (valid) {
#pragma unroll
            for (int e = 0; e < E; ++e) a.S[rowoff + t + TPF * e] = x[e];
        }
    }
}

// Shared-memory map of the streamed row kernels (bytes from the 128-byte aligned base).
template <class P, int MODE, int NT>
struct RowSmem {
    static constexpr int RP = NT / P::TPF;
    static constexpr size_t kTw = 0;
    static constexpr size_t kBuf = align_up(sizeof(float2) * (P::S - 1) * P::E * P::TPF, 128);
    static constexpr size_t kStage = kBuf + align_up(sizeof(float2) * RP * P::NPAD, 128);
    static constexpr size_t kStageBytes = align_up(sizeof(float2) * RP * P::N, 128);
    static constexpr size_t kAux = kStage + 2 * kStageBytes;
    // ROWS_RATIO: two uint16 rows (plane a, plane b) per row;  ROWS_UPDATE: the psi row (float2)
    static constexpr size_t kAuxRow = MODE == ROWS_RATIO ? 2 * sizeof(uint16_t) * P::N : sizeof(float2) * P::N;
    static constexpr size_t kAuxBytes = align_up(kAuxRow * RP, 128);
    static constexpr size_t kBar = kAux + 2 * kAuxBytes;
    static constexpr size_t kTotal = kBar + 2 * sizeof(uint64_t);
};

// rows_ratio / rows_update with the inputs of the NEXT pass streamed into shared memory by bulk
// copies (one spectrum row + the uint16 rows of the two planes, or the psi row) while the current
// pass is transformed.  Each row's first thread issues that row's copies.
template <class P, int MODE, int NT>
__global__ void __launch_bounds__(NT) fft_rows_tma_kernel(RowArgs a, const float2* __restrict__ tw_g) {
    using L = RowSmem<P, MODE, NT>;
    constexpr int E = P::E, TPF = P::TPF, W = P::N, RP = NT / TPF;
    static_assert(MODE == ROWS_RATIO || MODE == ROWS_UPDATE, "ROWS_FIRST has its own kernel");
    static_assert(NT % TPF == 0 && RP >= 1, "block must hold whole FFTs");
    static_assert(P::S >= 2, "the stage-buffer reuse relies on the barriers of a multi-stage FFT");
    extern __shared__ __align__(128) unsigned char smem_rows_tma[];
    float2* tw = reinterpret_cast<float2*>(smem_rows_tma + L::kTw);
    float2* buf = reinterpret_cast<float2*>(smem_rows_tma + L::kBuf);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_rows_tma + L::kBar);
    const int r = threadIdx.x / TPF, t = threadIdx.x % TPF;
    const RowAddr<P> addr{r * P::NPAD};
    const size_t npx = (size_t)a.H * W;
    const uint16_t* vp = a.views + (size_t)a.v * a.view_stride;

    if (threadIdx.x == 0) {
        mbar_init(&bar[0], RP);
        mbar_init(&bar[1], RP);
        fence_mbar_init();
    }
    for (int k = threadIdx.x; k < (P::S - 1) * E * TPF; k += NT) tw[k] = tw_g[k];
    __syncthreads();

    // the row's first thread fetches the row's inputs of pass `row0` into stage `s`
    auto issue = [&](int row0, int s) {
        if (t != 0) return;
        const int row = row0 + r;
        if (row >= a.total_rows) { mbar_arrive(&bar[s]); return; }
        const int pair = row / a.H, y = row % a.H;
        const bool has_b = 2 * pair + 1 < a.n_planes;
        const size_t vxa = (size_t)(2 * pair) * a.view_plane + (size_t)y * a.view_row;
        unsigned char* st = smem_rows_tma + L::kStage + (size_t)s * L::kStageBytes + sizeof(float2) * W * r;
        unsigned char* ax = smem_rows_tma + L::kAux + (size_t)s * L::kAuxBytes + L::kAuxRow * r;
        const uint32_t row_bytes = sizeof(float2) * W;
        if (MODE == ROWS_RATIO) {
            const uint32_t pb = sizeof(uint16_t) * W;
            mbar_arrive_expect_tx(&bar[s], row_bytes + (has_b ? 2 * pb : pb));
            bulk_g2s(st, a.S + (size_t)row * W, row_bytes, &bar[s]);
            bulk_g2s(ax, vp + vxa, pb, &bar[s]);
            if (has_b) bulk_g2s(ax + pb, vp + vxa + a.view_plane, pb, &bar[s]);
        } else {
            mbar_arrive_expect_tx(&bar[s], 2 * row_bytes);
            bulk_g2s(st, a.S + (size_t)row * W, row_bytes, &bar[s]);
            bulk_g2s(ax, a.Z + (size_t)row * W, row_bytes, &bar[s]);
        }
    };

    const int stride = gridDim.x * RP;
    int row0 = blockIdx.x * RP;
    if (row0 < a.total_rows) issue(row0, 0);
    for (int i = 0; row0 < a.total_rows; row0 += stride, ++i) {
        const int s = i & 1;
        if (row0 + stride < a.total_rows) issue(row0 + stride, s ^ 1);
        const int row = row0 + r;
        const bool valid = row < a.total_rows;
        const int pair = valid ? row / a.H : 0, y = valid ? row % a.H : 0;
        const bool has_b = 2 * pair + 1 < a.n_planes;
        const size_t rowoff = (size_t)row * W;
        const size_t pxa = (size_t)(2 * pair) * npx + (size_t)y * W, pxb = pxa + npx;
        const float2* st = reinterpret_cast<const float2*>(smem_rows_tma + L::kStage + (size_t)s * L::kStageBytes) + (size_t)W * r;
        const unsigned char* ax = smem_rows_tma + L::kAux + (size_t)s * L::kAuxBytes + L::kAuxRow * r;

        mbar_wait(&bar[s], (i >> 1) & 1);
        float2 x[E];
#pragma unroll
        for (int e = 0; e < E; ++e) x[e] = valid ? st[t + TPF * e] : make_float2(0.f, 0.f);
        fft_run<P, +1>(x, buf, tw, t, addr);
        if (MODE == ROWS_RATIO) {
            const uint16_t* pa = reinterpret_cast<const uint16_t*>(ax);
            const float tau = a.guard_rel * __uint_as_float(a.gmax[pair]);
            float bmin = 3.0e38f;
#pragma unroll
            for (int e = 0; e < E; ++e) {                                 // a2
                const int pos = t + TPF * e;
                const float fa = valid ? (float)pa[pos] : 0.f;
                const float fb = (valid && has_b) ? (float)pa[W + pos] : 0.f;
                bmin = fminf(bmin, fminf(fa > 0.f ? x[e].x : 3.0e38f, fb > 0.f ? x[e].y : 3.0e38f));
                x[e].x = div_approx(fa, fmaxf(x[e].x, a.eps));
                x[e].y = div_approx(fb, fmaxf(x[e].y, a.eps));
            }
            if (bmin < tau) a.gflag[pair] = 1u;
        } else {
            const float2* zr = reinterpret_cast<const float2*>(ax);
            const float* wa = a.weights ? a.weights + (size_t)a.v * a.w_view + pxa : nullptr;   // weights share out's layout
#pragma unroll
            for (int e = 0; e < E; ++e) {                                 // a4
                const int pos = t + TPF * e;
                const float2 z = valid ? zr[pos] : make_float2(0.f, 0.f);
                if (wa && valid) {                                        // a4w
                    const float w0 = __ldg(wa + pos), w1 = has_b ? __ldg(wa + npx + pos) : 0.f;
                    x[e] = make_float2(fmaf(w0, x[e].x, 1.f - w0), fmaf(w1, x[e].y, 1.f - w1));
                }
                x[e] = make_float2(z.x * x[e].x, z.y * x[e].y);
                if (valid) {
                    if (a.final) {
                        if (a.out16) {
                            a.out16[pxa + pos] = to_u16(x[e].x);
                            if (has_b) a.out16[pxb + pos] = to_u16(x[e].y);
                        } else {
                            a.out[pxa + pos] = x[e].x;
                            if (has_b) a.out[pxb + pos] = x[e].y;
                        }
                    } else {
                        a.Z[rowoff + pos] = x[e];
                    }
                }
            }
            if (a.final) {
                __syncthreads();   // every thread is done with this stage's psi row before it is refilled
                continue;
            }
        }
        fft_run<P, -1>(x, buf, tw, t, addr);
        if (valid) {
#pragma unroll
            for (int e = 0; e < E; ++e) a.S[rowoff + t + TPF * e] = x[e];
        }
    }
}

// Column pass with the next pair's tile streamed in by a 2D tiled TMA copy.  Two tile buffers: the
// one the tile arrived in becomes the exchange buffer of its own transforms once the registers are
// loaded, the other one receives the next tile meanwhile.
template <class P, int TC>
struct ColSmem {
    static constexpr int BOXH = P::N <= 256 ? P::N : (P::N % 256 == 0 ? 256 : (P::N % 200 == 0 ? 200 : (P::N % 160 == 0 ? 160 : 128)));
    static_assert(P::N % BOXH == 0, "tile rows must split into whole TMA boxes");
    static constexpr size_t kTw = 0;
    static constexpr size_t kTile = align_up(sizeof(float2) * (P::S - 1) * P::E * P::TPF, 128);
    static constexpr size_t kTileBytes = align_up(sizeof(float2) * ColAddr<P, TC>::NPOS * TC, 128);
    static constexpr size_t kBar = kTile + 2 * kTileBytes;
    static constexpr size_t kTotal = kBar + 2 * sizeof(uint64_t);
};

template <class P, int TC, bool OTF_REGS>
__global__ void __launch_bounds__(TC* P::TPF)
fft_cols_tma_kernel(const __grid_constant__ CUtensorMap tmap, float2* __restrict__ S,
                    const float2* __restrict__ otf, int conj_otf, int pairs, int W,
                    const float2* __restrict__ tw_g) {
    using L = ColSmem<P, TC>;
    constexpr int E = P::E, TPF = P::TPF, H = P::N, NT = TC * TPF;
    static_assert(P::S >= 2, "the tile-buffer reuse relies on the barriers of a multi-stage FFT");
    extern __shared__ __align__(128) unsigned char smem_cols_tma[];
    float2* tw = reinterpret_cast<float2*>(smem_cols_tma + L::kTw);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_cols_tma + L::kBar);
    const int c = threadIdx.x % TC, t = threadIdx.x / TC;
    const ColAddr<P, TC> addr{c};
    const int xg = blockIdx.x * TC + c;
    const float sgn = conj_otf ? -1.f : 1.f;

    if (threadIdx.x == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        fence_mbar_init();
    }
    for (int k = threadIdx.x; k < (P::S - 1) * E * TPF; k += NT) tw[k] = tw_g[k];
    __syncthreads();

    auto issue = [&](int p, int s) {
        if (threadIdx.x != 0) return;
        unsigned char* dst = smem_cols_tma + L::kTile + (size_t)s * L::kTileBytes;
        mbar_arrive_expect_tx(&bar[s], (uint32_t)(sizeof(float2) * H * TC));
#pragma unroll
        for (int b = 0; b < H / L::BOXH; ++b)
            tma_2d_g2s(dst + sizeof(float2) * TC * L::BOXH * b, &tmap, 2 * (int)(blockIdx.x * TC),
                       p * H + b * L::BOXH, &bar[s]);
    };

    float2 o[OTF_REGS ? E : 1];
    if (OTF_REGS) {
#pragma unroll
        for (int e = 0; e < E; ++e) {
            o[e] = __ldg(otf + (size_t)(t + TPF * e) * W + xg);
            o[e].y *= sgn;
        }
    }
    int p = blockIdx.y;
    if (p < pairs) issue(p, 0);
    for (int i = 0; p < pairs; p += gridDim.y, ++i) {
        const int s = i & 1;
        if (p + (int)gridDim.y < pairs) issue(p + gridDim.y, s ^ 1);
        float2* tile = reinterpret_cast<float2*>(smem_cols_tma + L::kTile + (size_t)s * L::kTileBytes);
        float2* Sp = S + (size_t)p * H * W + xg;
        mbar_wait(&bar[s], (i >> 1) & 1);
        float2 x[E];
#pragma unroll
        for (int e = 0; e < E; ++e) x[e] = tile[(t + TPF * e) * TC + c];
        __syncthreads();   // the tile buffer turns into the exchange buffer
        fft_run<P, -1>(x, tile, tw, t, addr);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            float2 w;
            if (OTF_REGS) {
                w = o[e];
            } else {
                w = __ldg(otf + (size_t)(t + TPF * e) * W + xg);
                w.y *= sgn;
            }
            x[e] = cmul(x[e], w);
        }
        fft_run<P, +1>(x, tile, tw, t, addr);
#pragma unroll
        for (int e = 0; e < E; ++e) Sp[(size_t)(t + TPF * e) * W] = x[e];
    }
}

// ---------------------------------------------------------------------------------------------
// host-side descriptors (one per supported length)
// ---------------------------------------------------------------------------------------------
struct PlanInfo {
    int E, TPF, S;
    int radices[5];
};
struct SizeOps {
    int N;
    PlanInfo row, col;               // the length's plan when it is the row (x) / column (z) length
    int row_threads;                 // NT of the row kernels
    size_t row_smem, col_smem;       // dynamic shared memory (bytes)
    int col_tc;                      // TC of the column kernel
    cudaError_t (*rows)(int mode, const RowArgs& a, const float2* tw, int grid, cudaStream_t st);
    int col_box_h;                   // rows per TMA box of the column kernel's tile
    cudaError_t (*cols)(const CUtensorMap& tmap, const CUtensorMap& otf_map, float2* S, const float2* otf, int conj_otf, int pairs, int W,
                        const float2* tw, dim3 grid, cudaStream_t st);
    cudaError_t (*prepare_rows)();   // opt in to > 48 KB dynamic shared memory (length used as W)
    cudaError_t (*prepare_cols)();   // same (length used as H)
    int col_box_w = 0;               // generation 2: floats per TMA box row (2 x columns per team)
    int col_otf_regs = 0;            // generation 2: the column kernel keeps its tile's OTF in registers
    int row_cps = 0, col_cps = 0;    // generation 2: resident CTAs per SM the persistent grids are sized for
    int row_cps_w = 0;               // ... of the weighted update kernel (twice the landing zone)
    int generation = 1;              // 1: CTA-synchronous TMA-staged kernels (this file); 2: team kernels (mvd_fft_v2.cuh)
    int col_real_otf = 0;            // the column kernel takes conj_otf == 2: a REAL transfer function stored as float (and its float tensor map)
    int col_tw_custom = 0;           // 1: the column kernel's twiddle table is [R0][N / R0]: exp(-2 pi i t k / N) at [k][t] (two-stage plans with unequal thread counts)
};

template <class P, int NT, class PC, int TC, bool OTF_REGS>
struct OpsFor {
    static_assert(P::N == PC::N, "row and column plan of one entry describe the same length");
    static constexpr size_t kFirstSmem = sizeof(float2) * ((size_t)(P::S - 1) * P::E * P::TPF + (size_t)(NT / P::TPF) * P::NPAD);
    static constexpr size_t kRatioSmem = RowSmem<P, ROWS_RATIO, NT>::kTotal;
    static constexpr size_t kUpdateSmem = RowSmem<P, ROWS_UPDATE, NT>::kTotal;
    static constexpr size_t kColSmem = ColSmem<PC, TC>::kTotal;

    static cudaError_t rows(int mode, const RowArgs& a, const float2* tw, int grid, cudaStream_t st) {
        if (mode == ROWS_FIRST) fft_rows_kernel<P, ROWS_FIRST, NT><<<grid, NT, kFirstSmem, st>>>(a, tw);
        else if (mode == ROWS_RATIO) fft_rows_tma_kernel<P, ROWS_RATIO, NT><<<grid, NT, kRatioSmem, st>>>(a, tw);
        else fft_rows_tma_kernel<P, ROWS_UPDATE, NT><<<grid, NT, kUpdateSmem, st>>>(a, tw);   // also ROWS_UPDATE_W
        return cudaGetLastError();
    }
    static cudaError_t cols(const CUtensorMap& tmap, const CUtensorMap& otf_map, float2* S, const float2* otf, int conj_otf, int pairs, int W,
                            const float2* tw, dim3 grid, cudaStream_t st) {
        (void)otf_map;
        fft_cols_tma_kernel<PC, TC, OTF_REGS><<<grid, TC * PC::TPF, kColSmem, st>>>(tmap, S, otf, conj_otf, pairs, W, tw);
        return cudaGetLastError();
    }
    static cudaError_t prepare_rows() {
        cudaError_t e;
        e = cudaFuncSetAttribute(fft_rows_kernel<P, ROWS_FIRST, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFirstSmem);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(fft_rows_tma_kernel<P, ROWS_RATIO, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRatioSmem);
        if (e != cudaSuccess) return e;
        return cudaFuncSetAttribute(fft_rows_tma_kernel<P, ROWS_UPDATE, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kUpdateSmem);
    }
    static cudaError_t prepare_cols() {
        return cudaFuncSetAttribute(fft_cols_tma_kernel<PC, TC, OTF_REGS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kColSmem);
    }
    static SizeOps make() {
        SizeOps o;
        o.N = P::N;
        o.row = PlanInfo{P::E, P::TPF, P::S, {P::radix(0), P::radix(1), P::radix(2), P::radix(3), P::radix(4)}};
        o.col = PlanInfo{PC::E, PC::TPF, PC::S, {PC::radix(0), PC::radix(1), PC::radix(2), PC::radix(3), PC::radix(4)}};
        o.row_threads = NT;
        o.row_smem = kRatioSmem > kUpdateSmem ? kRatioSmem : kUpdateSmem;
        o.col_smem = kColSmem; o.col_tc = TC; o.col_box_h = ColSmem<PC, TC>::BOXH;
        o.rows = &rows; o.cols = &cols; o.prepare_rows = &prepare_rows; o.prepare_cols = &prepare_cols;
        return o;
    }
};

}  // namespace mvdfft

// one translation unit per group of sizes (parallel compilation); each returns nullptr for other N
const mvdfft::SizeOps* mvd_fft_ops_small(int N);
const mvdfft::SizeOps* mvd_fft_ops_mid(int N);
const mvdfft::SizeOps* mvd_fft_ops_large(int N);
const mvdfft::SizeOps* mvd_fft_ops_more_a(int N);   // 384, 768, 1536
const mvdfft::SizeOps* mvd_fft_ops_more_b(int N);   // 640, 1280, 1600
const mvdfft::SizeOps* mvd_fft_ops_v2(int N);      // power-of-two lengths (and 800-point columns), team kernels
const mvdfft::SizeOps* mvd_fft_ops_v2b(int N);     // 384, 768, 1536, 640, 1280, team kernels
