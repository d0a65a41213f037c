// FFT engine, generation-2 (team-synchronous) kernels for the lengths 2^a 3 and 2^a 5: 384, 768, 1536, 640, 1280.
// Three-stage plans with the large composite radix (24 = 8 x 3, 40 = 8 x 5) first, so that the exchange regions are padded by
// one slot per 24 / 40 positions; rows and columns use the same plan.
#include "mvd_fft_v2.cuh"
using namespace mvdfft;

const SizeOps* mvd_fft_ops_v2b(int N) {
    using P384 = Plan<384, 24, 24, 4, 4>;
    using P768 = Plan<768, 24, 24, 8, 4>;
    using P1536 = Plan<1536, 24, 24, 8, 8>;
    using P640 = Plan<640, 40, 40, 4, 4>;
    using P1280 = Plan<1280, 40, 40, 8, 4>;
    static const SizeOps o384 = OpsFor2<P384, 256, P384, 128, false, 3>::make();
    static const SizeOps o768 = OpsFor2<P768, 256, P768, 512, false, 1>::make();       // columns: four teams share one twiddle table (16 warps per SM)
    static const SizeOps o1536 = OpsFor2<P1536, 256, P1536, 512, false, 1>::make();     // columns: two 256-thread teams share one twiddle table (225 KB)
    static const SizeOps o640 = OpsFor2<P640, 128, P640, 128, false, 2, true, 4, 3>::make();     // E = 40: 168 registers, 3 CTAs
    static const SizeOps o1280 = OpsFor2<P1280, 128, P1280, 128, false, 2, true, 4, 3>::make();
    switch (N) {
        case 384: return &o384;
        case 768: return &o768;
        case 1536: return &o1536;
        case 640: return &o640;
        case 1280: return &o1280;
        default: return nullptr;
    }
}
