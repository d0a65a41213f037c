// FFT engine instantiations: lengths 32 .. 192.
#include "mvd_fft_kernels.cuh"
using namespace mvdfft;

const SizeOps* mvd_fft_ops_small(int N) {
    using P32 = Plan<32, 8, 8, 4>;
    using P64 = Plan<64, 8, 8, 8>;
    using P80 = Plan<80, 20, 5, 4, 4>;
    using P96 = Plan<96, 24, 8, 4, 3>;
    using P128 = Plan<128, 16, 16, 8>;
    using P160 = Plan<160, 40, 8, 5, 4>;
    using P192 = Plan<192, 24, 8, 8, 3>;
    static const SizeOps o32 = OpsFor<P32, 256, P32, 16, true>::make();
    static const SizeOps o64 = OpsFor<P64, 256, P64, 16, true>::make();
    static const SizeOps o80 = OpsFor<P80, 128, P80, 16, true>::make();
    static const SizeOps o96 = OpsFor<P96, 128, P96, 16, true>::make();
    static const SizeOps o128 = OpsFor<P128, 256, P128, 16, true>::make();
    static const SizeOps o160 = OpsFor<P160, 128, P160, 16, false>::make();
    static const SizeOps o192 = OpsFor<P192, 128, P192, 16, true>::make();
    switch (N) {
        case 32: return &o32;
        case 64: return &o64;
        case 80: return &o80;
        case 96: return &o96;
        case 128: return &o128;
        case 160: return &o160;
        case 192: return &o192;
        default: return nullptr;
    }
}
