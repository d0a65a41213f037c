// FFT engine instantiations: lengths 1024 .. 2048.
#include "mvd_fft_kernels.cuh"
using namespace mvdfft;

const SizeOps* mvd_fft_ops_large(int N) {
    using P1024 = Plan<1024, 16, 16, 16, 4>;
    using P2048 = Plan<2048, 16, 16, 16, 8>;
    using P2048C = Plan<2048, 32, 16, 16, 8>;
    static const SizeOps o1024 = OpsFor<P1024, 256, P1024, 8, true>::make();
    static const SizeOps o2048 = OpsFor<P2048, 256, P2048C, 4, false>::make();
    switch (N) {
        case 1024: return &o1024;
        case 2048: return &o2048;
        default: return nullptr;
    }
}
