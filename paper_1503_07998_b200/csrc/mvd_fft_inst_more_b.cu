// FFT engine instantiations: lengths 2^a x 5^b with a radix-40 first stage (640, 1280, 1600), generation-1 kernels.
#include "mvd_fft_kernels.cuh"
using namespace mvdfft;

const SizeOps* mvd_fft_ops_more_b(int N) {
    using P640 = Plan<640, 40, 40, 8, 2>;
    using P1280 = Plan<1280, 40, 40, 8, 4>;
    using P1600 = Plan<1600, 40, 40, 40>;
    static const SizeOps o640 = OpsFor<P640, 64, P640, 8, false>::make();
    static const SizeOps o1280 = OpsFor<P1280, 64, P1280, 4, false>::make();
    static const SizeOps o1600 = OpsFor<P1600, 80, P1600, 4, false>::make();
    switch (N) {
        case 640: return &o640;
        case 1280: return &o1280;
        case 1600: return &o1600;
        default: return nullptr;
    }
}
