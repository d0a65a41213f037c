// FFT engine instantiations: lengths 2^a x 3 (384, 768, 1536), generation-1 kernels.
#include "mvd_fft_kernels.cuh"
using namespace mvdfft;

const SizeOps* mvd_fft_ops_more_a(int N) {
    using P384 = Plan<384, 24, 8, 4, 4, 3>;
    using P768 = Plan<768, 24, 8, 8, 4, 3>;
    using P1536 = Plan<1536, 24, 8, 8, 8, 3>;
    static const SizeOps o384 = OpsFor<P384, 128, P384, 8, false>::make();
    static const SizeOps o768 = OpsFor<P768, 128, P768, 8, false>::make();
    static const SizeOps o1536 = OpsFor<P1536, 64, P1536, 4, false>::make();
    switch (N) {
        case 384: return &o384;
        case 768: return &o768;
        case 1536: return &o1536;
        default: return nullptr;
    }
}
