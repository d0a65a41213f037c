// FFT engine instantiations: lengths 256 .. 800.
#include "mvd_fft_kernels.cuh"
using namespace mvdfft;

const SizeOps* mvd_fft_ops_mid(int N) {
    using P256 = Plan<256, 16, 16, 16>;
    using P320 = Plan<320, 40, 8, 8, 5>;
    using P512 = Plan<512, 8, 8, 8, 8>;
    using P800 = Plan<800, 40, 8, 5, 5, 4>;
    static const SizeOps o256 = OpsFor<P256, 256, P256, 16, true>::make();
    static const SizeOps o320 = OpsFor<P320, 64, P320, 8, false>::make();
    static const SizeOps o512 = OpsFor<P512, 256, P512, 8, true>::make();
    static const SizeOps o800 = OpsFor<P800, 80, P800, 8, false>::make();
    switch (N) {
        case 256: return &o256;
        case 320: return &o320;
        case 512: return &o512;
        case 800: return &o800;
        default: return nullptr;
    }
}
