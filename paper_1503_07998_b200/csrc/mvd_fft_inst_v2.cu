// FFT engine, generation-2 (team-synchronous) kernels: 256, 512, 1024, 2048.
#include "mvd_fft_v2.cuh"
using namespace mvdfft;

const SizeOps* mvd_fft_ops_v2(int N) {
    using P256 = Plan<256, 16, 16, 16>;
    using P512 = Plan<512, 32, 32, 16>;
    using P1024 = Plan<1024, 32, 32, 32>;
    using P2048 = Plan<2048, 32, 32, 32, 2>;
    static const SizeOps o256 = OpsFor2<P256, 256, P256, 256, true, true, 2>::make();
    static const SizeOps o512 = OpsFor2<P512, 256, P512, 128, false, true, 3>::make();
    static const SizeOps o1024 = OpsFor2<P1024, 256, P1024, 128, false, true, 3>::make();
    static const SizeOps o2048 = OpsFor2<P2048, 256, P2048, 256, false, false, 2>::make();
    switch (N) {
        case 256: return &o256;
        case 512: return &o512;
        case 1024: return &o1024;
        case 2048: return &o2048;
        default: return nullptr;
    }
}
