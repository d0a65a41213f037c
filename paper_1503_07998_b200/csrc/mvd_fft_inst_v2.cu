// FFT engine, generation-2 (team-synchronous) kernels: 256, 512, 1024, 2048.
#include "mvd_fft_v2.cuh"
using namespace mvdfft;

const SizeOps* mvd_fft_ops_v2(int N) {
    using P256 = Plan<256, 16, 16, 16>;
    using P512 = Plan<512, 32, 32, 16>;
    using P1024 = Plan<1024, 32, 32, 32>;
    using P2048 = Plan<2048, 32, 32, 32, 2>;
    // columns: OTF in registers, two regions per team in ping-pong (the next slice is requested a whole item ahead)
    static const SizeOps o256 = OpsFor2<P256, 256, P256, 128, true, 4, true, 4, 2, true>::make();
    static const SizeOps o512 = OpsFor2<P512, 256, P512, 128, false, 3>::make();
    static const SizeOps o1024 = OpsFor2<P1024, 256, P1024, 128, false, 3>::make();
    // rows: the exchange in front of the radix-2 stage goes through warp shuffles; 2 CTAs of 4 teams at 128 registers (since the
    // instruction diet they fit without spills).  3 CTAs of 2 teams at 168 registers run the update pass 3 % faster ALONE but the
    // whole step, with two batches in flight, 1.5 % slower (profiles/r2_experiments.md).
    // columns: one 256-thread team per SM (166 KB: both regions of 2048 rows and a 32 KB twiddle table); the cp.async kernel
    // it replaces fitted two CTAs but ran at 0.28 of the copy peak against 0.44 (2048 x 2048 planes: 75 -> 92 GVoxel/s);
    // the shuffle exchange serves the columns too (lanes l and l ^ 16 hold threads t and t ^ 32 of a column)
    static const SizeOps o2048 = OpsFor2<ShflTail<P2048>, 256, ShflTail<P2048>, 256, false, 1, true, 4, 2>::make();
    // columns only: 800 = 25 x 32 with unequal thread counts per stage, four columns per team of four warps
    static const SizeOps o800 = ColsNu2<25, 32, 256, 2>::make();
    switch (N) {
        case 256: return &o256;
        case 512: return &o512;
        case 800: return &o800;
        case 1024: return &o1024;
        case 2048: return &o2048;
        default: return mvd_fft_ops_v2b(N);
    }
}
