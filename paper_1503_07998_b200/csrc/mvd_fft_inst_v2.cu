// FFT engine, generation-2 (team-synchronous) kernels: 256, 512, 1024, 2048.
#include <stdio.h>
#include <stdlib.h>

#include "mvd_fft_v2.cuh"
using namespace mvdfft;

const SizeOps* mvd_fft_ops_v2(int N) {
    using P256 = Plan<256, 16, 16, 16>;
    using P512 = Plan<512, 32, 32, 16>;
    using P1024 = Plan<1024, 32, 32, 32>;
    using P2048 = Plan<2048, 32, 32, 32, 2>;
    static const SizeOps o256 = OpsFor2<P256, 256, P256, 128, true, 4>::make();
    static const SizeOps o512 = OpsFor2<P512, 256, P512, 128, false, 3>::make();
    static const SizeOps o1024 = OpsFor2<P1024, 256, P1024, 128, false, 3>::make();
    // rows: 3 CTAs of 2 teams, 168 registers; the exchange in front of the radix-2 stage goes through warp shuffles
    static const SizeOps o2048 = OpsFor2<ShflTail<P2048>, 128, P2048, 256, false, 2, false, 4, 3>::make();
    // columns only: 800 = 25 x 32 with unequal thread counts per stage, four columns per team of four warps
    static const SizeOps o800 = ColsNu2<25, 32, 256, 2>::make();
    using P800C = Plan<800, 40, 40, 20>;     // the uniform plan (eight columns per team of 160 threads), dev builds only
    (void)sizeof(P800C);
#ifdef MVD_DEV
    {   // experiment variants of a dev build (_work/devbuild.py): MVD_DEV_V<N>=<letter>
        char name[32];
        snprintf(name, sizeof name, "MVD_DEV_V%d", N);
        const char* v = getenv(name);
        if (v) {
            if (N == 800 && v[0] == 'l') { static const SizeOps o = ColsLean2<P800C, 160, 3, 8>::make(); return &o; }
            if (N == 1024 && v[0] == 'l') { static const SizeOps o = ColsLean2<P1024, 128, 4, 4>::make(&o1024); return &o; }
            if (N == 1024 && v[0] == 'm') { static const SizeOps o = ColsLean2<P1024, 256, 2, 8>::make(&o1024); return &o; }
            if (N == 512 && v[0] == 'l') { static const SizeOps o = ColsLean2<P512, 128, 4, 4>::make(&o512); return &o; }
            if (N == 512 && v[0] == 'm') { static const SizeOps o = ColsLean2<P512, 128, 4, 8>::make(&o512); return &o; }
            if (N == 800 && v[0] == 'u') { static const SizeOps o = ColsOnly2<P800C, 160, false, 2, 8>::make(); return &o; }
            if (N == 2048 && v[0] == 'u') { static const SizeOps o = OpsFor2<P2048, 128, P2048, 256, false, 2, false, 4, 3>::make(); return &o; }
            if (N == 800 && v[0] == 'o') { static const SizeOps o = ColsNu2<25, 32, 128, 4>::make(); return &o; }
            if (N == 800 && v[0] == 'a') { static const SizeOps o = ColsOnly2<P800C, 320, false, 1, 8>::make(); return &o; }
            if (N == 2048 && v[0] == 'f') { static const SizeOps o = OpsFor2<ShflTail<P2048>, 128, P2048, 256, false, 2, false, 4, 4>::make(); return &o; }
            if (N == 2048 && v[0] == 'a') { static const SizeOps o = OpsFor2<Plan<2048, 16, 16, 16, 8>, 256, P2048, 256, false, 2, false, 4, 3>::make(); return &o; }
            if (N == 2048 && v[0] == 'b') { static const SizeOps o = OpsFor2<Plan<2048, 16, 16, 16, 8>, 512, P2048, 256, false, 2, false, 4, 2>::make(); return &o; }
            if (N == 1024 && v[0] == 'a') { static const SizeOps o = OpsFor2<P1024, 256, Plan<1024, 16, 16, 16, 4>, 256, false, 2>::make(); return &o; }
            if (N == 512 && v[0] == 'c') { static const SizeOps o = OpsFor2<P512, 256, P512, 128, false, 3, true, 8>::make(); return &o; }
            if (N == 1024 && v[0] == 'c') { static const SizeOps o = OpsFor2<P1024, 256, P1024, 256, false, 1, true, 8>::make(); return &o; }
            if (N == 2048 && v[0] == 'c') { static const SizeOps o = OpsFor2<P2048, 128, P2048, 256, false, 2, false, 4, 2>::make(); return &o; }
            if (N == 2048 && v[0] == 'd') { static const SizeOps o = OpsFor2<P2048, 256, P2048, 256, false, 2, false, 4, 2>::make(); return &o; }
            if (N == 2048 && v[0] == 'e') { static const SizeOps o = OpsFor2<P2048, 64, P2048, 256, false, 2, false, 4, 6>::make(); return &o; }
            if (N == 512 && v[0] == 'a') { static const SizeOps o = OpsFor2<P512, 256, Plan<512, 16, 16, 8, 4>, 128, false, 5>::make(); return &o; }
            if (N == 512 && v[0] == 'b') { static const SizeOps o = OpsFor2<P512, 256, Plan<512, 16, 16, 16, 2>, 128, false, 5>::make(); return &o; }
        }
    }
#endif
    switch (N) {
        case 256: return &o256;
        case 512: return &o512;
        case 800: return &o800;
        case 1024: return &o1024;
        case 2048: return &o2048;
        default: return nullptr;
    }
}
