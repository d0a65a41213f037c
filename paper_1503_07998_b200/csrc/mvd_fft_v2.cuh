// mvd_fft_v2.cuh -- second-generation FFT-engine kernels for power-of-two lengths (sm_100a).
//
// Same passes and the same arithmetic as mvd_fft_kernels.cuh (rows_first, cols . OTF, rows_ratio,
// rows_update), organised around TEAMS instead of CTAs:
//   * a row FFT is owned by a team of TPF threads that sits inside one warp (TPF <= 32) or is made of
//     whole warps; the team's exchange region in shared memory is private, so the only synchronisation
//     of a transform is __syncwarp / a named barrier of the team.  Warps of a CTA drift apart and hide
//     each other's shared-memory and HBM latency; nothing in the steady state is a CTA-wide barrier;
//   * a column team owns FOUR adjacent columns (one 32-byte sector per image row) and 4 TPF threads, so
//     every global load and store of the column pass moves whole sectors without a staging tile;
//   * plans have two stages wherever E = 32 elements per thread allows it (256 = 16 x 16, 512 = 32 x 16,
//     1024 = 32 x 32): one exchange per transform, i.e. half the shared-memory traffic of the 8 x 8 x 8
//     plans, which matters because at HBM speed the exchanges alone need ~50 % of an SM's shared-memory
//     bandwidth;
//   * the spectrum S and the OTFs are stored TILE-MAJOR: plane element (y, x) lives at
//     ((x / 16) H + y) 16 + x % 16, i.e. 16-column tiles of H rows with 128 contiguous bytes per row.  A
//     column team then walks one contiguous tile (DRAM pages stay open) instead of touching 32 bytes in
//     every 8 W-byte image row, and a row team still reads whole 128-byte lines;
//   * exchange regions are conflict-free for 8-byte elements for both the stride-R0 stores of stage 0 and the
//     unit-stride loads: padded (position p in slot p + p / R0) in the row kernels and the TMA-fed column kernels --
//     every address an immediate offset from one base (round 1 used an XOR swizzle, p ^ ((p / R0) & 15)).
#pragma once

#include "mvd_fft_kernels.cuh"

namespace mvdfft {

// programmatic dependent launch: let the next kernel in the stream start its prologue early, and wait
// for the previous kernel's memory before touching anything it wrote
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// L2 prefetch of a contiguous span (16-byte aligned, size a multiple of 16)
__device__ __forceinline__ void prefetch_l2(const void* p, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// One FFT per region of N + N / R0 slots, position p in slot p + p / R0 (one spare slot per R0).  For the ROW kernels this
// padding does what the XOR swizzle does -- stage 0's stores (positions R0 t + m: slots (R0 + 1) t + m) and the loads
// (positions t + TPF e: consecutive slots) are both conflict-free for 8-byte elements -- and, unlike the XOR, it leaves
// every address an immediate offset from one per-thread base: no LOP3 / IADD3 per access (9 % of the row kernels'
// instructions).
template <class P>
struct RowAddr2 {
    int base;
    __device__ __forceinline__ int operator()(int pos) const { return base + pos + pos / P::radix(0); }
};
template <class P>
__host__ __device__ constexpr int row_pitch(int slots) { return slots + slots / P::radix(0); }
// CPT FFTs (adjacent columns) interleaved, [slot][CPT], with the same padding: position p in slot p + p / R0 of a region of
// H + H / R0 slots.  Stage 0's stores ((R0 + 1) t + m: four consecutive t fall into the four 32-byte groups of a line) and
// the loads (consecutive slots) stay conflict-free, and every address is an immediate offset from one base.
template <class P, int CPT = 4>
struct ColAddrPad {
    int base;   // team region + column within the team
    __device__ __forceinline__ int operator()(int pos) const { return base + CPT * (pos + pos / P::radix(0)); }
};

// 16-byte asynchronous copy global -> shared (SASS LDGSTS), no registers in between
__device__ __forceinline__ void cp_async16(void* dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// ---------------------------------------------------------------------------------------------
// row passes: rows_first (MODE 0), rows_ratio (1), rows_update (2)
//
// rows_ratio / rows_update keep a team's exchange region busy all the time: while a transform runs
// its register-only last stage the region is the landing zone of the next input (cp.async, no
// registers involved), so no global load latency sits on a team's critical path:
//     [S row landed]  -> registers -> inverse FFT head | issue phi / psi row | inverse FFT tail
//     [aux landed]    -> pointwise step               -> forward FFT head | issue next S row | tail -> store
// ---------------------------------------------------------------------------------------------
template <class P, int MODE, int NT, int RMINB = 2>
__global__ void __launch_bounds__(NT, RMINB) fft2_rows_kernel(RowArgs a, const float2* __restrict__ tw_g) {
    constexpr int E = P::E, TPF = P::TPF, W = P::N, RP = NT / TPF;
    constexpr bool UPD = MODE == ROWS_UPDATE || MODE == ROWS_UPDATE_W, WT = MODE == ROWS_UPDATE_W;
    constexpr int RW = WT ? 2 * W : W;   // float2 slots of a team's region: exchange / landing zone (+ the weight rows)
    static_assert(NT % TPF == 0 && (TPF <= 32 ? 32 % TPF == 0 : TPF % 32 == 0), "teams are warp-aligned");
    static_assert(TPF % 16 == 0 && W % 16 == 0, "tile-major addressing assumes whole 16-element groups per team step");
    static_assert(TPF <= 32 || RP <= 15, "one named barrier per team");
    static_assert(E % 8 == 0 && TPF % 8 == 0, "the landing copies split evenly over the team");
    (void)UPD;
    extern __shared__ __align__(16) float2 smem_rows2[];
    float2* tw = smem_rows2;                                  // [(S-1) E][TPF]
    float2* buf = smem_rows2 + (P::S - 1) * E * TPF;          // [RP][RW]
    for (int k = threadIdx.x; k < (P::S - 1) * E * TPF; k += NT) tw[k] = tw_g[k];
    __syncthreads();
    pdl_launch_dependents();
    pdl_wait();
    const int team = threadIdx.x / TPF;
    // ShflTail plans: threads t and t ^ 32 of an FFT sit in lanes l and l ^ 16 of one warp
    const int t = shfl_tail<P>() ? ((int)(threadIdx.x & 16) << 1) | ((int)(threadIdx.x & 32) >> 1) | (int)(threadIdx.x & 15)
                                 : (int)threadIdx.x % TPF;
    constexpr int RWP = row_pitch<P>(RW);   // pitch of a team's region
    const RowAddr2<P> addr{team * RWP};
    const TeamSync<TPF> sync{team};
    const size_t npx = (size_t)a.H * W;
    const int stride = gridDim.x * RP;
    const uint16_t* vp = a.views + (size_t)a.v * a.view_stride;
    float2* land = buf + team * RWP;                          // the team's region, used linearly as landing zone
    const float* wv = WT ? a.weights + (size_t)a.v * a.w_view : nullptr;
    const int last_row = a.total_rows - 1;

    // S is tile-major: 16-byte chunk q = t + TPF k of image row `row` (elements 2q, 2q+1) sits in tile q / 8 at
    // chunk q % 8 of the row's 128 bytes.  TPF is a multiple of 8, so the source address is LINEAR in k
    // (one base + k * step): no per-chunk 64-bit offsets for the compiler to hoist and spill.
    const size_t chunk_step = (size_t)(TPF / 8) * a.H * 16;
    auto issue_S = [&](int row) {
        const int pair = row / a.H, y = row % a.H;
        const float2* src = a.S + (size_t)pair * npx + (size_t)y * 16 + (size_t)(t >> 3) * (a.H * 16) + 2 * (t & 7);
#pragma unroll
        for (int k = 0; k < E / 2; ++k) cp_async16(land + 2 * (t + TPF * k), src + k * chunk_step);
        cp_async_commit();
    };

    if (MODE != ROWS_FIRST && (int)blockIdx.x * RP < a.total_rows) issue_S(min((int)blockIdx.x * RP + team, last_row));

    for (int row0 = blockIdx.x * RP; row0 < a.total_rows; row0 += stride) {
        // A team whose row is past the end works on the last row again and stores nothing, so the
        // control flow (and every barrier) is uniform.
        const bool valid = row0 + team < a.total_rows;
        const int row = valid ? row0 + team : last_row;
        const int pair = row / a.H, y = row % a.H;
        const bool has_b = 2 * pair + 1 < a.n_planes;
        const size_t rowoff = (size_t)row * W;                                      // into Z
        const size_t pxa = (size_t)(2 * pair) * npx + (size_t)y * W;                // into out
        const size_t pxb = has_b ? pxa + npx : pxa;                                 // odd tail: plane a again, discarded
        const size_t vxa = (size_t)(2 * pair) * a.view_plane + (size_t)y * a.view_row;   // into views
        const size_t vxb = has_b ? vxa + a.view_plane : vxa;
        const bool st_a = valid, st_b = valid && has_b;
        float2* Srow = a.S + (size_t)pair * npx + (size_t)(t >> 4) * (a.H * 16) + (size_t)y * 16 + (t & 15);
        const size_t Sstep = (size_t)TPF * a.H;       // x advances by TPF: TPF / 16 tiles of H * 16 elements
        float2* Zrow = a.Z + rowoff + t;
        const bool more = row0 + stride < a.total_rows;
        const int next_row = min(row0 + stride + team, last_row);
        float2 x[E];

        if (MODE == ROWS_FIRST) {
#pragma unroll
            for (int e = 0; e < E; ++e) x[e] = make_float2(0.f, 0.f);
            for (int v = 0; v < a.V; ++v) {
                const uint16_t* qa = a.views + (size_t)v * a.view_stride + vxa + t;
                const uint16_t* qb = a.views + (size_t)v * a.view_stride + vxb + t;
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    x[e].x += (float)__ldg(qa + TPF * e);
                    x[e].y += (float)__ldg(qb + TPF * e);
                }
            }
            const float fv = (float)a.V;
            float gm = 0.f;
#pragma unroll
            for (int e = 0; e < E; ++e) {
                x[e] = make_float2(x[e].x / fv, x[e].y / fv);       // a0
                gm = fmaxf(gm, fmaxf(x[e].x, x[e].y));
            }
            if (valid && !a.final) guard_note_max(a.gmax, pair, gm);
            if (a.final) {   // iterations == 0: the mean is the result (uniform over the grid)
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    if (a.out16) {
                        if (st_a) a.out16[pxa + t + TPF * e] = to_u16(x[e].x);
                        if (st_b) a.out16[pxb + t + TPF * e] = to_u16(x[e].y);
                    } else {
                        if (st_a) a.out[pxa + t + TPF * e] = x[e].x;
                        if (st_b) a.out[pxb + t + TPF * e] = x[e].y;
                    }
                }
                continue;
            }
            if (valid) {
#pragma unroll
                for (int e = 0; e < E; ++e) Zrow[TPF * e] = x[e];
            }
            fft_run<P, -1>(x, buf, tw, t, addr, sync);
        } else {
            cp_async_wait_all();
            sync();
#pragma unroll
            for (int e = 0; e < E; ++e) x[e] = land[t + TPF * e];
            sync();
            fft_run_head<P, +1>(x, buf, tw, t, addr, sync);
            if (MODE == ROWS_RATIO) {
                // phi rows of the two planes: W uint16 each, [0, W) plane a, [W, 2 W) plane b;
                // W / 8 chunks of 8 uint16 per plane, E / 8 of them per thread and plane
                uint16_t* lu = reinterpret_cast<uint16_t*>(land);
                const uint16_t* qa = vp + vxa + 8 * t;
                const uint16_t* qb = vp + vxb + 8 * t;
#pragma unroll
                for (int k = 0; k < E / 8; ++k) {
                    cp_async16(lu + 8 * (t + TPF * k), qa + 8 * TPF * k);
                    cp_async16(lu + W + 8 * (t + TPF * k), qb + 8 * TPF * k);
                }
            } else {
#pragma unroll
                for (int k = 0; k < E / 2; ++k) {
                    const int q = t + TPF * k;
                    cp_async16(land + 2 * q, a.Z + rowoff + 2 * q);
                }
                if (WT) {   // the weight rows of the two planes: W floats each, behind the Z row
                    float* lw = reinterpret_cast<float*>(land + W);
                    const float* qa = wv + pxa + 4 * t;
                    const float* qb = wv + pxb + 4 * t;
#pragma unroll
                    for (int k = 0; k < E / 4; ++k) {
                        cp_async16(lw + 4 * (t + TPF * k), qa + 4 * TPF * k);
                        cp_async16(lw + W + 4 * (t + TPF * k), qb + 4 * TPF * k);
                    }
                }
            }
            cp_async_commit();
            fft_run_tail<P, +1>(x, buf, tw, t, addr, sync);
            cp_async_wait_all();
            sync();
            if (MODE == ROWS_RATIO) {
                const uint16_t* lu = reinterpret_cast<const uint16_t*>(land);
                const float tau = a.guard_rel * __uint_as_float(a.gmax[pair]);
                // guard: some pixel holds photons (phi >= 1) where the blur is below tau
                //   <=>  max over the pixels of phi (tau - b) > 0     (two packed operations and one 3-input maximum)
                float gpos = 0.f;
                const float2 tau2 = make_float2(tau, tau);
#pragma unroll
                for (int e = 0; e < E; ++e) {                                 // a2
                    const int pos = t + TPF * e;
                    // uint16 -> float on the FP32 pipe: 2^23 + u is exact, subtract 2^23 (no conversion-unit trip)
                    const float2 f = sub2(make_float2(__uint_as_float(0x4B000000u | lu[pos]), __uint_as_float(0x4B000000u | lu[W + pos])),
                                          make_float2(8388608.f, 8388608.f));
                    const float2 g = mul2(f, sub2(tau2, x[e]));
                    gpos = fmaxf(gpos, fmaxf(g.x, g.y));
                    x[e].x = div_approx(f.x, fmaxf(x[e].x, a.eps));
                    x[e].y = div_approx(f.y, fmaxf(x[e].y, a.eps));
                }
                if (valid && gpos > 0.f) a.gflag[pair] = 1u;
                sync();
            } else {
                if (WT) {
                    const float* lw = reinterpret_cast<const float*>(land + W);
#pragma unroll
                    for (int e = 0; e < E; ++e) {                             // a4w: q <- w q + (1 - w)
                        const float w0 = lw[t + TPF * e], w1 = lw[W + t + TPF * e];
                        x[e] = make_float2(fmaf(w0, x[e].x, 1.f - w0), fmaf(w1, x[e].y, 1.f - w1));
                    }
                }
#pragma unroll
                for (int e = 0; e < E; ++e) {                                 // a4
                    const float2 z = land[t + TPF * e];
                    x[e] = make_float2(z.x * x[e].x, z.y * x[e].y);
                }
                sync();
                if (a.final) {   // last update: psi is the result (uniform over the grid)
                    if (more) issue_S(next_row);
#pragma unroll
                    for (int e = 0; e < E; ++e) {
                        if (a.out16) {
                            if (st_a) a.out16[pxa + t + TPF * e] = to_u16(x[e].x);
                            if (st_b) a.out16[pxb + t + TPF * e] = to_u16(x[e].y);
                        } else {
                            if (st_a) a.out[pxa + t + TPF * e] = x[e].x;
                            if (st_b) a.out[pxb + t + TPF * e] = x[e].y;
                        }
                    }
                    continue;
                }
                if (valid) {
#pragma unroll
                    for (int e = 0; e < E; ++e) Zrow[TPF * e] = x[e];
                }
            }
            fft_run_head<P, -1>(x, buf, tw, t, addr, sync);
            if (more) issue_S(next_row);
            fft_run_tail<P, -1>(x, buf, tw, t, addr, sync);
        }
        if (valid) {
#pragma unroll
            for (int e = 0; e < E; ++e) Srow[Sstep * e] = x[e];
        }
    }
}

// ---------------------------------------------------------------------------------------------
// column passes: forward column FFT, . OTF (or its conjugate), inverse column FFT, in place
// ---------------------------------------------------------------------------------------------
// rows per TMA box of a column slice: the largest supported divisor of H up to 256 (a box dimension is at most 256)
__host__ __device__ constexpr int col_box_h(int H) {
    return H <= 256 ? H : H % 256 == 0 ? 256 : H % 200 == 0 ? 200 : H % 192 == 0 ? 192 : H % 160 == 0 ? 160 : 128;
}

// 2D tiled tensor copy shared -> global (SASS UTMASTG), bulk-group completion
__device__ __forceinline__ void tma_2d_s2g(const CUtensorMap* map, int x, int y, const void* src) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];"
                 ::"l"(map), "r"(x), "r"(y), "r"(smem_u32(src)) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// Column pass fed and drained by the TMA unit.  The spectrum is a 2D tensor of 128-byte rows
// (tile-major: row index (pair * W/16 + tile) * H + p); a team's slice of an item is the box of
// 32 bytes x H rows at column offset 8 * (team's column group) floats.  One lane per team issues the
// box load of the NEXT item into the team's exchange region when the inverse transform has done its
// last exchange, and the box store of the results from a second region -- no global load or store
// instruction, and no L1 tag traffic, is left in the loop.
template <class P, int NT, bool OTF_REGS, int MINB, int CPT = 4>
__global__ void __launch_bounds__(NT, MINB)
fft2_cols_tma_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ CUtensorMap omap,
                     const float2* __restrict__ otf, int conj_otf, int pairs, int W, const float2* __restrict__ tw_g) {
    constexpr int E = P::E, TPF = P::TPF, H = P::N, TEAM = CPT * TPF, NTEAM = NT / TEAM, TC = CPT * NTEAM;
    constexpr int BOXH = col_box_h(H);
    static_assert(H % BOXH == 0 && (CPT == 4 || CPT == 8 || CPT == 16), "whole boxes; a team owns whole 32-byte sectors of a row");
    static_assert(NT % TEAM == 0 && TEAM % 32 == 0 && (TEAM == 32 || NTEAM <= 15), "column teams are whole warps");
    extern __shared__ __align__(128) float2 smem_cols3[];
    constexpr int TW = (P::S - 1) * E * TPF;                  // a multiple of 16 float2: regions stay 128-byte aligned
    static_assert(TW % 16 == 0, "twiddle table keeps the regions aligned");
    float2* tw = smem_cols3;                                  // [(S-1) E][TPF]
    // the exchange region (padded: H + H / R0 slots per column) is the landing zone of the next item
    constexpr int HP = H + H / P::radix(0);
    static_assert((HP * CPT) % 16 == 0, "regions stay 128-byte aligned");
    float2* buf = smem_cols3 + TW;                            // [NTEAM][HP][CPT]  exchange regions / landing zones
    float2* obuf = buf + NTEAM * HP * CPT;                    // [NTEAM][H][CPT]  OTF slices, then results on their way out
    uint64_t* bars = reinterpret_cast<uint64_t*>(obuf + NTEAM * H * CPT);   // [2][NTEAM]
    if (threadIdx.x < 2 * NTEAM) mbar_init(&bars[threadIdx.x], 1);
    if (threadIdx.x == 0) fence_mbar_init();
    for (int k = threadIdx.x; k < TW; k += NT) tw[k] = tw_g[k];
    __syncthreads();
    pdl_launch_dependents();
    const int team = threadIdx.x / TEAM, l = threadIdx.x % TEAM;
    // ShflTail plans (2048 points): threads t and t ^ 32 of a column sit in lanes l and l ^ 16 of one warp, so that the
    // exchange in front of the radix-2 stage goes through shuffles (fft_stage); a half-warp still covers 4 consecutive t
    // x CPT = 4 columns = one 128-byte line of the regions
    static_assert(!shfl_tail<P>() || (CPT == 4 && TPF == 64), "shuffle exchange: four columns, 64 threads per column");
    const int c4 = l % CPT;
    const int t = shfl_tail<P>() ? (((l >> 4) & 1) << 5) | (((l >> 5) & 7) << 2) | ((l >> 2) & 3) : l / CPT;
    const ColAddrPad<P, CPT> addr{team * HP * CPT + c4};
    const TeamSync<TEAM> sync{team};
    const float sgn = conj_otf == 1 ? -1.f : 1.f;
    const bool real_otf = conj_otf == 2;         // omap / otf describe a float array (mvd_fft.cu: real transfer functions)
    float2* land = buf + team * HP * CPT;
    float2* outz = obuf + team * H * CPT;
    uint64_t* full = &bars[team];
    uint64_t* full_otf = &bars[NTEAM + team];   // !OTF_REGS: the team's OTF slice lands in the out region
    const int tiles = W / TC;            // column groups of TC columns
    const int items = tiles * pairs;
    auto first_col = [&](int item) { return (item % tiles) * TC + team * CPT; };
    auto plane_off = [&](int x) { return (size_t)(x >> 4) * (H * 16) + (x & 15); };
    // tensor coordinates of the team's slice of an item: x in floats within the 128-byte row, y = tile row
    auto box_x = [&](int item) { return 2 * (first_col(item) & 15); };
    auto box_y = [&](int item) { return ((item / tiles) * (W / 16) + (first_col(item) >> 4)) * H; };
    auto issue = [&](int item) {   // one lane
        fence_proxy_async();
        mbar_arrive_expect_tx(full, (uint32_t)(sizeof(float2) * H * CPT));
#pragma unroll
        for (int b = 0; b < H / BOXH; ++b) tma_2d_g2s(land + b * BOXH * CPT, &tmap, box_x(item), box_y(item) + b * BOXH, full);
    };

    int item = blockIdx.x;
    float2 o[OTF_REGS ? E : 1];
    if (OTF_REGS && item < items) {   // the OTF is written once in mvd_create: no dependency on the previous kernel
        const int xg = first_col(item) + c4;
        if (real_otf) {
            const float* of = reinterpret_cast<const float*>(otf);
#pragma unroll
            for (int e = 0; e < E; ++e) o[e] = make_float2(__ldg(of + plane_off(xg) + (size_t)(t + TPF * e) * 16), 0.f);
        } else {
#pragma unroll
            for (int e = 0; e < E; ++e) {
                o[e] = __ldg(otf + plane_off(xg) + (size_t)(t + TPF * e) * 16);
                o[e].y *= sgn;
            }
        }
    }
    pdl_wait();
    if (item < items && l == 0) issue(item);
    uint32_t phase = 0;
    for (; item < items; item += gridDim.x) {
        const int xg = first_col(item) + c4;
        float2 x[E];
        mbar_wait(full, phase);
        phase ^= 1;
#pragma unroll
        for (int e = 0; e < E; ++e) x[e] = land[(t + TPF * e) * CPT + c4];
        sync();
        if (!OTF_REGS && l == 0) {
            // The OTF slice of these columns (same tile-major tensor shape as S, one "pair" per view)
            // comes through the TMA unit into the out region, which the previous item's results have
            // left by now; it has the whole forward transform's time to arrive.
            bulk_wait_read();
            fence_proxy_async();
            const int oy = (first_col(item) >> 4) * H;
            if (real_otf) {     // a REAL transfer function (centro-symmetric PSF): one float per element, half the box
                mbar_arrive_expect_tx(full_otf, (uint32_t)(sizeof(float) * H * CPT));
#pragma unroll
                for (int b = 0; b < H / BOXH; ++b)
                    tma_2d_g2s(reinterpret_cast<float*>(outz) + b * BOXH * CPT, &omap, box_x(item) >> 1, oy + b * BOXH, full_otf);
            } else {
                mbar_arrive_expect_tx(full_otf, (uint32_t)(sizeof(float2) * H * CPT));
#pragma unroll
                for (int b = 0; b < H / BOXH; ++b) tma_2d_g2s(outz + b * BOXH * CPT, &omap, box_x(item), oy + b * BOXH, full_otf);
            }
        }
        fft_run<P, -1>(x, buf, tw, t, addr, sync);
        if (OTF_REGS) {
            if (real_otf) {
#pragma unroll
                for (int e = 0; e < E; ++e) x[e] = mul2(x[e], make_float2(o[e].x, o[e].x));
            } else {
#pragma unroll
                for (int e = 0; e < E; ++e) x[e] = cmul(x[e], o[e]);
            }
        } else {
            mbar_wait(full_otf, phase ^ 1);      // same parity sequence as `full`: one completion per item
            if (real_otf) {
                const float* of = reinterpret_cast<const float*>(outz);
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    const float w = of[(t + TPF * e) * CPT + c4];
                    x[e] = mul2(x[e], make_float2(w, w));
                }
            } else {
#pragma unroll
            for (int e = 0; e < E; ++e) {
                float2 w = outz[(t + TPF * e) * CPT + c4];
                w.y *= sgn;
                x[e] = cmul(x[e], w);
            }
            }
            // no barrier here: the inverse transform's exchanges (team barriers) lie between these
            // reads of the out region and the next writes to it
        }
        fft_run_head<P, +1>(x, buf, tw, t, addr, sync);
        if (l == 0) {
            if (item + (int)gridDim.x < items) issue(item + gridDim.x);
            if (OTF_REGS) bulk_wait_read();   // the previous item's results have left the out region
        }
        fft_run_tail<P, +1>(x, buf, tw, t, addr, sync);
        if (OTF_REGS) sync();            // ... and every thread of the team knows it (without OTF registers lane 0
                                         // waited at the start of the item, many team barriers ago)
#pragma unroll
        for (int e = 0; e < E; ++e) outz[(t + TPF * e) * CPT + c4] = x[e];
        fence_proxy_async();
        sync();
        if (l == 0) {
#pragma unroll
            for (int b = 0; b < H / BOXH; ++b) tma_2d_s2g(&tmap, box_x(item), box_y(item) + b * BOXH, outz + b * BOXH * CPT);
            bulk_commit();
        }
    }
    if (l == 0) bulk_wait_read();
}

// Column pass for plans that keep their OTF in registers (256-point columns), two regions per team in PING-PONG: item i
// transforms in the region its slice landed in and leaves its results there for the box store, while item i + 1's slice
// is requested into the other region at the TOP of item i (as soon as item i - 1's results have left it) -- a whole item
// of lead time instead of one register-only stage, at no extra shared memory (fft2_cols_tma_kernel's second region
// only holds results on their way out).
template <class P, int NT, int MINB, int CPT = 4>
__global__ void __launch_bounds__(NT, MINB)
fft2_cols_pp_kernel(const __grid_constant__ CUtensorMap tmap, const float2* __restrict__ otf, int conj_otf, int pairs, int W,
                    const float2* __restrict__ tw_g) {
    constexpr int E = P::E, TPF = P::TPF, H = P::N, TEAM = CPT * TPF, NTEAM = NT / TEAM, TC = CPT * NTEAM;
    constexpr int BOXH = col_box_h(H);
    static_assert(H % BOXH == 0 && NT % TEAM == 0 && TEAM % 32 == 0 && (TEAM == 32 || NTEAM <= 15), "whole boxes, whole-warp teams");
    extern __shared__ __align__(128) float2 smem_cols6[];
    constexpr int TW = (P::S - 1) * E * TPF;
    constexpr int HP = H + H / P::radix(0);
    static_assert(TW % 16 == 0 && (HP * CPT) % 16 == 0, "regions stay 128-byte aligned");
    float2* tw = smem_cols6;                                  // [(S-1) E][TPF]
    float2* buf = smem_cols6 + TW;                            // [NTEAM][2][HP][CPT]
    uint64_t* bars = reinterpret_cast<uint64_t*>(buf + NTEAM * 2 * HP * CPT);   // [NTEAM]
    if (threadIdx.x < NTEAM) mbar_init(&bars[threadIdx.x], 1);
    if (threadIdx.x == 0) fence_mbar_init();
    for (int k = threadIdx.x; k < TW; k += NT) tw[k] = tw_g[k];
    __syncthreads();
    pdl_launch_dependents();
    const int team = threadIdx.x / TEAM, l = threadIdx.x % TEAM;
    const int c4 = l % CPT, t = l / CPT;
    const ColAddrPad<P, CPT> addr{c4};                        // relative to the region in use
    const TeamSync<TEAM> sync{team};
    const float sgn = conj_otf == 1 ? -1.f : 1.f;
    const bool real_otf = conj_otf == 2;
    float2* reg0 = buf + team * 2 * HP * CPT;
    uint64_t* full = &bars[team];
    const int tiles = W / TC;
    const int items = tiles * pairs;
    auto first_col = [&](int item) { return (item % tiles) * TC + team * CPT; };
    auto plane_off = [&](int x) { return (size_t)(x >> 4) * (H * 16) + (x & 15); };
    auto box_x = [&](int item) { return 2 * (first_col(item) & 15); };
    auto box_y = [&](int item) { return ((item / tiles) * (W / 16) + (first_col(item) >> 4)) * H; };
    auto issue = [&](int item, float2* dst) {   // one lane
        fence_proxy_async();
        mbar_arrive_expect_tx(full, (uint32_t)(sizeof(float2) * H * CPT));
#pragma unroll
        for (int b = 0; b < H / BOXH; ++b) tma_2d_g2s(dst + b * BOXH * CPT, &tmap, box_x(item), box_y(item) + b * BOXH, full);
    };

    int item = blockIdx.x;
    float2 o[E];
    if (item < items) {   // the OTF is written once in mvd_create: no dependency on the previous kernel
        const int xg = first_col(item) + c4;
        if (real_otf) {
            const float* of = reinterpret_cast<const float*>(otf);
#pragma unroll
            for (int e = 0; e < E; ++e) o[e] = make_float2(__ldg(of + plane_off(xg) + (size_t)(t + TPF * e) * 16), 0.f);
        } else {
#pragma unroll
            for (int e = 0; e < E; ++e) {
                o[e] = __ldg(otf + plane_off(xg) + (size_t)(t + TPF * e) * 16);
                o[e].y *= sgn;
            }
        }
    }
    pdl_wait();
    if (item < items && l == 0) issue(item, reg0);
    uint32_t phase = 0;
    int cur = 0;
    for (; item < items; item += gridDim.x, cur ^= 1) {
        float2* X = reg0 + cur * HP * CPT;            // this item's slice, exchange region, results
        float2* Y = reg0 + (cur ^ 1) * HP * CPT;      // the next item's landing zone
        float2 x[E];
        mbar_wait(full, phase);
        phase ^= 1;
#pragma unroll
        for (int e = 0; e < E; ++e) x[e] = X[(t + TPF * e) * CPT + c4];
        sync();
        if (l == 0 && item + (int)gridDim.x < items) {
            bulk_wait_read();                         // the previous item's results have left Y
            issue(item + gridDim.x, Y);
        }
        fft_run<P, -1>(x, X, tw, t, addr, sync);
        if (real_otf) {
#pragma unroll
            for (int e = 0; e < E; ++e) x[e] = mul2(x[e], make_float2(o[e].x, o[e].x));
        } else {
#pragma unroll
            for (int e = 0; e < E; ++e) x[e] = cmul(x[e], o[e]);
        }
        fft_run<P, +1>(x, X, tw, t, addr, sync);      // (its last exchange ends with a team barrier: X is free)
#pragma unroll
        for (int e = 0; e < E; ++e) X[(t + TPF * e) * CPT + c4] = x[e];
        fence_proxy_async();
        sync();
        if (l == 0) {
#pragma unroll
            for (int b = 0; b < H / BOXH; ++b) tma_2d_s2g(&tmap, box_x(item), box_y(item) + b * BOXH, X + b * BOXH * CPT);
            bulk_commit();
        }
    }
    if (l == 0) bulk_wait_read();
}

// Column pass for lengths H = RA x RB whose two radices differ (800 = 25 x 32): a two-stage transform in which the
// stages use different numbers of threads.  RB threads (one warp's worth per column) each hold rows t + RB e and
// run one radix-RA butterfly; after the exchange RA of them hold RB elements each and run one radix-RB butterfly
// (X[k1 + RA k2] in thread k1), multiply by the OTF, run the inverse radix-RB butterfly and hand the data back for
// the inverse radix-RA stage.  Against the uniform 40 x 20 plan (20 threads x 40 elements, five warps per team of
// eight columns) a team is FOUR columns x 32 threads = four warps (one per scheduler), holds half the shared memory
// and at most 64 data registers per thread, so four teams are resident per SM instead of two; the price is that
// 7 of 32 lanes idle in the middle stage.  Loads, OTF slices and stores go through the TMA unit exactly as in
// fft2_cols_tma_kernel.  Twiddles: tw[k1 RB + t] = exp(-2 pi i t k1 / H).
template <int RA, int RB, int NT, int MINB>
__global__ void __launch_bounds__(NT, MINB)
fft2_cols_nu_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ CUtensorMap omap,
                    int conj_otf, int pairs, int W, const float2* __restrict__ tw_g) {
    constexpr int H = RA * RB, TPF = RB, CPT = 4, TEAM = CPT * TPF, NTEAM = NT / TEAM, TC = CPT * NTEAM;
    constexpr int BOXH = col_box_h(H);
    static_assert(RB == 32 && RA <= RB, "one warp's worth of threads per column");
    static_assert(H % BOXH == 0 && NT % TEAM == 0 && NTEAM <= 15, "whole boxes, whole teams");
    extern __shared__ __align__(128) float2 smem_cols5[];
    constexpr int TW = RA * RB;
    static_assert(TW % 16 == 0, "twiddle table keeps the regions aligned");
    float2* tw = smem_cols5;                                  // [RA][RB]
    constexpr int PB = (RA * (RB + 1) * CPT + 15) / 16 * 16;  // exchange region: slot (k1, t) at k1 (RB + 1) + t, 128-byte aligned
    float2* buf = smem_cols5 + TW;                            // [NTEAM][PB]  exchange regions / landing zones ([H][CPT] linear)
    float2* obuf = buf + NTEAM * PB;                          // [NTEAM][H][CPT]  OTF slices, then results on their way out
    uint64_t* bars = reinterpret_cast<uint64_t*>(obuf + NTEAM * H * CPT);   // [2][NTEAM]
    if (threadIdx.x < 2 * NTEAM) mbar_init(&bars[threadIdx.x], 1);
    if (threadIdx.x == 0) fence_mbar_init();
    for (int k = threadIdx.x; k < TW; k += NT) tw[k] = tw_g[k];
    __syncthreads();
    pdl_launch_dependents();
    const int team = threadIdx.x / TEAM, l = threadIdx.x % TEAM;
    const int c = l % CPT, t = l / CPT;
    const TeamSync<TEAM> sync{team};
    const float sgn = conj_otf == 1 ? -1.f : 1.f;
    const bool real_otf = conj_otf == 2;         // omap describes a float array (real transfer functions)
    float2* land = buf + team * PB;
    float2* outz = obuf + team * H * CPT;
    uint64_t* full = &bars[team];
    uint64_t* full_otf = &bars[NTEAM + team];
    // exchange slot of (k1, t) = k1 (RB + 1) + t: four consecutive t (stage A stores) and four consecutive k1 (stage B,
    // RB + 1 = 1 mod 4) both spread over the four 32-byte groups of a 128-byte line, and every address is an immediate
    // offset from one per-thread base
    auto slot = [&](int k1, int tt) { return land + ((k1 * (RB + 1) + tt) * CPT + c); };
    const int tiles = W / TC;
    const int items = tiles * pairs;
    auto first_col = [&](int item) { return (item % tiles) * TC + team * CPT; };
    auto box_x = [&](int item) { return 2 * (first_col(item) & 15); };
    auto box_y = [&](int item) { return ((item / tiles) * (W / 16) + (first_col(item) >> 4)) * H; };
    auto issue = [&](int item) {   // one lane
        fence_proxy_async();
        mbar_arrive_expect_tx(full, (uint32_t)(sizeof(float2) * H * CPT));
#pragma unroll
        for (int b = 0; b < H / BOXH; ++b) tma_2d_g2s(land + b * BOXH * CPT, &tmap, box_x(item), box_y(item) + b * BOXH, full);
    };
    const bool act = t < RA;    // threads of the radix-RB stage

    int item = blockIdx.x;
    pdl_wait();
    if (item < items && l == 0) issue(item);
    uint32_t phase = 0;
    for (; item < items; item += gridDim.x) {
        float2 xa[RA];
        mbar_wait(full, phase);
        phase ^= 1;
#pragma unroll
        for (int e = 0; e < RA; ++e) xa[e] = land[(t + RB * e) * CPT + c];
        sync();
        if (l == 0) {   // this item's OTF slice -> the out region, which the previous item's results have left by now
            bulk_wait_read();
            fence_proxy_async();
            const int oy = (first_col(item) >> 4) * H;
            if (real_otf) {
                mbar_arrive_expect_tx(full_otf, (uint32_t)(sizeof(float) * H * CPT));
#pragma unroll
                for (int b = 0; b < H / BOXH; ++b)
                    tma_2d_g2s(reinterpret_cast<float*>(outz) + b * BOXH * CPT, &omap, box_x(item) >> 1, oy + b * BOXH, full_otf);
            } else {
                mbar_arrive_expect_tx(full_otf, (uint32_t)(sizeof(float2) * H * CPT));
#pragma unroll
                for (int b = 0; b < H / BOXH; ++b) tma_2d_g2s(outz + b * BOXH * CPT, &omap, box_x(item), oy + b * BOXH, full_otf);
            }
        }
        Bfly<RA, -1>::run(xa);
#pragma unroll
        for (int k1 = 1; k1 < RA; ++k1) xa[k1] = cmul(xa[k1], tw[k1 * RB + t]);
#pragma unroll
        for (int k1 = 0; k1 < RA; ++k1) *slot(k1, t) = xa[k1];
        sync();
        if (act) {      // thread t is k1: it reads, transforms and writes back its own RB slots
            float2 xb[RB];
#pragma unroll
            for (int j = 0; j < RB; ++j) xb[j] = *slot(t, j);
            Bfly<RB, -1>::run(xb);
            mbar_wait(full_otf, phase ^ 1);      // same parity sequence as `full`: one completion per item
            if (real_otf) {
                const float* of = reinterpret_cast<const float*>(outz);
#pragma unroll
                for (int k2 = 0; k2 < RB; ++k2) {
                    const float w = of[(t + RA * k2) * CPT + c];
                    xb[k2] = mul2(xb[k2], make_float2(w, w));
                }
            } else {
#pragma unroll
                for (int k2 = 0; k2 < RB; ++k2) {
                    float2 w = outz[(t + RA * k2) * CPT + c];
                    w.y *= sgn;
                    xb[k2] = cmul(xb[k2], w);
                }
            }
            Bfly<RB, +1>::run(xb);
#pragma unroll
            for (int j = 0; j < RB; ++j) *slot(t, j) = xb[j];
        }
        sync();
#pragma unroll
        for (int k1 = 0; k1 < RA; ++k1) xa[k1] = *slot(k1, t);
        sync();
        if (l == 0 && item + (int)gridDim.x < items) issue(item + gridDim.x);
#pragma unroll
        for (int k1 = 1; k1 < RA; ++k1) xa[k1] = cmulc(xa[k1], tw[k1 * RB + t]);
        Bfly<RA, +1>::run(xa);
#pragma unroll
        for (int e = 0; e < RA; ++e) outz[(t + RB * e) * CPT + c] = xa[e];
        fence_proxy_async();
        sync();
        if (l == 0) {
#pragma unroll
            for (int b = 0; b < H / BOXH; ++b) tma_2d_s2g(&tmap, box_x(item), box_y(item) + b * BOXH, outz + b * BOXH * CPT);
            bulk_commit();
        }
    }
    if (l == 0) bulk_wait_read();
}

// ---------------------------------------------------------------------------------------------
// host-side descriptor of a v2 length
// ---------------------------------------------------------------------------------------------
template <class Kern, class... Args>
inline cudaError_t launch_pdl(Kern kern, dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, args...);
}

template <class P, int NT, class PC, int NTC, bool OTF_REGS, int MINB, bool TMA = true, int CPT = 4, int RMINB = 2, bool PP = false>
struct OpsFor2 {
    static_assert(TMA, "every generation-2 column kernel is TMA-fed");
    static_assert(!PP || OTF_REGS, "the ping-pong column kernel keeps its OTF in registers");
    static_assert(P::N == PC::N, "row and column plan of one entry describe the same length");
    static constexpr size_t kRowSmem = sizeof(float2) * ((size_t)(P::S - 1) * P::E * P::TPF + (size_t)(NT / P::TPF) * row_pitch<P>(P::N));
    static constexpr size_t kRowSmemW = sizeof(float2) * ((size_t)(P::S - 1) * P::E * P::TPF + (size_t)(NT / P::TPF) * row_pitch<P>(2 * P::N));
    static constexpr int kRowCpsW = (int)((228u * 1024u) / (kRowSmemW + 1024)) < RMINB ? (int)((228u * 1024u) / (kRowSmemW + 1024)) : RMINB;
    static_assert(kRowSmemW <= 227u * 1024u && kRowCpsW >= 1, "the weighted update kernel fits one CTA");
    static constexpr int kTeam = CPT * PC::TPF, kNTeam = NTC / kTeam, kTC = CPT * kNTeam;
    static constexpr size_t kColSmem = sizeof(float2) * ((size_t)(PC::S - 1) * PC::E * PC::TPF +
                                                         (size_t)kNTeam * CPT * (PP ? 2 * (PC::N + PC::N / PC::radix(0))
                                                                                    : TMA ? 2 * PC::N + PC::N / PC::radix(0) : PC::N)) +
                                       (TMA ? 2 * sizeof(uint64_t) * kNTeam : 0);

    static cudaError_t rows(int mode, const RowArgs& a, const float2* tw, int grid, cudaStream_t st) {
        if (mode == ROWS_FIRST) return launch_pdl(fft2_rows_kernel<P, ROWS_FIRST, NT, RMINB>, dim3(grid), dim3(NT), kRowSmem, st, a, tw);
        if (mode == ROWS_RATIO) return launch_pdl(fft2_rows_kernel<P, ROWS_RATIO, NT, RMINB>, dim3(grid), dim3(NT), kRowSmem, st, a, tw);
        if (mode == ROWS_UPDATE_W) return launch_pdl(fft2_rows_kernel<P, ROWS_UPDATE_W, NT, kRowCpsW>, dim3(grid), dim3(NT), kRowSmemW, st, a, tw);
        return launch_pdl(fft2_rows_kernel<P, ROWS_UPDATE, NT, RMINB>, dim3(grid), dim3(NT), kRowSmem, st, a, tw);
    }
    static cudaError_t cols(const CUtensorMap& tmap, const CUtensorMap& otf_map, float2* S, const float2* otf, int conj_otf, int pairs, int W,
                            const float2* tw, dim3 grid, cudaStream_t st) {
        if constexpr (PP)
            return launch_pdl(fft2_cols_pp_kernel<PC, NTC, MINB, CPT>, grid, dim3(NTC), kColSmem, st, tmap, otf, conj_otf, pairs, W, tw);
        else
            return launch_pdl(fft2_cols_tma_kernel<PC, NTC, OTF_REGS, MINB, CPT>, grid, dim3(NTC), kColSmem, st, tmap, otf_map, otf, conj_otf, pairs, W, tw);
    }
    static cudaError_t prepare_rows() {
        cudaError_t e;
        e = cudaFuncSetAttribute(fft2_rows_kernel<P, ROWS_FIRST, NT, RMINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRowSmem);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(fft2_rows_kernel<P, ROWS_RATIO, NT, RMINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRowSmem);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(fft2_rows_kernel<P, ROWS_UPDATE_W, NT, kRowCpsW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRowSmemW);
        if (e != cudaSuccess) return e;
        return cudaFuncSetAttribute(fft2_rows_kernel<P, ROWS_UPDATE, NT, RMINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRowSmem);
    }
    static cudaError_t prepare_cols() {
        if constexpr (PP)
            return cudaFuncSetAttribute(fft2_cols_pp_kernel<PC, NTC, MINB, CPT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kColSmem);
        else
            return cudaFuncSetAttribute(fft2_cols_tma_kernel<PC, NTC, OTF_REGS, MINB, CPT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kColSmem);
    }
    static SizeOps make() {
        SizeOps o;
        o.N = P::N;
        o.row = PlanInfo{P::E, P::TPF, P::S, {P::radix(0), P::radix(1), P::radix(2), P::radix(3), P::radix(4)}};
        o.col = PlanInfo{PC::E, PC::TPF, PC::S, {PC::radix(0), PC::radix(1), PC::radix(2), PC::radix(3), PC::radix(4)}};
        o.row_threads = NT;
        o.row_smem = kRowSmem;
        o.col_smem = kColSmem; o.col_tc = kTC; o.col_box_h = col_box_h(PC::N); o.col_box_w = 2 * CPT;
        o.rows = &rows; o.cols = &cols; o.prepare_rows = &prepare_rows; o.prepare_cols = &prepare_cols;
        o.generation = 2;
        o.row_cps = RMINB;
        o.row_cps_w = kRowCpsW;
        o.col_cps = MINB;
        o.col_otf_regs = OTF_REGS ? 1 : 0;
        o.col_real_otf = TMA ? 1 : 0;
        return o;
    }
};

// A column-only length served by fft2_cols_nu_kernel.
template <int RA, int RB, int NTC, int MINB>
struct ColsNu2 {
    static constexpr int kN = RA * RB, kNTeam = NTC / (4 * RB), kTC = 4 * kNTeam;
    static constexpr int kBoxH = col_box_h(kN);
    static constexpr size_t kColSmem = sizeof(float2) * ((size_t)RA * RB + (size_t)kNTeam * ((RA * (RB + 1) * 4 + 15) / 16 * 16 + kN * 4)) +
                                       2 * sizeof(uint64_t) * kNTeam;
    static cudaError_t cols(const CUtensorMap& tmap, const CUtensorMap& otf_map, float2*, const float2*, int conj_otf, int pairs, int W,
                            const float2* tw, dim3 grid, cudaStream_t st) {
        return launch_pdl(fft2_cols_nu_kernel<RA, RB, NTC, MINB>, grid, dim3(NTC), kColSmem, st, tmap, otf_map, conj_otf, pairs, W, tw);
    }
    static cudaError_t prepare_cols() {
        return cudaFuncSetAttribute(fft2_cols_nu_kernel<RA, RB, NTC, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kColSmem);
    }
    static SizeOps make() {
        SizeOps o;
        o.N = kN;
        o.row = PlanInfo{0, 0, 0, {0, 0, 0, 0, 0}};
        o.col = PlanInfo{RB, RB, 2, {RA, RB, 1, 1, 1}};
        o.row_threads = 0; o.row_smem = 0;
        o.col_smem = kColSmem; o.col_tc = kTC; o.col_box_h = kBoxH; o.col_box_w = 8;
        o.rows = nullptr; o.cols = &cols; o.prepare_rows = nullptr; o.prepare_cols = &prepare_cols;
        o.generation = 2; o.row_cps = 0; o.col_cps = MINB; o.col_otf_regs = 0; o.col_tw_custom = 1; o.col_real_otf = 1;
        return o;
    }
};

}  // namespace mvdfft
