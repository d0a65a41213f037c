"""GPU-vs-oracle parity, through the C ABI (binding -> libmvd.so).  Run with -m gpu on the B200 box.

Element-by-element comparison on the same seeded inputs; tolerance per north_star (parity_util).
Integer / exact work (uint16 ingest, iterations = 0, delta PSFs, chunking, host pipeline) is bit-exact.
Every case runs on both engines where the engine supports the shape.
"""
import json
import os

import numpy as np
import pytest

from oracle import mvd_oracle
from paper_1503_07998_b200 import binding, build, synth
from parity_util import assert_parity

pytestmark = pytest.mark.gpu

PATHS = [binding.PATH_DIRECT, binding.PATH_FFT]
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


@pytest.fixture(scope="module", autouse=True)
def _lib():
    build.build()
    return binding.lib()


def _need(path, W, H, K):
    if not binding.path_supported(path, W, H, K):
        pytest.skip(f"{binding.PATH_NAMES[path]} engine does not take {W}x{H} K={K}")


def _run(views, psfs, T, path, **kw):
    return binding.deconvolve(views, psfs, T, float(synth.EPS), path=path, **kw)


# ---------------------------------------------------------------------------------------------
# BASELINE.json configs
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("path", PATHS)
def test_config1_full_volume(path):
    cfg = synth.config(1)
    _need(path, cfg.W, cfg.H, cfg.K)
    psfs, views = synth.config_psfs(1), synth.views(cfg)
    ref = mvd_oracle.deconvolve(views, psfs, cfg.T, cfg.eps)
    out = _run(views, psfs, cfg.T, path)
    assert_parity(out, ref, f"config1 {binding.PATH_NAMES[path]}")


@pytest.mark.parametrize("path", PATHS)
def test_config2_plane_subset_full_size(path):
    """Full-size 512x256 planes, K = 21, T = 10 (the bench workload's shape), oracle computed live."""
    cfg = synth.config(2)
    _need(path, cfg.W, cfg.H, cfg.K)
    planes = [0, 255, 256, 511, 100, 37]
    psfs, views = synth.config_psfs(2), synth.views(cfg, planes)
    ref = mvd_oracle.deconvolve(views, psfs, cfg.T, cfg.eps)
    out = _run(views, psfs, cfg.T, path)
    assert_parity(out, ref, f"config2 {binding.PATH_NAMES[path]}")


@pytest.mark.parametrize("cid", [3, 4, 5])
def test_large_configs_against_stored_oracle_planes(cid):
    """Configs 3-5 at full plane size against oracle planes stored by tests/golden/make_golden.py."""
    fn = os.path.join(GOLDEN, f"config{cid}_samples.json")
    if not os.path.exists(fn):
        pytest.skip(f"{fn} not generated yet")
    with open(fn) as f:
        g = json.load(f)
    cfg = synth.config(cid)
    psfs = synth.config_psfs(cid)
    planes = [rec["plane"] for rec in g["planes"]]
    views = synth.views(cfg, planes, psfs)
    for k, rec in enumerate(g["planes"]):   # the stored planes belong to exactly these inputs
        assert [int(views[v, k].astype(np.int64).sum()) for v in range(cfg.V)] == rec["view_sums"]
    out = binding.deconvolve(views, psfs, cfg.T, cfg.eps)   # the path mvd_create picks
    for k, rec in enumerate(g["planes"]):
        flat = out[k].astype(np.float64).ravel()
        pos, val = np.array(rec["pos"]), np.array(rec["val"])
        d = flat[pos] - val
        rel_l2 = np.sqrt((d ** 2).sum() / (val ** 2).sum())
        bright = val > 0.01 * rec["max"]
        max_rel = (np.abs(d[bright]) / val[bright]).max()
        assert rel_l2 <= 1e-4 and max_rel <= 1e-3, (cid, rec["plane"], rel_l2, max_rel)
        assert abs(flat.sum() - rec["sum"]) <= 2e-5 * rec["sum"]
        assert abs((flat ** 2).sum() - rec["sumsq"]) <= 2e-4 * rec["sumsq"]


# ---------------------------------------------------------------------------------------------
# Configs 3-5, element by element against WHOLE stored oracle planes (tests/golden/config*_planes.npz)
# ---------------------------------------------------------------------------------------------
def _whole_planes(cid):
    fn = os.path.join(GOLDEN, f"config{cid}_planes.npz")
    if not os.path.exists(fn):
        pytest.skip(f"{fn} not generated yet")
    g = np.load(fn)
    planes = [int(p) for p in g["planes"]]
    ref = np.stack([g[f"plane_{p}"] for p in planes]).astype(np.float64)
    return planes, ref, g["view_sums"], int(g["pipeline_batch"])


@pytest.mark.parametrize("path", [binding.PATH_FFT, binding.PATH_DIRECT])
@pytest.mark.parametrize("cid", [3, 4, 5])
def test_large_configs_whole_planes_both_engines(cid, path):
    """Planes {0, B-1, B, N/2, N-1} of configs 3-5 at full size as a five-plane stack (odd: the last pair is
    half empty), every pixel against the stored fp64 oracle plane, on the FFT engine AND the direct engine
    (K = 31 / 41 / 51 templated kernels)."""
    cfg = synth.config(cid)
    _need(path, cfg.W, cfg.H, cfg.K)
    planes, ref, view_sums, _ = _whole_planes(cid)
    psfs = synth.config_psfs(cid)
    views = synth.views(cfg, planes, psfs)
    for k in range(len(planes)):      # the stored planes belong to exactly these inputs
        assert [int(views[v, k].astype(np.int64).sum()) for v in range(cfg.V)] == [int(x) for x in view_sums[k]]
    out = _run(views, psfs, cfg.T, path)
    l2, pooled, mx = assert_parity(out, ref, f"config{cid} whole planes {binding.PATH_NAMES[path]}")
    print(f"config{cid} {binding.PATH_NAMES[path]}: rel L2 {l2:.2e} (pooled {pooled:.2e}) max rel {mx:.2e}")


def _load_bench():
    import importlib.util
    spec = importlib.util.spec_from_file_location("bench", os.path.join(os.path.dirname(GOLDEN), "..", "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    return bench


@pytest.mark.parametrize("cid", [3, 4, 5])
def test_large_configs_full_stack_in_the_bench_launch_configuration(cid):
    """The whole N-plane stack of configs 3-5 exactly as bench.py times it (same stack builder, default batches
    dealt to the library's internal streams), with the canonical planes that have stored oracle planes written
    at their own positions -- first, last, middle and both sides of a batch boundary of the launch
    configuration -- and compared element by element; plus, on EVERY plane, pin P12: psi >= 0, finite,
    sum(psi) = sum(phi_last)."""
    import torch
    bench = _load_bench()
    cfg = synth.config(cid)
    planes, ref, _, b_stored = _whole_planes(cid)
    psfs, views = bench.make_stack(cfg)
    canon = synth.views(cfg, planes, psfs)
    with binding.Mvd(cfg.W, cfg.H, cfg.V, psfs, cfg.K, cfg.T, cfg.eps) as m:
        B = m.get_batch_planes(cfg.N)
        where = {p: k for k, p in enumerate(planes)}          # stack position -> index into ref
        if B != b_stored:                                      # the boundary moved: put the stored pair on it
            where[B - 1], where[B] = planes.index(b_stored - 1), planes.index(b_stored)
        for pos, k in where.items():
            views[:, pos] = canon[:, k]
        assert {0, B - 1, B, cfg.N // 2, cfg.N - 1} <= set(where)
        m.reserve(cfg.N)
        dv = torch.empty((cfg.V, cfg.N, cfg.H, cfg.W), dtype=torch.int16, device="cuda")
        step = 64
        for p0 in range(0, cfg.N, step):                       # upload in slices: no second 13 GB host copy
            dv[:, p0:p0 + step] = torch.from_numpy(views[:, p0:p0 + step].view(np.int16)).cuda()
        do = torch.empty((cfg.N, cfg.H, cfg.W), dtype=torch.float32, device="cuda")
        m.deconvolve_planes(dv, do, cfg.N)
        torch.cuda.synchronize()
        assert bool(torch.isfinite(do).all()) and bool((do >= 0).all())
        got = do.sum(dim=(1, 2), dtype=torch.float64).cpu().numpy()
        want = np.array([views[-1, p].astype(np.int64).sum() for p in range(cfg.N)], dtype=np.float64)
        np.testing.assert_allclose(got, want, rtol=2e-5)
        pos = sorted(where)
        out = do[torch.tensor(pos, device="cuda")].cpu().numpy()
    assert_parity(out, ref[[where[p] for p in pos]], f"config{cid} full stack, planes {pos}")


def test_host_pipeline_with_ramp_and_odd_plane_count_is_bit_identical():
    """with the batch ramp (B/4, B/2 at both ends) and an odd n_planes every non-final batch must
    still start on an even plane, or the FFT engine pairs (2m+1, 2m+2) and the bits differ."""
    import torch
    V, W, H, K, T = 2, 256, 256, 5, 2
    N = 8 * 32 + 9                     # >= 8 B with B = 32 planes of 256 x 256 (the 2 Mvoxel floor): ramp on, odd
    pr = synth.make_problem(V, 16, W, H, K, T, seed=991)
    views = np.concatenate([np.roll(pr.views, 7 * k, axis=3) for k in range(N // 16 + 1)], axis=1)[:, :N]
    views = np.ascontiguousarray(views)
    with binding.Mvd(W, H, V, pr.psfs, K, T, pr.eps, binding.PATH_FFT) as m:
        B = m.get_batch_planes(N)
        assert B >= 8 and N >= 8 * B and N % 2 == 1
        hv = torch.from_numpy(views.view(np.int16)).pin_memory()
        ho = torch.empty((N, H, W), dtype=torch.float32).pin_memory()
        m.deconvolve_host(hv, ho, N)
        dv = hv.cuda()
        do = torch.empty((N, H, W), dtype=torch.float32, device="cuda")
        m.deconvolve_planes(dv, do, N)
        torch.cuda.synchronize()
        assert torch.equal(ho, do.cpu())
    ref = mvd_oracle.deconvolve(np.ascontiguousarray(views[:, -3:]), pr.psfs, T, pr.eps)
    assert_parity(ho.numpy()[-3:], ref, "odd tail of the ramped pipeline")


@pytest.mark.parametrize("path", PATHS)
def test_three_and_four_pipeline_streams_are_bit_identical(path):
    """mvd_set_pipeline_streams: the paper's three streams and the default four give the same bits as the resident call."""
    import torch
    V, N, W, H, K, T = 2, 23, 96, 64, 7, 3
    _need(path, W, H, K)
    pr = synth.make_problem(V, N, W, H, K, T, seed=99)
    ref = _run(pr.views, pr.psfs, T, path)
    hv = torch.from_numpy(pr.views.view(np.int16)).pin_memory()
    for n in (3, 4):
        ho = torch.empty((N, H, W), dtype=torch.float32).pin_memory()
        with binding.Mvd(W, H, V, pr.psfs, K, T, float(synth.EPS), path) as m:
            m.set_pipeline_streams(n)
            m.set_batch_planes(2)
            m.deconvolve_host(hv, ho, N)
            m.deconvolve_host(hv, ho, N)          # second call: replayed batches
            with pytest.raises(binding.MvdError):
                m.set_pipeline_streams(5)
        assert np.array_equal(ho.numpy(), ref), n


@pytest.mark.parametrize("path", PATHS)
def test_reserved_handle_is_capturable_into_a_cuda_graph(path):
    """After mvd_reserve the device-resident call only enqueues (no allocation, no synchronisation): it can be
    captured into a CUDA graph and replayed, with the same bits as the eager call."""
    import torch
    V, N, W, H, K, T = 2, 6, 64, 64, 9, 3
    _need(path, W, H, K)
    pr = synth.make_problem(V, N, W, H, K, T, seed=4242)
    with binding.Mvd(W, H, V, pr.psfs, K, T, pr.eps, path) as m:
        m.reserve(N)
        dv = torch.from_numpy(pr.views.view(np.int16)).cuda()
        eager = torch.empty((N, H, W), dtype=torch.float32, device="cuda")
        st = torch.cuda.Stream()
        m.deconvolve_planes(dv, eager, N, st)
        st.synchronize()
        out = torch.zeros_like(eager)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            m.deconvolve_planes(dv, out, N, st)
        assert not out.any()                    # capture enqueued nothing
        for _ in range(2):
            out.zero_()
            g.replay()
            torch.cuda.synchronize()
            assert torch.equal(out, eager)
        del g


# ---------------------------------------------------------------------------------------------
# Cases the configs lack: asymmetric PSFs (conv vs corr, flip, centre), ragged shapes, aliasing
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("V,N,W,H,K,T,psf", [
    (3, 3, 96, 80, 7, 4, "random"),      # asymmetric, smooth sizes (both engines)
    (2, 5, 160, 80, 13, 3, "random"),    # odd plane count; radix-5 lengths
    (1, 2, 128, 64, 21, 5, "sparse"),    # templated K, single view
    (2, 2, 200, 150, 31, 2, "random"),   # several tiles + ragged tail, 2-chunk PSF rows
    (2, 1, 70, 50, 5, 6, "random"),      # W, H not multiples of anything useful
    (4, 2, 60, 36, 9, 3, "gauss"),
    (2, 2, 37, 23, 5, 3, "random"),      # primes: direct only
    (2, 2, 192, 320, 51, 1, "random"),   # largest templated K, 3-chunk rows
    (2, 3, 160, 96, 41, 2, "random"),    # config 4's PSF size on the direct engine (direct_corr2_kernel<41, 7>)
    (2, 2, 256, 800, 9, 2, "random"),    # config 4's column length (800 = 2^5 5^2)
    (1, 3, 2048, 64, 7, 2, "random"),    # config 4's row length
    (2, 2, 64, 1024, 5, 2, "random"),    # config 5's column length
    (2, 2, 1024, 512, 5, 1, "sparse"),   # config 3's plane
    (2, 2, 32, 2048, 5, 1, "random"),    # longest column transform
    (2, 3, 512, 256, 9, 2, "random"),    # generation-2 kernels, odd plane count (half-empty last pair)
    (1, 2, 256, 2048, 5, 1, "random"),   # generation 2: 2048-point columns (cp.async column kernel)
    (2, 1, 2048, 256, 7, 2, "random"),   # generation 2: 2048-point rows, a single plane
    (3, 5, 256, 256, 11, 2, "sparse"),   # generation 2: 256 x 256, three views
    (2, 2, 1024, 1024, 7, 1, "random"),  # generation 2: config 5's plane with an asymmetric PSF
    (1, 2, 2048, 2048, 5, 1, "random"),  # the largest plane the FFT engine takes
    (2, 3, 64, 32, 1, 3, "random"),      # psf_size 1: a scalar "PSF"
    (2, 3, 384, 640, 7, 2, "random"),    # lengths 2^a 3 and 2^a 5 (generation 1): rows 384, columns 640
    (2, 2, 640, 384, 5, 2, "random"),    # ... and the other way round
    (1, 2, 768, 1280, 5, 1, "random"),
    (2, 2, 1280, 768, 7, 1, "sparse"),
    (1, 2, 1536, 1600, 5, 1, "random"),
    (2, 1, 1600, 1536, 5, 1, "random"),
    (2, 2, 2048, 1280, 5, 1, "random"),  # a generation-2 length next to a generation-1 one: both run generation 1
    (2, 2, 800, 160, 7, 2, "random"),    # 800-point ROWS (generation 1)
    (2, 3, 320, 80, 5, 2, "random"),
    (1, 2, 800, 2048, 5, 1, "random"),   # generation-1 2048-point columns
])
def test_asymmetric_and_ragged(path, V, N, W, H, K, T, psf):
    _need(path, W, H, K)
    pr = synth.make_problem(V, N, W, H, K, T, seed=K * 1000 + W, psf=psf)
    ref = mvd_oracle.deconvolve(pr.views, pr.psfs, T, pr.eps)
    out = _run(pr.views, pr.psfs, T, path)
    assert_parity(out, ref, f"{binding.PATH_NAMES[path]} {V}v {N}x{W}x{H} K{K} {psf}")


@pytest.mark.parametrize("path", PATHS)
def test_psf_larger_than_plane_aliases(path):
    """K > W: taps alias around the plane (oracle pin P5 covers the same case against brute force)."""
    V, N, W, H, K, T = 2, 2, 8, 12, 9, 3
    _need(path, W, H, K)
    rng = np.random.default_rng(5)
    psfs = np.stack([synth.random_psf(K, rng) for _ in range(V)])
    views = synth.random_views(V, N, W, H, seed=3, lo=50, hi=3000)
    ref = mvd_oracle.deconvolve(views, psfs, T)
    assert_parity(_run(views, psfs, T, path), ref, "aliasing")


# ---------------------------------------------------------------------------------------------
# Exact work
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("V", [1, 2, 4, 6])
def test_zero_iterations_is_mean_of_views(path, V):
    """A17 / P11: uint16 ingest is exact; the mean is bit-exact for V in {1,2,4}, 1 ulp for V = 6."""
    W, H, N = 64, 32, 3
    _need(path, W, H, 3)
    views = synth.random_views(V, N, W, H, seed=V, lo=0, hi=65536)
    psfs = np.stack([synth.delta_psf(3)] * V)
    out = _run(views, psfs, 0, path)
    want = (views.astype(np.float64).sum(axis=0) / V)
    if V in (1, 2, 4):
        assert np.array_equal(out, want.astype(np.float32))
    else:
        np.testing.assert_allclose(out, want, rtol=1.2e-7)
    if V == 1:
        assert np.array_equal(out.astype(np.uint16), views[0])   # ingest round-trips every uint16 value


@pytest.mark.parametrize("T", [1, 3])
def test_centred_delta_is_identity_direct(T):
    """P1 on the direct engine: x/x = 1 and x*1 are exact in fp32, so psi == phi bit for bit."""
    W, H, N, K = 64, 48, 2, 5
    views = synth.random_views(1, N, W, H, seed=11, lo=1, hi=60000)
    out = _run(views, synth.delta_psf(K)[None], T, binding.PATH_DIRECT)
    assert np.array_equal(out, views[0].astype(np.float32))


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("dz,dx", [(1, -2), (-2, 1)])
def test_offcentre_delta_shifts_by_plus_d(path, dz, dx):
    """P2 closed form: psi(x) = phi(x + d).  Swapping convolution and correlation gives phi(x - d)."""
    W, H, N, K, T = 64, 32, 2, 5, 2
    _need(path, W, H, K)
    views = synth.random_views(1, N, W, H, seed=21, lo=100, hi=5000)
    out = _run(views, synth.delta_psf(K, dz, dx)[None], T, path)
    want = np.roll(views[0].astype(np.float64), shift=(-dz, -dx), axis=(1, 2))
    np.testing.assert_allclose(out, want, rtol=2e-5)
    assert not np.allclose(out, np.roll(views[0].astype(np.float64), shift=(dz, dx), axis=(1, 2)), rtol=1e-2)


@pytest.mark.parametrize("path", PATHS)
def test_chunking_and_host_pipeline_are_bit_identical(path):
    """P12: planes are independent, so chunk size, batch size and the 3-stream pipeline change nothing."""
    V, N, W, H, K, T = 2, 11, 96, 64, 7, 3
    _need(path, W, H, K)
    pr = synth.make_problem(V, N, W, H, K, T, seed=77)
    base = _run(pr.views, pr.psfs, T, path)
    assert np.array_equal(base, _run(pr.views, pr.psfs, T, path, chunk_planes=4))
    assert np.array_equal(base, _run(pr.views, pr.psfs, T, path, host=True))
    assert np.array_equal(base, _run(pr.views, pr.psfs, T, path, host=True, batch_planes=2, chunk_planes=2))
    assert np.array_equal(base, _run(pr.views, pr.psfs, T, path, host=True, batch_planes=5))


@pytest.mark.parametrize("W,H,N", [(512, 256, 11),      # ping-pong 256-point columns, 512-point rows
                                   (2048, 800, 5),      # config 4: 25 x 32 columns, shuffle-exchange rows
                                   (1024, 1024, 4),     # config 5: TMA-fed OTF slices
                                   (768, 640, 6)])      # three-stage plans with radix-24 / radix-40 first stages
def test_generation2_is_deterministic_and_independent_of_batching(W, H, N):
    """The team-synchronous kernels (private exchange regions, cp.async / TMA landing zones, persistent
    grids) must give the same bits run after run and for every chunk / batch split: a missing team
    barrier or an early landing shows up here as a flipped bit.  compute-sanitizer is not available
    on the GPU pool, so this is the race check."""
    V, K, T = 2, 9, 3
    pr = synth.make_problem(V, N, W, H, K, T, seed=123)
    base = _run(pr.views, pr.psfs, T, binding.PATH_FFT)
    for _ in range(4):
        assert np.array_equal(base, _run(pr.views, pr.psfs, T, binding.PATH_FFT))
    assert np.array_equal(base, _run(pr.views, pr.psfs, T, binding.PATH_FFT, chunk_planes=4))
    assert np.array_equal(base, _run(pr.views, pr.psfs, T, binding.PATH_FFT, chunk_planes=2))
    for streams in (1, 2, 3):          # forked internal streams of the device-resident call
        assert np.array_equal(base, _run(pr.views, pr.psfs, T, binding.PATH_FFT, batch_planes=2, resident_streams=streams))
    assert np.array_equal(base, _run(pr.views, pr.psfs, T, binding.PATH_FFT, host=True))
    assert np.array_equal(base, _run(pr.views, pr.psfs, T, binding.PATH_FFT, host=True, batch_planes=2, chunk_planes=2))
    assert np.array_equal(base, _run(pr.views, pr.psfs, T, binding.PATH_FFT, host=True, batch_planes=6))
    ref = mvd_oracle.deconvolve(pr.views, pr.psfs, T, pr.eps)
    assert_parity(base, ref, f"generation 2, {W}x{H}")


@pytest.mark.parametrize("path", PATHS)
def test_sum_conservation_and_nonnegativity(path):
    """P6 / P4 on the GPU output: sum(psi) = sum(phi_{V-1}) per plane, psi >= 0."""
    cfg = synth.config(2).with_planes(4)
    _need(path, cfg.W, cfg.H, cfg.K)
    psfs, views = synth.config_psfs(2), synth.views(cfg, [3, 4, 5, 6])
    out = _run(views, psfs, 3, path).astype(np.float64)
    assert (out >= 0).all()
    np.testing.assert_allclose(out.sum(axis=(1, 2)), views[-1].astype(np.float64).sum(axis=(1, 2)), rtol=2e-5)


def test_single_plane_and_repeated_calls_on_one_handle():
    import torch
    pr = synth.make_problem(2, 3, 64, 64, 9, 2, seed=5)
    ref = mvd_oracle.deconvolve(pr.views, pr.psfs, 2)
    with binding.Mvd(64, 64, 2, pr.psfs, 9, 2) as m:
        st = torch.cuda.Stream()
        for n in (1, 3, 2, 3):     # scratch grows, shrinks, is reused
            dv = torch.from_numpy(np.ascontiguousarray(pr.views[:, :n]).view(np.int16)).cuda()
            do = torch.empty((n, 64, 64), dtype=torch.float32, device="cuda")
            torch.cuda.synchronize()
            m.deconvolve_planes(dv, do, n, st)
            st.synchronize()
            assert_parity(do.cpu().numpy(), ref[:n], f"n={n}")
        assert m.launch_count() > 0
        m.deconvolve_planes(dv, do, 0, st)       # no-op
        with pytest.raises(binding.MvdError):
            m.deconvolve_planes(None, do, 1, st)


def test_profile_hooks_report_every_launch():
    pr = synth.make_problem(2, 2, 64, 64, 9, 2, seed=6)
    import torch
    with binding.Mvd(64, 64, 2, pr.psfs, 9, 2) as m:
        dv = torch.from_numpy(pr.views.view(np.int16)).cuda()
        do = torch.empty((2, 64, 64), dtype=torch.float32, device="cuda")
        m.profile_enable(True)
        m.launch_count_reset()
        m.deconvolve_planes(dv, do, 2)
        prof = m.profile_read()
        assert sum(n for _, n in prof.values()) == m.launch_count() > 0
        assert all(ms >= 0 for ms, _ in prof.values())


def test_fp32_peak_microbenchmark_is_plausible():
    tf, mhz = binding.measure_fp32_peak()
    assert 20.0 < tf < 120.0 and 500.0 < mhz < 3000.0


def test_config2_full_stack_in_the_bench_launch_configuration():
    """The whole 512-plane stack exactly as bench.py times it (default batches dealt to two streams):
    P12 on every plane (sum(psi) = sum(phi_last)), planes sampled from different batches bit-identical to
    the same plane pair run on its own, and two sampled planes against the oracle."""
    import importlib.util
    import torch
    spec = importlib.util.spec_from_file_location("bench", os.path.join(os.path.dirname(GOLDEN), "..", "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    cfg = synth.config(2)
    psfs, views = bench.make_stack(cfg)
    with binding.Mvd(cfg.W, cfg.H, cfg.V, psfs, cfg.K, cfg.T, cfg.eps) as m:
        dv = torch.from_numpy(views.view(np.int16)).cuda()
        do = torch.empty((cfg.N, cfg.H, cfg.W), dtype=torch.float32, device="cuda")
        m.deconvolve_planes(dv, do, cfg.N)
        torch.cuda.synchronize()
        out = do.cpu().numpy()
        assert np.isfinite(out).all() and (out >= 0).all()
        np.testing.assert_allclose(out.astype(np.float64).sum(axis=(1, 2)),
                                   views[-1].astype(np.float64).sum(axis=(1, 2)), rtol=2e-5)
        for p0 in (0, 30, 32, 254, 300, 510):                       # pairs from different batches / streams
            sub = np.ascontiguousarray(views[:, p0:p0 + 2])
            ds = torch.from_numpy(sub.view(np.int16)).cuda()
            d2 = torch.empty((2, cfg.H, cfg.W), dtype=torch.float32, device="cuda")
            m.deconvolve_planes(ds, d2, 2)
            torch.cuda.synchronize()
            assert np.array_equal(d2.cpu().numpy(), out[p0:p0 + 2]), p0
    sample = [1, 257]
    ref = mvd_oracle.deconvolve(np.ascontiguousarray(views[:, sample]), psfs, cfg.T, cfg.eps)
    assert_parity(out[sample], ref, "config2 full stack, sampled planes")
