"""SURVEY 8(f2) per-view weights and 8(f3) uint16 output on the CUDA path, through the C ABI.

Weights ("weights, float, 4 v bytes/pixel", never defined; READING W1 of DESIGN.md section 2):
a4 becomes psi <- psi . (w_v q + 1 - w_v).  The oracle's arithmetic for that reading is pinned by
tests/test_oracle_pins.py (PW1-PW4); here the kernels are compared with it element by element, and the cases any
reading must satisfy are bit-exact: unit weights = the unweighted run, zero weights = psi_0.

uint16 output: psi rounded to nearest even and saturated at 65535 in the final store.  Integer work, so the bar
is bit-exact: against the engine's own fp32 output rounded on the host, and against the rounded oracle wherever
the oracle is not within the fp32 error of a .5 boundary.
"""
import numpy as np
import pytest

from oracle import mvd_oracle
from paper_1503_07998_b200 import binding, build, synth
from parity_util import assert_parity

pytestmark = pytest.mark.gpu

PATHS = [binding.PATH_DIRECT, binding.PATH_FFT]


@pytest.fixture(scope="module", autouse=True)
def _lib():
    build.build()
    return binding.lib()


def _need(path, W, H, K):
    if not binding.path_supported(path, W, H, K):
        pytest.skip(f"{binding.PATH_NAMES[path]} engine does not take {W}x{H} K={K}")


def _run(views, psfs, T, path, **kw):
    return binding.deconvolve(views, psfs, T, float(synth.EPS), path=path, **kw)


def _weights(shape, seed):
    """Smooth-ish random weights in [0, 1] with exact 0 and exact 1 regions (feathered view borders)."""
    rng = np.random.default_rng([synth.SEED, 5000 + seed])
    w = rng.random(shape).astype(np.float32)
    w[0, :, : shape[2] // 4] = 0.0
    w[-1, :, :, -shape[3] // 4:] = 1.0
    return w


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("V,N,W,H,K,T", [
    (2, 3, 96, 80, 7, 4),       # generation-1 FFT kernels / on-chip direct kernel (4 tiles), odd plane count
    (3, 4, 512, 256, 9, 3),     # generation-2 FFT kernels / tiled direct kernels
    (2, 2, 64, 64, 9, 5),       # config 1's shape
    (2, 2, 2048, 256, 5, 2),    # 2048-point rows (the weighted row kernel's largest landing zone)
    (2, 3, 37, 23, 5, 3),       # primes: direct only
])
def test_weighted_update_matches_the_oracle(path, V, N, W, H, K, T):
    _need(path, W, H, K)
    pr = synth.make_problem(V, N, W, H, K, T, seed=6000 + W)
    w = _weights(pr.views.shape, W)
    ref = mvd_oracle.deconvolve(pr.views, pr.psfs, T, pr.eps, weights=w)
    out = _run(pr.views, pr.psfs, T, path, weights=w)
    assert_parity(out, ref, f"weighted {binding.PATH_NAMES[path]} {W}x{H}")
    assert np.array_equal(out, _run(pr.views, pr.psfs, T, path, weights=w, host=True))     # pipeline: same bits
    plain = mvd_oracle.deconvolve(pr.views, pr.psfs, T, pr.eps)
    assert np.linalg.norm(ref - plain) > 1e-2 * np.linalg.norm(plain)                       # the weights matter


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("W,H", [(96, 80), (512, 256)])
def test_unit_and_zero_weights_are_exact(path, W, H):
    """PW1 / PW2 on the GPU: w = 1 reproduces the unweighted run bit for bit (fma(1, q, 0) = q); w = 0 everywhere
    leaves psi_0, the mean of the views, bit for bit (psi . fma(0, q, 1) = psi)."""
    V, N, K, T = 2, 3, 7, 3
    _need(path, W, H, K)
    pr = synth.make_problem(V, N, W, H, K, T, seed=6100 + W)
    plain = _run(pr.views, pr.psfs, T, path)
    assert np.array_equal(plain, _run(pr.views, pr.psfs, T, path, weights=np.ones(pr.views.shape, np.float32)))
    zero = _run(pr.views, pr.psfs, T, path, weights=np.zeros(pr.views.shape, np.float32))
    assert np.array_equal(zero, (pr.views.astype(np.float64).sum(0) / V).astype(np.float32))


@pytest.mark.parametrize("path", PATHS)
def test_weights_cure_a_view_that_does_not_cover_a_block(path):
    """The partial-overlap case weights exist for: view 0 is zero-filled in a block and carries weight 0 there
    (feathered to 1 over a few pixels), so its update no longer drives psi to 0 and the next view never divides
    by a vanished blur: parity holds on both engines and the FFT engine's guard has nothing to flag."""
    import torch
    V, N, W, H, K, T = 2, 4, 128, 64, 9, 3
    pr = synth.make_problem(V, N, W, H, K, T, seed=6200, psf="gauss")
    views = pr.views.copy()
    views[0, :, 16:48, 40:100] = 0
    w = np.ones(views.shape, np.float32)
    yy, xx = np.mgrid[0:H, 0:W]
    d = np.maximum(np.maximum(16 - yy, yy - 47), np.maximum(40 - xx, xx - 99))      # distance outside the block
    w[0] = np.clip(d / 8.0, 0.0, 1.0).astype(np.float32)[None]
    ref = mvd_oracle.deconvolve(views, pr.psfs, T, pr.eps, weights=w)
    assert ref[:, 20:44, 50:90].min() > 0.5                                            # the block stays alive
    with binding.Mvd(W, H, V, pr.psfs, K, T, pr.eps, path) as m:
        dv = torch.from_numpy(views.view(np.int16)).cuda()
        dw = torch.from_numpy(w).cuda()
        do = torch.empty((N, H, W), dtype=torch.float32, device="cuda")
        m.deconvolve_planes_weighted(dv, dw, do, N)
        torch.cuda.synchronize()
        assert_parity(do.cpu().numpy(), ref, f"feathered missing view {binding.PATH_NAMES[path]}")
        if path == binding.PATH_FFT:
            assert m.guard_flagged() == 0


# ---------------------------------------------------------------------------------------------
# uint16 output
# ---------------------------------------------------------------------------------------------
def _round_u16(a):
    return np.clip(np.rint(np.asarray(a, dtype=np.float64)), 0, 65535).astype(np.uint16)


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("V,N,W,H,K,T", [
    (2, 3, 96, 80, 7, 3),
    (2, 4, 512, 256, 9, 2),
    (2, 2, 64, 64, 9, 4),
    (2, 2, 37, 23, 5, 2),
])
def test_uint16_output_is_the_rounded_result(path, V, N, W, H, K, T):
    _need(path, W, H, K)
    pr = synth.make_problem(V, N, W, H, K, T, seed=6300 + W)
    f32 = _run(pr.views, pr.psfs, T, path)
    u16 = _run(pr.views, pr.psfs, T, path, out_u16=True)
    assert u16.dtype == np.uint16
    assert np.array_equal(u16, _round_u16(f32))                       # exactly the engine's own result, rounded
    assert np.array_equal(u16, _run(pr.views, pr.psfs, T, path, out_u16=True, host=True))
    ref = mvd_oracle.deconvolve(pr.views, pr.psfs, T, pr.eps)
    # against the oracle: identical wherever the oracle is further from a .5 boundary than the engine's error
    # (relative 1e-4 of the value, the parity bar, plus the FFT engine's absolute floor of 1e-6 of the maximum)
    margin = 1e-4 * ref + 2e-6 * ref.max()
    safe = np.abs(ref - np.floor(ref) - 0.5) > margin
    assert safe.mean() > 0.5
    assert np.array_equal(u16[safe], _round_u16(ref)[safe])
    assert np.abs(u16.astype(np.int64) - _round_u16(ref).astype(np.int64)).max() <= 1


@pytest.mark.parametrize("path", PATHS)
def test_uint16_output_saturates_and_handles_zero_iterations(path):
    W, H, N = 64, 32, 2
    _need(path, W, H, 3)
    views = synth.random_views(2, N, W, H, seed=64, lo=0, hi=65536)
    u16 = _run(views, np.stack([synth.delta_psf(3)] * 2), 0, path, out_u16=True)       # T = 0: the mean, rounded
    assert np.array_equal(u16, _round_u16(views.astype(np.float64).sum(0) / 2))
    # deconvolving saturated blobs overshoots 65535: the store clamps
    pr = synth.make_problem(1, N, W, H, 7, 6, seed=6400, psf="gauss", n_blobs=3)
    bright = np.minimum(pr.views.astype(np.int64) * 100, 65535).astype(np.uint16)
    f32 = _run(bright, pr.psfs, 6, path)
    assert f32.max() > 65535.0
    u16 = _run(bright, pr.psfs, 6, path, out_u16=True)
    assert u16.max() == 65535 and np.array_equal(u16, _round_u16(f32))
