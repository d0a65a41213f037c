"""Step a2's guard r = phi / max(b, eps) and zero-valued data on the CUDA path (reading A6).

The configs' background of 10 keeps b far above eps, so none of their planes ever reaches the clamp.
These cases do: zero blocks in every view, a view that is zero where the others are not (the estimate
collapses to 0 there and the NEXT view divides its photons by eps), and single pixels with phi > 0 and
b < eps -- on both engines, T >= 3, against the fp64 oracle (whose own guard is pinned by
tests/test_oracle_pins.py::test_eps_guard_value and P1-with-zeros).
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


def _run(views, psfs, T, path, **kw):
    return binding.deconvolve(views, psfs, T, float(synth.EPS), path=path, **kw)


def _name(path):
    return binding.PATH_NAMES[path]


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("T", [1, 3])
def test_centred_delta_with_zero_pixels(path, T):
    """P1 with zeros: 0 / max(0, eps) = 0 and psi stays phi.  Bit-exact on the direct engine; the FFT engine
    returns exact zeros where phi == 0 (0 . q) and phi elsewhere up to its transform round-off, which is relative
    to the plane's MAXIMUM (fp32 FFT: ~1e-7 x 65535 on every pixel), not to the pixel."""
    W, H, N = 64, 32, 3
    views = synth.random_views(1, N, W, H, seed=41, lo=0, hi=65536)
    views[0, 0, :7, :9] = 0
    views[0, 1, 10:20, 30:64] = 0
    views[0, 2, 4, 5] = 65535
    out = _run(views, synth.delta_psf(5)[None], T, path)
    want = views[0].astype(np.float64)
    assert np.isfinite(out).all()
    if path == binding.PATH_DIRECT:
        assert np.array_equal(out, want.astype(np.float32))
    else:
        assert (out[want == 0] == 0).all()
        np.testing.assert_allclose(out, want, rtol=2e-5, atol=4e-7 * 65535)


@pytest.mark.parametrize("path", PATHS)
def test_photons_where_the_estimate_is_zero_stay_dark(path):
    """tests/test_oracle_pins.py::test_eps_guard_value on the GPU: view 0 is empty, so its update sets psi = 0
    everywhere; view 1 then has phi > 0 with b = 0 < eps, r = phi / eps ~ 1e9..1e10, and psi . q stays 0."""
    W, H, N, K = 64, 32, 2, 7
    views = np.zeros((2, N, H, W), dtype=np.uint16)
    views[1] = synth.random_views(1, N, W, H, seed=42, lo=1, hi=9000)[0]
    views[1, 0, 3, 5] = 65535
    rng = np.random.default_rng(7)
    psfs = np.stack([synth.random_psf(K, rng), synth.random_psf(K, rng)])
    for T in (1, 3):
        ref = mvd_oracle.deconvolve(views, psfs, T, float(synth.EPS))
        assert not ref.any()
        out = _run(views, psfs, T, path)
        assert np.isfinite(out).all() and not out.any(), (_name(path), T, float(np.abs(out).max()))


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("psf", ["random", "gauss"])
def test_zero_background_blocks_in_every_view(path, psf):
    """A phantom on a background of 0: most of every view is exactly zero (no photons), b falls below eps away
    from the blobs, and r = 0 / eps = 0 there."""
    V, N, W, H, K, T = 2, 3, 128, 64, 9, 4
    pr = synth.make_problem(V, N, W, H, K, T, seed=4300 + (psf == "gauss"), psf=psf, n_blobs=6, background=0.0)
    assert (pr.views == 0).mean() > 0.5
    ref = mvd_oracle.deconvolve(pr.views, pr.psfs, T, pr.eps)
    out = _run(pr.views, pr.psfs, T, path)
    assert_parity(out, ref, f"zero background {psf} {_name(path)}")


def _missing_view_problem():
    V, N, W, H, K, T = 2, 6, 128, 64, 9, 3
    pr = synth.make_problem(V, N, W, H, K, T, seed=4400, psf="gauss")
    views = pr.views.copy()
    views[0, 1:3, 16:48, 40:100] = 0          # planes 1 and 2: pairs (0, 1) and (2, 3) are hit, pair (4, 5) is not
    return views, pr.psfs, T, pr.eps


@pytest.mark.parametrize("path", PATHS)
def test_view_that_is_zero_where_the_others_are_not(path):
    """View 0 is zero-filled in a block (a registered view that does not cover it) where view 1 has signal:
    view 0's update drives psi to 0 inside the block, view 1 then finds phi > 0 with b < eps at the pixels the
    PSF cannot reach from outside.  The direct engine keeps this local, like the oracle.  On the FFT engine the
    ratio plane would hold values of phi / eps ~ 1e9 whose fp32 transform round-off (~1e2) reaches every pixel of
    the plane PAIR (measured without the guard: output ~1e20): the engine flags such pairs and recomputes them
    with the direct engine's arithmetic."""
    views, psfs, T, eps = _missing_view_problem()
    ref = mvd_oracle.deconvolve(views, psfs, T, eps)
    out = _run(views, psfs, T, path)
    assert_parity(out, ref, f"missing view block {_name(path)}")


def test_fft_guard_hands_over_exactly_the_ill_conditioned_pairs():
    """The guard flags pairs (0, 1) and (2, 3) of the case above and leaves pair (4, 5) to the FFT engine; the
    handed-over planes carry the direct engine's bits; ordinary stacks (config 2's planes) flag nothing."""
    import torch
    views, psfs, T, eps = _missing_view_problem()
    V, N, H, W = views.shape
    direct = _run(views, psfs, T, binding.PATH_DIRECT)
    with binding.Mvd(W, H, V, psfs, psfs.shape[-1], T, eps, binding.PATH_FFT) as m:
        dv = torch.from_numpy(views.view(np.int16)).cuda()
        do = torch.empty((N, H, W), dtype=torch.float32, device="cuda")
        m.deconvolve_planes(dv, do, N)
        assert m.guard_flagged() == 2
        out = do.cpu().numpy()
        assert np.array_equal(out[:4], direct[:4])
        assert not np.array_equal(out[4:], direct[4:])           # the untouched pair is the FFT engine's result
        m.deconvolve_planes(dv, do, N)                           # the counter accumulates over calls
        assert m.guard_flagged() == 4
        assert np.array_equal(do.cpu().numpy(), out)
    cfg = synth.config(2)
    cpsfs, cviews = synth.config_psfs(2), synth.views(cfg, [0, 1, 300, 301])
    with binding.Mvd(cfg.W, cfg.H, cfg.V, cpsfs, cfg.K, cfg.T, cfg.eps, binding.PATH_FFT) as m:
        dv = torch.from_numpy(cviews.view(np.int16)).cuda()
        do = torch.empty((4, cfg.H, cfg.W), dtype=torch.float32, device="cuda")
        m.deconvolve_planes(dv, do, 4)
        assert m.guard_flagged() == 0


@pytest.mark.parametrize("path", PATHS)
def test_single_hot_pixel_in_an_empty_plane(path):
    """One plane with a single non-zero pixel per view (everything else exactly 0), asymmetric PSFs."""
    V, N, W, H, K, T = 2, 2, 64, 32, 5, 3
    views = np.zeros((V, N, H, W), dtype=np.uint16)
    views[0, 0, 10, 20] = 900
    views[1, 0, 10, 21] = 700
    views[:, 1] = synth.random_views(V, 1, W, H, seed=45, lo=50, hi=500)[:, 0]   # its pair partner is ordinary
    rng = np.random.default_rng(8)
    psfs = np.stack([synth.random_psf(K, rng) for _ in range(V)])
    ref = mvd_oracle.deconvolve(views, psfs, T, float(synth.EPS))
    out = _run(views, psfs, T, path)
    assert np.isfinite(out).all()
    assert_parity(out[1:], ref[1:], f"ordinary partner plane {_name(path)}")
    # the hot-pixel plane: compare where the oracle is not negligible, absolute elsewhere
    scale = ref[0].max()
    assert scale > 0
    np.testing.assert_allclose(out[0], ref[0], rtol=1e-3, atol=1e-4 * scale)
