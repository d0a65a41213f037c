"""The update as printed in PAPER.md:79 (simultaneous / product form; mvd_set_update_mode) against
oracle.deconvolve_product (pins PP1-PP3 in test_oracle_pins.py), on both engines."""
import numpy as np
import pytest

from oracle import mvd_oracle
from paper_1503_07998_b200 import binding, build, synth
from parity_util import assert_parity

pytestmark = pytest.mark.gpu
PATHS = [binding.PATH_FFT, binding.PATH_DIRECT]


@pytest.fixture(scope="module", autouse=True)
def _lib():
    build.build()
    return binding.lib()


def _need(path, W, H, K):
    if not binding.path_supported(path, W, H, K):
        pytest.skip(f"{binding.PATH_NAMES[path]} engine does not take {W}x{H} K={K}")


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("V,N,W,H,K,T,psf", [
    (3, 3, 96, 80, 7, 4, "random"),      # generation-1 FFT kernels, odd plane count, asymmetric PSFs
    (2, 4, 512, 256, 9, 3, "random"),    # generation-2 FFT kernels
    (1, 2, 64, 64, 5, 5, "random"),      # one view: the two forms coincide
    (2, 2, 2048, 800, 5, 2, "gauss"),    # config 4's shape (25 x 32 columns, shuffle rows); separable PSFs on the direct engine
    (4, 2, 200, 150, 11, 2, "sparse"),   # direct engine only (no transform lengths)
])
def test_product_form_matches_oracle(path, V, N, W, H, K, T, psf):
    _need(path, W, H, K)
    pr = synth.make_problem(V, N, W, H, K, T, seed=K * 100 + W, psf=psf)
    ref = mvd_oracle.deconvolve_product(pr.views, pr.psfs, T, pr.eps)
    out = binding.deconvolve(pr.views, pr.psfs, T, pr.eps, path=path, product=True)
    assert_parity(out, ref, f"product form {binding.PATH_NAMES[path]} {V}v {W}x{H}")
    if V > 1:
        seq = binding.deconvolve(pr.views, pr.psfs, T, pr.eps, path=path)
        assert np.abs(seq - out).max() > 1e-4 * np.abs(out).max()          # really a different update


@pytest.mark.parametrize("path", PATHS)
def test_product_form_config1(path):
    cfg = synth.config(1)
    psfs, views = synth.config_psfs(1), synth.views(cfg)
    ref = mvd_oracle.deconvolve_product(views, psfs, cfg.T, cfg.eps)
    out = binding.deconvolve(views, psfs, cfg.T, cfg.eps, path=path, product=True)
    assert_parity(out, ref, f"product form config 1 {binding.PATH_NAMES[path]}")


@pytest.mark.parametrize("path", PATHS)
def test_product_form_weights_pipeline_chunks_u16(path):
    V, N, W, H, K, T = 2, 7, 256, 256, 7, 3
    pr = synth.make_problem(V, N, W, H, K, T, seed=9, psf="random")
    wts = np.random.default_rng(4).random((V, N, H, W)).astype(np.float32)
    ref = mvd_oracle.deconvolve_product(pr.views, pr.psfs, T, pr.eps, weights=wts)
    out = binding.deconvolve(pr.views, pr.psfs, T, pr.eps, path=path, product=True, weights=wts)
    assert_parity(out, ref, "product form, weighted")
    a = binding.deconvolve(pr.views, pr.psfs, T, pr.eps, path=path, product=True)
    b = binding.deconvolve(pr.views, pr.psfs, T, pr.eps, path=path, product=True, host=True, batch_planes=2)
    c = binding.deconvolve(pr.views, pr.psfs, T, pr.eps, path=path, product=True, chunk_planes=4, resident_streams=1)
    assert np.array_equal(a, b) and np.array_equal(a, c)
    u = binding.deconvolve(pr.views, pr.psfs, T, pr.eps, path=path, product=True, out_u16=True)
    near_tie = np.abs(a - np.floor(a) - 0.5) < 1e-3
    assert np.array_equal(u[~near_tie], np.clip(np.rint(a.astype(np.float64)), 0, 65535)[~near_tie].astype(np.uint16))


def test_product_form_guard_repairs_collapsed_estimates():
    """A scalar 'PSF' (K = 1) in the product form: psi^{t+1} = phi_0 phi_1 / psi^t drives the estimate towards zero where one
    view is dark, the blur falls below the transforms' round-off and a2 divides noise.  The FFT engine flags those plane
    pairs and hands them to the direct engine's arithmetic -- in the product form too."""
    import torch
    V, N, W, H, K, T = 2, 5, 512, 512, 1, 2
    pr = synth.make_problem(V, N, W, H, K, T, seed=228, psf="sparse")
    ref = mvd_oracle.deconvolve_product(pr.views, pr.psfs, T, pr.eps)
    with binding.Mvd(W, H, V, pr.psfs, K, T, pr.eps, binding.PATH_FFT) as m:
        m.set_update_mode(binding.UPDATE_PRODUCT)
        dv = torch.from_numpy(pr.views.view(np.int16)).cuda()
        do = torch.empty((N, H, W), dtype=torch.float32, device="cuda")
        m.deconvolve_planes(dv, do, N)
        torch.cuda.synchronize()
        flagged = m.guard_flagged()
        out = do.cpu().numpy()
    direct = binding.deconvolve(pr.views, pr.psfs, T, pr.eps, path=binding.PATH_DIRECT, product=True)
    assert_parity(direct, ref, "product form, K = 1, direct engine")
    assert_parity(out, ref, f"product form, K = 1, FFT engine ({flagged} pairs repaired)")
