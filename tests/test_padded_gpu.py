"""Padded plans (mvd_create_padded, reading PD1 = zero fill) against oracle.deconvolve_padded.

The oracle pads by hand, runs its periodic iteration and crops (pins PD1-PD3 in test_oracle_pins.py); the library
embeds the planes in the next supported transform size (FFT engine) or in plane + K - 1 (direct engine).
"""
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


def _psfs(V, K, seed):
    rng = np.random.default_rng(seed)
    return np.stack([synth.random_psf(K, rng) for _ in range(V)])


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("W,H,K,V,T,N", [(100, 37, 9, 2, 5, 3), (61, 45, 7, 3, 4, 2), (256, 256, 21, 2, 3, 2), (17, 200, 5, 1, 6, 5)])
def test_padded_matches_oracle(path, W, H, K, V, T, N):
    views = synth.random_views(V, N, W, H, seed=W + H + K, lo=0, hi=3000)
    psfs = _psfs(V, K, K * 7 + V)
    ref = mvd_oracle.deconvolve_padded(views, psfs, T, float(synth.EPS))
    out = binding.deconvolve(views, psfs, T, float(synth.EPS), path=path, padded=True)
    assert out.shape == (N, H, W)
    assert_parity(out, ref, f"padded {W}x{H} K={K} {binding.PATH_NAMES[path]}")


def test_padded_camera_sized_plane_runs_on_the_fft_engine():
    """2000 x 700 planes (no supported transform length) with a 21 x 21 PSF: padded to 2048 x 768 / 800 inside the library."""
    W, H, K, V, T, N = 2000, 700, 21, 2, 3, 2
    psfs = np.stack([synth.gaussian_psf64(K, 1.5, 5.0), synth.gaussian_psf64(K, 5.0, 1.5)]).astype(np.float32)
    views = synth.random_views(V, N, W, H, seed=2000, lo=0, hi=2000)
    views[:, :, :40, :] = 0            # a dark band and a bright edge: the boundaries differ there
    views[:, :, -3:, :] += 3000
    with binding.Mvd(W, H, V, psfs, K, T, float(synth.EPS), None, None, True) as m:
        ew, eh = m.engine_plane()         # the cheapest supported pair of lengths >= plane + K - 1 (2048 x 768 at present)
        assert m.path == binding.PATH_FFT and ew >= W + K - 1 and eh >= H + K - 1 and (ew, eh) in ((2048, 768), (2048, 800))
    ref = mvd_oracle.deconvolve_padded(views, psfs, T, float(synth.EPS))
    out = binding.deconvolve(views, psfs, T, float(synth.EPS), padded=True)
    assert_parity(out, ref, "padded 2000x700")
    per = binding.deconvolve(views, psfs, T, float(synth.EPS), path=binding.PATH_DIRECT)     # periodic reading: differs
    assert np.abs(per - ref).max() > 1e-2 * ref.max()


@pytest.mark.parametrize("path", PATHS)
def test_padded_host_pipeline_chunks_and_u16_are_consistent(path):
    W, H, K, V, T, N = 120, 50, 9, 2, 4, 11
    views = synth.random_views(V, N, W, H, seed=5, lo=0, hi=900)
    psfs = _psfs(V, K, 3)
    a = binding.deconvolve(views, psfs, T, float(synth.EPS), path=path, padded=True)
    b = binding.deconvolve(views, psfs, T, float(synth.EPS), path=path, padded=True, host=True, batch_planes=4)
    c = binding.deconvolve(views, psfs, T, float(synth.EPS), path=path, padded=True, chunk_planes=2, resident_streams=1)
    assert np.array_equal(a, b) and np.array_equal(a, c)
    u = binding.deconvolve(views, psfs, T, float(synth.EPS), path=path, padded=True, out_u16=True)
    exp = np.clip(np.rint(a.astype(np.float64)), 0, 65535)
    near_tie = np.abs(a - np.floor(a) - 0.5) < 1e-3
    assert np.array_equal(u[~near_tie], exp[~near_tie].astype(np.uint16))


@pytest.mark.parametrize("path", PATHS)
def test_padded_with_weights(path):
    """Per-view weights on a padded plan, device-resident and through the host pipeline (several batches)."""
    W, H, K, V, T, N = 100, 60, 9, 2, 4, 7
    views = synth.random_views(V, N, W, H, seed=31, lo=0, hi=2500)
    psfs = _psfs(V, K, 13)
    wts = np.random.default_rng(8).random((V, N, H, W)).astype(np.float32)
    wts[0, :, :20] = 0.0                                  # view 0 does not cover the top of the planes
    ref = mvd_oracle.deconvolve_padded(views, psfs, T, float(synth.EPS), weights=wts)
    out = binding.deconvolve(views, psfs, T, float(synth.EPS), path=path, padded=True, weights=wts)
    assert_parity(out, ref, f"padded, weighted {binding.PATH_NAMES[path]}")
    again = binding.deconvolve(views, psfs, T, float(synth.EPS), path=path, padded=True, weights=wts, host=True, batch_planes=2)
    assert np.array_equal(out, again)


def test_padded_rejects_camera_order():
    import torch
    W, H, K, V, N = 64, 40, 5, 2, 2
    psfs = _psfs(V, K, 1)
    views = torch.from_numpy(synth.random_views(V, N, W, H, seed=1).view(np.int16)).cuda()
    out = torch.empty((N, H, W), dtype=torch.float32, device="cuda")
    with binding.Mvd(W, H, V, psfs, K, 2, 1e-6, None, None, True) as m:
        with pytest.raises(binding.MvdError) as e:
            m.deconvolve_host_ex(views.cpu(), out.cpu(), N, camera_order=True)
        assert e.value.code == binding.MVD_ERR_UNSUPPORTED
