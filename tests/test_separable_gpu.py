"""Separable fast path of the direct engine (csrc/mvd_sep.cu): PSFs that are outer products run a1 / a3 as an x pass and
a z pass (2 K FMAs per output instead of K^2).  Same oracle, same tolerance; the kernel classes reported by the library
prove which kernels ran."""
import numpy as np
import pytest

from oracle import mvd_oracle
from paper_1503_07998_b200 import binding, build, synth
from parity_util import assert_parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _lib():
    build.build()
    return binding.lib()


def _outer_psfs(V, K, seed):
    """Asymmetric separable PSFs: P_v = u_v w_v^T with random positive, non-symmetric factors."""
    rng = np.random.default_rng(seed)
    out = []
    for _ in range(V):
        u, w = rng.random(K) + 0.05, rng.random(K) + 0.05
        P = np.outer(u, w)
        out.append(P / P.sum())
    return np.stack(out).astype(np.float32)


def _classes_run(views, psfs, T, **kw):
    import torch
    V, N, H, W = views.shape
    with binding.Mvd(W, H, V, psfs, psfs.shape[-1], T, 1e-6, binding.PATH_DIRECT) as m:
        m.profile_enable(True)
        dv = torch.from_numpy(views.view(np.int16)).cuda()
        do = torch.empty((N, H, W), dtype=torch.float32, device="cuda")
        m.deconvolve_planes(dv, do, N)
        prof = m.profile_read()
        return {k for k, (ms, n) in prof.items() if n}, do.cpu().numpy()


@pytest.mark.parametrize("V,N,W,H,K,T", [
    (2, 3, 96, 200, 9, 3),       # templated K, odd plane count, several tiles in z
    (2, 2, 512, 256, 21, 2),     # config 2's shape and PSF size
    (1, 2, 200, 150, 41, 2),     # config 4's PSF size
    (3, 2, 400, 300, 13, 3),     # runtime K (chunks of 8 taps)
    (2, 2, 301, 260, 27, 2),     # W not a multiple of 4: scalar staging
    (2, 2, 61, 45, 27, 2),       # planes that fit on chip keep the whole-run kernel (2D taps)
    (2, 1, 37, 300, 5, 4),       # a single plane (half-empty pair), K > nothing special
    (2, 2, 24, 20, 31, 2),       # K > W and K > H: taps alias around the plane
])
def test_separable_psfs_match_oracle(V, N, W, H, K, T):
    psfs = _outer_psfs(V, K, seed=K + W)
    views = synth.random_views(V, N, W, H, seed=W * 3 + K, lo=0, hi=3000)
    ref = mvd_oracle.deconvolve(views, psfs, T, 1e-6)
    classes, out = _classes_run(views, psfs, T)
    if W * H * 16 > 227 * 1024:      # larger than the on-chip whole-run kernel takes: the separable kernels must have run
        assert "sep_blur_ratio" in classes and "sep_backproject_update" in classes and "direct_blur_ratio" not in classes
    assert_parity(out, ref, f"separable {W}x{H} K={K}")


def test_non_separable_psfs_keep_the_2d_kernels():
    V, N, W, H, K, T = 2, 2, 96, 64, 9, 2
    rng = np.random.default_rng(1)
    psfs = np.stack([synth.random_psf(K, rng) for _ in range(V)])
    views = synth.random_views(V, N, W, H, seed=7)
    classes, out = _classes_run(views, psfs, T)
    assert "sep_blur_ratio" not in classes and ("direct_blur_ratio" in classes or "small_resident" in classes)
    assert_parity(out, mvd_oracle.deconvolve(views, psfs, T, 1e-6), "2D kernels")


def test_separable_with_weights_u16_and_host_pipeline():
    V, N, W, H, K, T = 2, 5, 256, 300, 21, 3
    psfs = _outer_psfs(V, K, seed=5)
    views = synth.random_views(V, N, W, H, seed=11, lo=0, hi=2000)
    wts = np.random.default_rng(2).random((V, N, H, W)).astype(np.float32)
    ref = mvd_oracle.deconvolve(views, psfs, T, 1e-6, weights=wts)
    out = binding.deconvolve(views, psfs, T, 1e-6, path=binding.PATH_DIRECT, weights=wts)
    assert_parity(out, ref, "separable, weighted")
    a = binding.deconvolve(views, psfs, T, 1e-6, path=binding.PATH_DIRECT)
    b = binding.deconvolve(views, psfs, T, 1e-6, path=binding.PATH_DIRECT, host=True, batch_planes=2)
    assert np.array_equal(a, b)
    u = binding.deconvolve(views, psfs, T, 1e-6, path=binding.PATH_DIRECT, out_u16=True)
    near_tie = np.abs(a - np.floor(a) - 0.5) < 1e-3
    assert np.array_equal(u[~near_tie], np.clip(np.rint(a.astype(np.float64)), 0, 65535)[~near_tie].astype(np.uint16))
