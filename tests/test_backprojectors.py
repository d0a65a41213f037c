"""The other back-projectors of Supp. Note 2 s.1: host-side builder against the
oracle's numpy builder (CPU), and the CUDA path with explicit X_v against the oracle (GPU)."""
import ctypes

import numpy as np
import pytest

from oracle import mvd_oracle
from paper_1503_07998_b200 import binding, build, synth
from parity_util import assert_parity

VARIANTS = [(binding.BP_INDEPENDENT, "independent"), (binding.BP_EFFICIENT_BAYESIAN, "efficient_bayesian"),
            (binding.BP_OPTIMIZATION1, "optimization1")]


@pytest.fixture(scope="module", autouse=True)
def _lib():
    build.build()
    return binding.lib()


def _psfs(V, K, seed):
    rng = np.random.default_rng(seed)
    return np.stack([synth.random_psf(K, rng) for _ in range(V)])


@pytest.mark.parametrize("variant,name", VARIANTS)
@pytest.mark.parametrize("V,K", [(1, 5), (2, 3), (3, 7), (4, 9)])
def test_builder_matches_the_oracle_builder(variant, name, V, K):
    psfs = _psfs(V, K, 10 * V + K)
    got = binding.build_backprojectors(variant, psfs)
    want = mvd_oracle.backprojectors(psfs, name)
    np.testing.assert_allclose(got, want, rtol=2e-6, atol=1e-12)
    if variant != binding.BP_INDEPENDENT:
        np.testing.assert_allclose(got.sum(axis=(1, 2)), 1.0, rtol=1e-6)


def test_builder_on_config_psfs_and_bad_arguments():
    psfs = synth.config_psfs(1)
    for variant, name in VARIANTS:
        np.testing.assert_allclose(binding.build_backprojectors(variant, psfs),
                                   mvd_oracle.backprojectors(psfs, name), rtol=2e-6, atol=1e-14)
    with pytest.raises(binding.MvdError):
        binding.build_backprojectors(3, psfs)                       # Optimization II is not offered
    bad = psfs.copy()
    bad[0, 0, 0] = np.nan
    with pytest.raises(binding.MvdError):
        binding.build_backprojectors(1, bad)


def test_create_backprojectors_validates_before_touching_the_device():
    lib = binding.lib()
    h = ctypes.c_void_p()
    P = np.ascontiguousarray(_psfs(2, 5, 1))
    X = np.ascontiguousarray(_psfs(2, 7, 2))
    fp = ctypes.POINTER(ctypes.c_float)
    call = lambda xs, kx: lib.mvd_create_backprojectors(64, 64, 2, P.ctypes.data_as(fp), 5, xs, kx, 3, 1e-6, 0,
                                                        ctypes.byref(h))
    assert call(None, 7) == binding.MVD_ERR_INVALID
    assert call(X.ctypes.data_as(fp), 6) == binding.MVD_ERR_INVALID       # even size
    Xn = X.copy()
    Xn[1, 2, 2] = np.inf
    assert call(Xn.ctypes.data_as(fp), 7) == binding.MVD_ERR_INVALID
    assert not h.value


# ---------------------------------------------------------------------------------------------
# GPU
# ---------------------------------------------------------------------------------------------
PATHS = [binding.PATH_DIRECT, binding.PATH_FFT]


@pytest.mark.gpu
@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("V,N,W,H,K,KX,T", [
    (2, 3, 96, 80, 5, 9, 3),       # X larger than P, generation-1 FFT lengths
    (3, 2, 512, 256, 9, 5, 2),     # X smaller than P, generation-2 kernels
    (2, 2, 64, 64, 7, 7, 4),
    (1, 2, 70, 50, 3, 5, 3),       # direct only
])
def test_explicit_asymmetric_backprojectors_match_the_oracle(path, V, N, W, H, K, KX, T):
    if not binding.path_supported(path, W, H, max(K, KX)):
        pytest.skip("shape not supported by this engine")
    pr = synth.make_problem(V, N, W, H, K, T, seed=K * 100 + KX)
    xs = _psfs(V, KX, 500 + KX)                      # random, asymmetric, sum 1
    ref = mvd_oracle.deconvolve(pr.views, pr.psfs, T, pr.eps, backprojectors=xs)
    out = binding.deconvolve(pr.views, pr.psfs, T, pr.eps, path=path, backprojectors=xs)
    assert_parity(out, ref, f"explicit X {binding.PATH_NAMES[path]} {W}x{H} K{K} KX{KX}")
    # a flipped X must NOT pass: the pin has teeth on the GPU side too
    wrong = mvd_oracle.deconvolve(pr.views, pr.psfs, T, pr.eps, backprojectors=xs[:, ::-1, ::-1])
    assert np.abs(wrong - ref).max() > 1e-2 * ref.max()


@pytest.mark.gpu
@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("variant,name", VARIANTS)
def test_paper_variants_on_config1(path, variant, name):
    cfg = synth.config(1)
    if not binding.path_supported(path, cfg.W, cfg.H, cfg.K):
        pytest.skip("shape not supported by this engine")
    psfs, views = synth.config_psfs(1), synth.views(cfg)
    xs = binding.build_backprojectors(variant, psfs)
    ref = mvd_oracle.deconvolve(views, psfs, cfg.T, cfg.eps, backprojectors=mvd_oracle.backprojectors(psfs, name))
    out = binding.deconvolve(views, psfs, cfg.T, cfg.eps, path=path, backprojectors=xs)
    assert_parity(out, ref, f"{name} {binding.PATH_NAMES[path]}")
    if variant == binding.BP_INDEPENDENT:            # the same numbers as mvd_create's built-in X = P_v^*
        base = binding.deconvolve(views, psfs, cfg.T, cfg.eps, path=path)
        np.testing.assert_allclose(out, base, rtol=2e-4, atol=1e-3)


@pytest.mark.gpu
def test_efficient_bayesian_on_config2_planes_with_the_host_pipeline():
    cfg = synth.config(2)
    planes = [0, 1, 300]
    psfs, views = synth.config_psfs(2), synth.views(cfg, planes)
    xs = binding.build_backprojectors(binding.BP_EFFICIENT_BAYESIAN, psfs)
    T = 4
    ref = mvd_oracle.deconvolve(views, psfs, T, cfg.eps, backprojectors=xs)
    out = binding.deconvolve(views, psfs, T, cfg.eps, backprojectors=xs)
    assert_parity(out, ref, "efficient bayesian config2")
    assert np.array_equal(out, binding.deconvolve(views, psfs, T, cfg.eps, backprojectors=xs, host=True, batch_planes=2))
