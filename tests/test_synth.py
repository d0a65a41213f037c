"""The seeded input generator: determinism, per-plane addressability, the structure DESIGN.md states."""
import numpy as np
import pytest

from paper_1503_07998_b200 import synth


@pytest.mark.parametrize("cid", [1, 2, 3, 4, 5])
def test_config_psfs(cid):
    cfg = synth.config(cid)
    P = synth.config_psfs(cid)
    assert P.dtype == np.float32 and P.shape == (cfg.V, cfg.K, cfg.K)
    assert (P >= 0).all() and np.isfinite(P).all()
    np.testing.assert_allclose(P.astype(np.float64).sum(axis=(1, 2)), 1.0, atol=2e-7)
    # every config PSF is centro-symmetric -> conv == corr on the configs;
    # this is why the parity suite adds asymmetric-PSF cases
    np.testing.assert_allclose(P, P[:, ::-1, ::-1], atol=1e-9)


def test_config_sizes_match_baseline():
    c = synth.CONFIGS
    assert (c[1].V, c[1].N, c[1].W, c[1].H, c[1].K, c[1].T) == (2, 8, 64, 64, 9, 10)
    assert (c[2].V, c[2].N, c[2].W, c[2].H, c[2].K, c[2].T) == (2, 512, 512, 256, 21, 10)
    assert (c[3].V, c[3].N, c[3].W, c[3].H, c[3].K, c[3].T) == (4, 1024, 1024, 512, 31, 10)
    assert (c[4].V, c[4].N, c[4].W, c[4].H, c[4].K, c[4].T) == (2, 2048, 2048, 800, 41, 10)
    assert (c[5].V, c[5].N, c[5].W, c[5].H, c[5].K, c[5].T) == (6, 256, 1024, 1024, 51, 20)
    assert c[2].units == 512 * 512 * 256 * 2 * 10
    assert c[1].n_blobs == 50 and c[2].n_blobs == 20000


def test_views_deterministic_and_plane_addressable():
    cfg = synth.config(1)
    a = synth.views(cfg)
    b = synth.views(cfg)
    assert a.dtype == np.uint16 and a.shape == (2, 8, 64, 64)
    assert np.array_equal(a, b)
    assert np.array_equal(a[:, 5], synth.views_plane(cfg, 5))
    sub = synth.views(cfg, planes=[6, 2])
    assert np.array_equal(sub[:, 0], a[:, 6]) and np.array_equal(sub[:, 1], a[:, 2])
    # nuclei-like: bright blobs over a background of ~10 counts (config 1 packs 50 blobs into 8 planes)
    assert a.min() <= 12 and np.percentile(a, 10) < 20 and a.max() > 200
    b2 = synth.views(synth.config(2), planes=[100])
    assert 5 < np.median(b2) < 20 and b2.max() > 100      # config 2: sparse


def test_rotated_psf_symmetry_and_angles():
    P = synth.config_psfs(5)
    np.testing.assert_allclose(P[0], P[3], atol=1e-8)     # theta and theta+180 give the same PSF
    assert np.abs(P[0] - P[1]).max() > 1e-4
    # view 0 is the unrotated (sigma_x, sigma_z) = (2, 10) Gaussian: elongated along z
    c = 25
    assert P[0][c + 8, c] > 10 * P[0][c, c + 8]


def test_make_problem_shapes_and_asymmetry():
    pr = synth.make_problem(3, 2, 24, 16, 7, 4, seed=3)
    assert pr.views.shape == (3, 2, 16, 24) and pr.psfs.shape == (3, 7, 7)
    assert np.abs(pr.psfs - pr.psfs[:, ::-1, ::-1]).max() > 1e-3
    np.testing.assert_allclose(pr.psfs.astype(np.float64).sum(axis=(1, 2)), 1.0, atol=2e-7)
    pr2 = synth.make_problem(3, 2, 24, 16, 7, 4, seed=3)
    assert np.array_equal(pr.views, pr2.views)
