"""Seeded random walk over shapes, PSFs, engines and call variants against the oracle (the parity bar of parity_util).

The hand-picked cases of the other files each aim at one thing; this one mixes them (it was a run of this kind that found
the product form + scalar PSF collapse on the FFT engine, now handled by the guard)."""
import numpy as np
import pytest

from oracle import mvd_oracle
from paper_1503_07998_b200 import binding, build, synth
from parity_util import errors

pytestmark = pytest.mark.gpu

WS = [256, 384, 512, 640, 768, 1024, 1280, 1536, 2048, 320, 96, 800]
HS = [256, 384, 512, 640, 768, 800, 1024, 1280, 1536, 2048, 160, 64]
MODES = ["plain", "weights", "u16", "product", "padded", "host", "padded_w"]


@pytest.fixture(scope="module", autouse=True)
def _lib():
    build.build()
    return binding.lib()


@pytest.mark.parametrize("seed", [11, 12, 13])
def test_random_cases_match_the_oracle(seed):
    rng = np.random.default_rng(seed)
    done = 0
    while done < 10:
        W, H = int(rng.choice(WS)), int(rng.choice(HS))
        if W * H > 1024 * 768:
            continue
        small = W * H <= 512 * 512
        V, T, N = int(rng.integers(1, 5)), int(rng.integers(0, 4)), int(rng.integers(1, 6))
        K = int(rng.choice([1, 3, 5, 7, 9] + ([13, 21] if small else [])))
        kind = str(rng.choice(["random", "sparse", "gauss"]))
        pr = synth.make_problem(V, N, W, H, K, T, seed=int(rng.integers(1 << 30)), psf=kind)
        mode = str(rng.choice(MODES))
        path = binding.PATH_FFT if rng.random() < 0.8 else binding.PATH_DIRECT
        if not binding.path_supported(path, W, H, K):
            path = binding.PATH_DIRECT
        wts = rng.random((V, N, H, W)).astype(np.float32) if mode in ("weights", "padded_w") else None
        what = f"seed {seed} case {done}: {W}x{H} V{V} K{K} T{T} N{N} {kind} {mode} {binding.PATH_NAMES[path]}"
        if mode in ("padded", "padded_w"):
            wu, hu = W - int(rng.integers(K, 40)), H - int(rng.integers(K, 40))
            views = np.ascontiguousarray(pr.views[:, :, :hu, :wu])
            w2 = None if wts is None else np.ascontiguousarray(wts[:, :, :hu, :wu])
            ref = mvd_oracle.deconvolve_padded(views, pr.psfs, T, pr.eps, weights=w2)
            out = binding.deconvolve(views, pr.psfs, T, pr.eps, path=path, padded=True, weights=w2)
        elif mode == "product":
            ref = mvd_oracle.deconvolve_product(pr.views, pr.psfs, T, pr.eps)
            out = binding.deconvolve(pr.views, pr.psfs, T, pr.eps, path=path, product=True)
        else:
            ref = mvd_oracle.deconvolve(pr.views, pr.psfs, T, pr.eps, weights=wts)
            out = binding.deconvolve(pr.views, pr.psfs, T, pr.eps, path=path, host=(mode == "host"), out_u16=(mode == "u16"),
                                     batch_planes=int(rng.choice([0, 2])), weights=wts)
        if mode == "u16":
            assert np.abs(out.astype(np.float64) - np.clip(np.rint(ref), 0, 65535)).max() <= 1.0, what
        else:
            l2, _, mx = errors(out, ref)
            assert l2 <= 1e-4 and mx <= 1e-3, f"{what}: rel L2 {l2:.2e}, max rel {mx:.2e}"
        done += 1
