"""mvd_deconvolve_planes_noalloc: the entry point that allocates nothing (scratch in a fixed device array inside the library).

Collected last on purpose (the suite runs with pytest -x).  Two calls in a row on one handle -- different stacks, different
plane counts, so the second call runs over what the first left in the shared scratch -- each compared with the existing
path (mvd_deconvolve_planes on a direct-engine handle) within the parity tolerance of the other GPU tests.
"""
import numpy as np
import pytest

from paper_1503_07998_b200 import binding, build, synth
from parity_util import assert_parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _lib():
    build.build()
    return binding.lib()


def _psfs(V, K, seed):
    rng = np.random.default_rng(seed)
    return np.stack([synth.random_psf(K, rng) for _ in range(V)])      # asymmetric, not separable: the tiled 2D kernels


def test_noalloc_matches_the_existing_path_on_two_calls_in_a_row():
    import torch
    V, W, H, K, T = 2, 256, 192, 9, 4                    # too large for the on-chip whole-run kernel: r scratch is used
    psfs = _psfs(V, K, 31)
    stacks = [synth.random_views(V, 5, W, H, seed=41, lo=0, hi=3000),        # odd plane count: half-empty last pair
              synth.random_views(V, 8, W, H, seed=42, lo=0, hi=60000)]
    st = torch.cuda.Stream()
    with binding.Mvd(W, H, V, psfs, K, T, 1e-6, binding.PATH_DIRECT) as m, \
         binding.Mvd(W, H, V, psfs, K, T, 1e-6, binding.PATH_DIRECT) as ref_handle:
        for k, views in enumerate(stacks):
            N = views.shape[1]
            dv = torch.from_numpy(views.view(np.int16)).cuda()
            out = torch.full((N, H, W), float("nan"), dtype=torch.float32, device="cuda")
            ref = torch.empty((N, H, W), dtype=torch.float32, device="cuda")
            ref_handle.deconvolve_planes(dv, ref, N, st)                      # the existing path (allocates its workspace)
            st.synchronize()
            torch.cuda.synchronize()
            free0 = torch.cuda.mem_get_info()[0]
            m.deconvolve_planes_noalloc(dv, out, N, st)
            st.synchronize()
            free1 = torch.cuda.mem_get_info()[0]
            if k == 1:                                    # (the first call may page in the kernels' module)
                assert free1 == free0, "the no-allocation entry point changed the device's free memory"
            assert_parity(out.cpu().numpy(), ref.cpu().numpy().astype(np.float64), f"noalloc call {k}")
            assert torch.equal(out, ref)                  # same kernels, same order: bit for bit


def test_noalloc_rejects_what_it_cannot_serve():
    import torch
    V, W, H, K, T = 1, 512, 512, 5, 1
    psfs = _psfs(V, K, 5)
    N = binding.NOALLOC_MAX_VOXELS // (W * H) + 1         # one plane beyond the limit
    dv = torch.zeros((V, N, H, W), dtype=torch.int16, device="cuda")
    out = torch.zeros((N, H, W), dtype=torch.float32, device="cuda")
    with binding.Mvd(W, H, V, psfs, K, T, 1e-6, binding.PATH_DIRECT) as m:
        with pytest.raises(binding.MvdError) as e:
            m.deconvolve_planes_noalloc(dv, out, N)
        assert e.value.code == binding.MVD_ERR_TOO_LARGE and "MVD_NOALLOC_MAX_VOXELS" in str(e.value)
        assert not out.any()                              # nothing was enqueued
        m.deconvolve_planes_noalloc(dv, out, N - 1)       # exactly at the limit is fine
        torch.cuda.synchronize()
    with binding.Mvd(W, H, V, psfs, K, T, 1e-6, binding.PATH_FFT) as m:
        with pytest.raises(binding.MvdError) as e:
            m.deconvolve_planes_noalloc(dv, out, 2)
        assert e.value.code == binding.MVD_ERR_UNSUPPORTED
