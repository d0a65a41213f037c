"""Reslicing folded into the first read (Fig. 1a).  The definition is a
transpose: a view acquired as a z-stack of camera frames [H (z)][N (camera lines)][W] holds plane p, row
z at frames[z][p]; the oracle is fed the transposed stack, the CUDA path reads the frames in place."""
import numpy as np
import pytest
import torch

from oracle import mvd_oracle
from paper_1503_07998_b200 import binding, build, synth
from parity_util import assert_parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _lib():
    build.build()
    return binding.lib()


@pytest.mark.parametrize("path", [binding.PATH_DIRECT, binding.PATH_FFT])
@pytest.mark.parametrize("V,N,W,H,K,T", [(2, 5, 96, 64, 7, 3), (2, 6, 512, 256, 9, 2), (3, 3, 64, 80, 5, 2)])
def test_camera_order_input_equals_the_resliced_stack(path, V, N, W, H, K, T):
    if not binding.path_supported(path, W, H, K):
        pytest.skip("shape not supported by this engine")
    pr = synth.make_problem(V, N, W, H, K, T, seed=31 + N)
    frames = np.ascontiguousarray(pr.views.transpose(0, 2, 1, 3))            # [V][H][N][W]
    ref = mvd_oracle.deconvolve(np.ascontiguousarray(frames.transpose(0, 2, 1, 3)), pr.psfs, T, pr.eps)
    base = binding.deconvolve(pr.views, pr.psfs, T, pr.eps, path=path)
    assert_parity(base, ref, "resliced stack")
    with binding.Mvd(W, H, V, pr.psfs, K, T, pr.eps, path) as m:
        dv = torch.from_numpy(frames.view(np.int16)).cuda()
        do = torch.empty((N, H, W), dtype=torch.float32, device="cuda")
        m.deconvolve_planes_strided(dv, H * N * W, W, N * W, do, N)
        torch.cuda.synchronize()
        assert np.array_equal(do.cpu().numpy(), base)                        # same bits, no reslicing pass
        # a sub-range of camera lines read in place: planes 2 .. N-1 start 2 W elements into every frame
        do2 = torch.empty((N - 2, H, W), dtype=torch.float32, device="cuda")
        m.set_chunk_planes(2)
        m.deconvolve_planes_strided(dv.data_ptr() + 2 * W * 2, H * N * W, W, N * W, do2, N - 2)
        torch.cuda.synchronize()
        assert np.array_equal(do2.cpu().numpy(), base[2:])
        m.set_chunk_planes(0)
        hv = torch.from_numpy(frames.view(np.int16)).pin_memory()
        ho = torch.empty((N, H, W), dtype=torch.float32).pin_memory()
        m.set_batch_planes(2)
        m.deconvolve_host_camera(hv, ho, N)
        assert np.array_equal(ho.numpy(), base)
        m.set_batch_planes(0)
        m.deconvolve_host_camera(hv, ho, N)
        assert np.array_equal(ho.numpy(), base)


def test_strided_call_rejects_bad_strides():
    pr = synth.make_problem(2, 2, 64, 64, 5, 1, seed=2)
    with binding.Mvd(64, 64, 2, pr.psfs, 5, 1, path=binding.PATH_FFT) as m:
        dv = torch.from_numpy(pr.views.view(np.int16)).cuda()
        do = torch.empty((2, 64, 64), dtype=torch.float32, device="cuda")
        with pytest.raises(binding.MvdError):
            m.deconvolve_planes_strided(dv, 2 * 4096, 4096, 32, do, 2)       # row stride < plane_w
        with pytest.raises(binding.MvdError):
            m.deconvolve_planes_strided(dv, 2 * 4096 + 4, 4096, 64, do, 2)   # FFT engine: not 16-byte aligned
