"""mvd_deconvolve_files: disk I/O as the outer pipeline stage (Algorithm 1)."""
import os

import numpy as np
import pytest

from paper_1503_07998_b200 import binding, build, synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _lib():
    build.build()
    return binding.lib()


@pytest.mark.parametrize("path", [binding.PATH_FFT, binding.PATH_DIRECT])
@pytest.mark.parametrize("N,u16", [(37, False), (64, True)])
def test_files_give_the_bytes_of_the_host_call(tmp_path, path, N, u16):
    """Several slabs (N / 4 planes each), an odd stack, both output types: the file holds exactly what
    mvd_deconvolve_host returns for the same stack."""
    V, W, H, K, T = 2, 128, 96, 7, 3
    pr = synth.make_problem(V, N, W, H, K, T, seed=N, psf="random")
    ref = binding.deconvolve(pr.views, pr.psfs, T, pr.eps, path=path, host=True, out_u16=u16)
    names = []
    for v in range(V):
        fn = tmp_path / f"view{v}.raw"
        extra = np.zeros((3, H, W), dtype=np.uint16) if v == 0 else np.zeros((0, H, W), dtype=np.uint16)
        np.concatenate([pr.views[v], extra]).tofile(fn)          # a longer file is fine: the first N planes are used
        names.append(str(fn))
    out_fn = str(tmp_path / "out.raw")
    with binding.Mvd(W, H, V, pr.psfs, K, T, pr.eps, path) as m:
        m.deconvolve_files(names, out_fn, N, out_u16=u16)
    got = np.fromfile(out_fn, dtype=np.uint16 if u16 else np.float32).reshape(N, H, W)
    assert np.array_equal(got, ref)


def test_files_errors(tmp_path):
    V, W, H, K, T, N = 2, 64, 64, 5, 1, 4
    pr = synth.make_problem(V, N, W, H, K, T, seed=1)
    good = str(tmp_path / "v0.raw")
    pr.views[0].tofile(good)
    short = str(tmp_path / "short.raw")
    pr.views[1][:2].tofile(short)
    with binding.Mvd(W, H, V, pr.psfs, K, T, pr.eps) as m:
        for names in ([good, str(tmp_path / "missing.raw")], [good, short]):
            with pytest.raises(binding.MvdError) as e:
                m.deconvolve_files(names, str(tmp_path / "o.raw"), N)
            assert e.value.code == binding.MVD_ERR_IO
        with pytest.raises(binding.MvdError) as e:
            m.deconvolve_files([good, good], str(tmp_path / "no_such_dir" / "o.raw"), N)
        assert e.value.code == binding.MVD_ERR_IO
