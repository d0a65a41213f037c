"""The C-ABI library builds, loads and exports every symbol include/mvd.h declares (no GPU needed)."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1503_07998_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.lib()


def _declared_symbols():
    with open(os.path.join(ROOT, "include", "mvd.h")) as f:
        text = f.read()
    return sorted(set(re.findall(r"MVD_API\s+[\w\s\*]+?\b(mvd_\w+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    names = _declared_symbols()
    assert len(names) >= 8 and "mvd_create" in names and "mvd_deconvolve_host" in names
    for n in names:
        assert hasattr(lib, n), f"libmvd.so does not export {n}"
    # and the binding marshals exactly the declared set
    assert sorted(binding.SIGNATURES) == names


def test_no_torch_types_in_header():
    with open(os.path.join(ROOT, "include", "mvd.h")) as f:
        text = f.read()
    assert "torch" not in text and "at::" not in text and "std::" not in text
    assert 'extern "C"' in text


def test_strerror_and_version(lib):
    assert binding.strerror(0) == "ok"
    for code in (-1, -2, -3, -4, -5, -99):
        assert isinstance(binding.strerror(code), str) and binding.strerror(code)
    assert "sm_100a" in binding.version()
    assert len(binding.kernel_class_names()) == binding.N_KERNEL_CLASSES


def test_path_supported_needs_no_device(lib):
    assert binding.path_supported(binding.PATH_DIRECT, 64, 64, 9)
    assert binding.path_supported(binding.PATH_DIRECT, 37, 23, 5)
    assert not binding.path_supported(binding.PATH_DIRECT, 64, 64, 8)        # even K
    assert not binding.path_supported(binding.PATH_DIRECT, 0, 64, 9)
    for cid_shape in ((64, 64, 9), (512, 256, 21), (1024, 512, 31), (2048, 800, 41), (1024, 1024, 51)):
        assert binding.path_supported(binding.PATH_AUTO, *cid_shape)


def test_fft_engine_length_set(lib):
    """Every 2^a 3^b 5^c length the kernels are instantiated for, as rows and as columns."""
    lengths = [32, 64, 80, 96, 128, 160, 192, 256, 320, 384, 512, 640, 768, 800, 1024, 1280, 1536, 1600, 2048]
    for w in lengths:
        for h in lengths:
            assert binding.path_supported(binding.PATH_FFT, w, h, 9), (w, h)
    for n in (33, 100, 2000, 4096):
        assert not binding.path_supported(binding.PATH_FFT, n, 256, 9)


def test_create_validates_before_touching_the_device(lib):
    """Argument errors are reported as MVD_ERR_INVALID even on a box without a GPU."""
    P = np.full((1, 3, 3), 1 / 9, dtype=np.float32)
    h = ctypes.c_void_p()

    def create(W=8, H=8, V=1, psf=P, K=3, T=1, eps=1e-6, out=h):
        return binding.lib().mvd_create(W, H, V, psf.ctypes.data_as(ctypes.POINTER(ctypes.c_float)) if psf is not None else None,
                                        K, T, eps, ctypes.byref(out) if out is not None else None)

    assert create(W=0) == binding.MVD_ERR_INVALID
    assert create(H=-1) == binding.MVD_ERR_INVALID
    assert create(V=0) == binding.MVD_ERR_INVALID
    assert create(K=4) == binding.MVD_ERR_INVALID
    assert create(T=-1) == binding.MVD_ERR_INVALID
    assert create(eps=0.0) == binding.MVD_ERR_INVALID
    assert create(eps=float("nan")) == binding.MVD_ERR_INVALID
    assert create(psf=None) == binding.MVD_ERR_INVALID
    assert create(out=None) == binding.MVD_ERR_INVALID
    bad = P.copy(); bad[0, 1, 1] = -0.5
    assert create(psf=bad) == binding.MVD_ERR_INVALID
    bad[0, 1, 1] = np.inf
    assert create(psf=bad) == binding.MVD_ERR_INVALID
    assert h.value is None


def test_null_handle_calls_are_safe(lib):
    L = binding.lib()
    L.mvd_destroy(None)
    assert L.mvd_deconvolve_planes(None, None, None, 1, None) == binding.MVD_ERR_INVALID
    assert L.mvd_deconvolve_host(None, None, None, 1) == binding.MVD_ERR_INVALID
    assert L.mvd_last_cuda_error(None) == 0
    assert L.mvd_launch_count(None) == 0


def test_product_does_not_import_the_oracle():
    """The CUDA package and the oracle share no code: neither imports, links or names the other."""
    pkg = os.path.join(ROOT, "paper_1503_07998_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                with open(os.path.join(dirpath, fn)) as f:
                    src = f.read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), fn
                assert "mvd_oracle" not in src and "oracle/" not in src, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c")):
            with open(os.path.join(ROOT, "oracle", fn)) as f:
                src = f.read()
            assert not re.search(r"^\s*(import|from)\s+paper_1503_07998_b200\b", src, flags=re.M), fn
            assert "libmvd.so" not in src and "csrc/" not in src and "mvd.h\"" not in src, fn


def test_header_constants_match_the_binding():
    with open(os.path.join(ROOT, "include", "mvd.h")) as f:
        text = f.read()
    def const(name):
        m = re.search(name + r"\s*=\s*(-?\d+)", text)
        assert m, name
        return int(m.group(1))
    assert const("MVD_NOALLOC_MAX_VOXELS") == binding.NOALLOC_MAX_VOXELS
    assert const("MVD_N_KERNEL_CLASSES") == binding.N_KERNEL_CLASSES
    for name, val in (("MVD_ERR_INVALID", binding.MVD_ERR_INVALID), ("MVD_ERR_UNSUPPORTED", binding.MVD_ERR_UNSUPPORTED),
                      ("MVD_ERR_CUDA", binding.MVD_ERR_CUDA), ("MVD_ERR_NOMEM", binding.MVD_ERR_NOMEM),
                      ("MVD_ERR_IO", binding.MVD_ERR_IO), ("MVD_ERR_TOO_LARGE", binding.MVD_ERR_TOO_LARGE),
                      ("MVD_UPDATE_PRODUCT", binding.UPDATE_PRODUCT), ("MVD_OUT_U16", binding.OUT_U16)):
        assert const(name) == val, name
