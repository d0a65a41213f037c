"""Thin ctypes binding of libmvd (include/mvd.h).  Argument marshalling only.

Every step of the hot path runs in the CUDA library; PyTorch is used for device memory, pinned
memory and streams.  There is no CPU fallback: if `libmvd.so` is missing, or no CUDA device is
present, the compute calls raise.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmvd.so")

MVD_OK, MVD_ERR_INVALID, MVD_ERR_UNSUPPORTED, MVD_ERR_CUDA, MVD_ERR_NOMEM, MVD_ERR_BUSY, MVD_ERR_IO, MVD_ERR_TOO_LARGE = 0, -1, -2, -3, -4, -5, -6, -7
PATH_AUTO, PATH_DIRECT, PATH_FFT = 0, 1, 2
N_KERNEL_CLASSES = 12
PATH_NAMES = {PATH_AUTO: "auto", PATH_DIRECT: "direct", PATH_FFT: "fft"}

# name -> (restype, argtypes): the symbols include/mvd.h declares (tests check the two agree)
_i, _f, _vp, _ll = ctypes.c_int, ctypes.c_float, ctypes.c_void_p, ctypes.c_longlong
_fp = ctypes.POINTER(ctypes.c_float)
SIGNATURES = {
    "mvd_create": (_i, [_i, _i, _i, _fp, _i, _i, _f, ctypes.POINTER(_vp)]),
    "mvd_create_path": (_i, [_i, _i, _i, _fp, _i, _i, _f, _i, ctypes.POINTER(_vp)]),
    "mvd_create_padded": (_i, [_i, _i, _i, _fp, _i, _i, _f, _i, ctypes.POINTER(_vp)]),
    "mvd_get_engine_plane": (_i, [_vp, ctypes.POINTER(_i), ctypes.POINTER(_i)]),
    "mvd_create_backprojectors": (_i, [_i, _i, _i, _fp, _i, _fp, _i, _i, _f, _i, ctypes.POINTER(_vp)]),
    "mvd_build_backprojectors": (_i, [_i, _i, _fp, _i, _fp]),
    "mvd_deconvolve_planes": (_i, [_vp, _vp, _vp, _i, _vp]),
    "mvd_deconvolve_host": (_i, [_vp, _vp, _vp, _i]),
    "mvd_deconvolve_planes_strided": (_i, [_vp, _vp, ctypes.c_size_t, ctypes.c_size_t, ctypes.c_size_t, _vp, _i, _vp]),
    "mvd_deconvolve_host_camera": (_i, [_vp, _vp, _vp, _i]),
    "mvd_destroy": (None, [_vp]),
    "mvd_strerror": (ctypes.c_char_p, [_i]),
    "mvd_last_cuda_error": (_i, [_vp]),
    "mvd_get_path": (_i, [_vp]),
    "mvd_path_supported": (_i, [_i, _i, _i, _i]),
    "mvd_guard_flagged": (_ll, [_vp]),
    "mvd_reserve": (_i, [_vp, _i]),
    "mvd_get_batch_planes": (_i, [_vp, _i]),
    "mvd_set_update_mode": (_i, [_vp, _i]),
    "mvd_set_chunk_planes": (_i, [_vp, _i]),
    "mvd_set_batch_planes": (_i, [_vp, _i]),
    "mvd_set_resident_streams": (_i, [_vp, _i]),
    "mvd_set_pipeline_streams": (_i, [_vp, _i]),
    "mvd_launch_count": (_ll, [_vp]),
    "mvd_launch_count_reset": (None, [_vp]),
    "mvd_profile_enable": (_i, [_vp, _i]),
    "mvd_profile_read": (_i, [_vp, _fp, ctypes.POINTER(_ll)]),
    "mvd_kernel_class_name": (ctypes.c_char_p, [_i]),
    "mvd_version": (ctypes.c_char_p, []),
    "mvd_measure_fp32_peak": (_i, [ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]),
}



class MvdIO(ctypes.Structure):
    """struct mvd_io of include/mvd.h."""
    _fields_ = [("views", _vp), ("view_stride", ctypes.c_size_t), ("plane_stride", ctypes.c_size_t),
                ("row_stride", ctypes.c_size_t), ("weights", _vp), ("out", _vp), ("out_type", _i),
                ("camera_order", _i)]


OUT_F32, OUT_U16 = 0, 1
UPDATE_SEQUENTIAL, UPDATE_PRODUCT = 0, 1
NOALLOC_MAX_VOXELS = 4194304
SIGNATURES.update({
    "mvd_deconvolve_planes_ex": (_i, [_vp, ctypes.POINTER(MvdIO), _i, _vp]),
    "mvd_deconvolve_host_ex": (_i, [_vp, ctypes.POINTER(MvdIO), _i]),
    "mvd_deconvolve_planes_weighted": (_i, [_vp, _vp, _vp, _vp, _i, _vp]),
    "mvd_deconvolve_host_weighted": (_i, [_vp, _vp, _vp, _vp, _i]),
    "mvd_deconvolve_planes_u16": (_i, [_vp, _vp, _vp, _i, _vp]),
    "mvd_deconvolve_host_u16": (_i, [_vp, _vp, _vp, _i]),
    "mvd_deconvolve_files": (_i, [_vp, ctypes.POINTER(ctypes.c_char_p), ctypes.c_char_p, _i, _i]),
    "mvd_deconvolve_planes_noalloc": (_i, [_vp, _vp, _vp, _i, _vp]),
})

_lib: Optional[ctypes.CDLL] = None


class MvdError(RuntimeError):
    def __init__(self, code: int, what: str, cuda: int = 0):
        self.code, self.cuda = code, cuda
        msg = f"{what}: {strerror(code)} (mvd {code}" + (f", cudaError {cuda})" if cuda else ")")
        super().__init__(msg)


def lib() -> ctypes.CDLL:
    """Load libmvd.so.  Fails loudly if it has not been built (python -m paper_1503_07998_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1503_07998_b200.build` "
                              "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def strerror(code: int) -> str:
    return lib().mvd_strerror(int(code)).decode()


def version() -> str:
    return lib().mvd_version().decode()


def path_supported(path: int, plane_w: int, plane_h: int, psf_size: int) -> bool:
    return bool(lib().mvd_path_supported(path, plane_w, plane_h, psf_size))


def kernel_class_names():
    return [lib().mvd_kernel_class_name(k).decode() for k in range(N_KERNEL_CLASSES)]


def measure_fp32_peak() -> Tuple[float, float]:
    """(TFLOP/s of an FFMA-saturating micro-kernel, its SM clock estimate in MHz) on the current device."""
    tf, mhz = ctypes.c_double(0.0), ctypes.c_double(0.0)
    rc = lib().mvd_measure_fp32_peak(ctypes.byref(tf), ctypes.byref(mhz))
    if rc != MVD_OK:
        raise MvdError(rc, "mvd_measure_fp32_peak")
    return tf.value, mhz.value


class Mvd:
    """One plan (mvd_create ... mvd_destroy).  Same names and argument order as the C ABI."""

    def __init__(self, plane_w: int, plane_h: int, n_views: int, psfs: np.ndarray, psf_size: int,
                 iterations: int, eps: float = 1e-6, path: Optional[int] = None,
                 backprojectors: Optional[np.ndarray] = None, padded: bool = False):
        psfs = np.ascontiguousarray(psfs, dtype=np.float32)
        if psfs.size != n_views * psf_size * psf_size:
            raise ValueError("psfs must hold n_views * psf_size * psf_size floats")
        self._h = _vp()
        self.plane_w, self.plane_h, self.n_views = plane_w, plane_h, n_views
        self.psf_size, self.iterations = psf_size, iterations
        p = psfs.ctypes.data_as(_fp)
        if padded:                          # mvd_create_padded: zero-padded planes, cropped result
            if backprojectors is not None:
                raise ValueError("padded plans take the Independent back-projector only")
            rc = lib().mvd_create_padded(plane_w, plane_h, n_views, p, psf_size, iterations, eps,
                                         PATH_AUTO if path is None else path, ctypes.byref(self._h))
        elif backprojectors is not None:    # mvd_create_backprojectors: explicit X_v for step a3
            xs = np.ascontiguousarray(backprojectors, dtype=np.float32)
            if xs.ndim != 3 or xs.shape[0] != n_views or xs.shape[1] != xs.shape[2]:
                raise ValueError("backprojectors must be [n_views][bp_size][bp_size]")
            rc = lib().mvd_create_backprojectors(plane_w, plane_h, n_views, p, psf_size, xs.ctypes.data_as(_fp),
                                                 xs.shape[1], iterations, eps, PATH_AUTO if path is None else path,
                                                 ctypes.byref(self._h))
        elif path is None:
            rc = lib().mvd_create(plane_w, plane_h, n_views, p, psf_size, iterations, eps, ctypes.byref(self._h))
        else:
            rc = lib().mvd_create_path(plane_w, plane_h, n_views, p, psf_size, iterations, eps, path,
                                       ctypes.byref(self._h))
        if rc != MVD_OK:
            self._h = _vp()
            raise MvdError(rc, "mvd_create")

    # -- C ABI, one to one ---------------------------------------------------------------------
    def deconvolve_planes(self, dev_views_u16, dev_out_f32, n_planes: int, stream=None) -> None:
        """dev_views_u16 / dev_out_f32: CUDA torch tensors (uint16 bits in an int16/uint16 tensor; float32)
        or raw device pointers (int).  Enqueues on `stream` (torch stream, raw handle or None = current)."""
        rc = lib().mvd_deconvolve_planes(self._h, _ptr(dev_views_u16), _ptr(dev_out_f32), n_planes,
                                         _stream(stream))
        self._raise(rc, "mvd_deconvolve_planes")

    def deconvolve_planes_strided(self, dev_views_u16, view_stride: int, plane_stride: int, row_stride: int,
                                  dev_out_f32, n_planes: int, stream=None) -> None:
        rc = lib().mvd_deconvolve_planes_strided(self._h, _ptr(dev_views_u16), view_stride, plane_stride,
                                                 row_stride, _ptr(dev_out_f32), n_planes, _stream(stream))
        if rc != MVD_OK:
            self._raise(rc, "mvd_deconvolve_planes_strided")

    def deconvolve_host_camera(self, host_frames_u16, host_out_f32, n_planes: int) -> None:
        rc = lib().mvd_deconvolve_host_camera(self._h, _ptr(host_frames_u16), _ptr(host_out_f32), n_planes)
        if rc != MVD_OK:
            self._raise(rc, "mvd_deconvolve_host_camera")

    def deconvolve_planes_ex(self, views, out, n_planes: int, stream=None, weights=None, out_u16: bool = False,
                             strides: Tuple[int, int, int] = (0, 0, 0)) -> None:
        io = MvdIO(_ptr(views), strides[0], strides[1], strides[2], _ptr(weights), _ptr(out),
                   OUT_U16 if out_u16 else OUT_F32, 0)
        self._raise(lib().mvd_deconvolve_planes_ex(self._h, ctypes.byref(io), n_planes, _stream(stream)),
                    "mvd_deconvolve_planes_ex")

    def deconvolve_host_ex(self, views, out, n_planes: int, weights=None, out_u16: bool = False,
                           camera_order: bool = False) -> None:
        io = MvdIO(_ptr(views), 0, 0, 0, _ptr(weights), _ptr(out), OUT_U16 if out_u16 else OUT_F32, int(camera_order))
        self._raise(lib().mvd_deconvolve_host_ex(self._h, ctypes.byref(io), n_planes), "mvd_deconvolve_host_ex")

    def deconvolve_planes_weighted(self, dev_views_u16, dev_weights_f32, dev_out_f32, n_planes: int, stream=None) -> None:
        self._raise(lib().mvd_deconvolve_planes_weighted(self._h, _ptr(dev_views_u16), _ptr(dev_weights_f32),
                                                         _ptr(dev_out_f32), n_planes, _stream(stream)),
                    "mvd_deconvolve_planes_weighted")

    def deconvolve_host_weighted(self, host_views_u16, host_weights_f32, host_out_f32, n_planes: int) -> None:
        self._raise(lib().mvd_deconvolve_host_weighted(self._h, _ptr(host_views_u16), _ptr(host_weights_f32),
                                                       _ptr(host_out_f32), n_planes), "mvd_deconvolve_host_weighted")

    def deconvolve_planes_u16(self, dev_views_u16, dev_out_u16, n_planes: int, stream=None) -> None:
        self._raise(lib().mvd_deconvolve_planes_u16(self._h, _ptr(dev_views_u16), _ptr(dev_out_u16), n_planes,
                                                    _stream(stream)), "mvd_deconvolve_planes_u16")

    def deconvolve_host_u16(self, host_views_u16, host_out_u16, n_planes: int) -> None:
        self._raise(lib().mvd_deconvolve_host_u16(self._h, _ptr(host_views_u16), _ptr(host_out_u16), n_planes),
                    "mvd_deconvolve_host_u16")

    def deconvolve_planes_noalloc(self, dev_views_u16, dev_out_f32, n_planes: int, stream=None) -> None:
        """mvd_deconvolve_planes_noalloc: allocates nothing; scratch in a fixed 16 MiB device array (NOALLOC_MAX_VOXELS)."""
        self._raise(lib().mvd_deconvolve_planes_noalloc(self._h, _ptr(dev_views_u16), _ptr(dev_out_f32), n_planes,
                                                        _stream(stream)), "mvd_deconvolve_planes_noalloc")

    def deconvolve_files(self, view_paths, out_path: str, n_planes: int, out_u16: bool = False) -> None:
        """mvd_deconvolve_files: raw uint16 view files in, raw float / uint16 file out, disk I/O overlapped.  Blocks."""
        if len(view_paths) != self.n_views:
            raise ValueError("one file per view")
        arr = (ctypes.c_char_p * len(view_paths))(*[os.fsencode(p) for p in view_paths])
        self._raise(lib().mvd_deconvolve_files(self._h, arr, os.fsencode(out_path), n_planes,
                                               OUT_U16 if out_u16 else OUT_F32), "mvd_deconvolve_files")

    def deconvolve_host(self, host_views_u16, host_out_f32, n_planes: int) -> None:
        """host buffers: pinned torch tensors, numpy arrays or raw host pointers.  Blocks."""
        rc = lib().mvd_deconvolve_host(self._h, _ptr(host_views_u16), _ptr(host_out_f32), n_planes)
        self._raise(rc, "mvd_deconvolve_host")

    def destroy(self) -> None:
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().mvd_destroy(self._h)
            self._h = _vp()

    @property
    def path(self) -> int:
        return lib().mvd_get_path(self._h)

    def engine_plane(self) -> Tuple[int, int]:
        """(w, h) of the planes the engine works on (the padded size of a padded plan)."""
        w, hh = _i(0), _i(0)
        self._raise(lib().mvd_get_engine_plane(self._h, ctypes.byref(w), ctypes.byref(hh)), "mvd_get_engine_plane")
        return w.value, hh.value

    def guard_flagged(self) -> int:
        """Plane pairs the FFT engine's guard has handed to the direct engine so far (synchronises)."""
        return int(lib().mvd_guard_flagged(self._h))

    def reserve(self, max_planes: int) -> None:
        self._raise(lib().mvd_reserve(self._h, max_planes), "mvd_reserve")

    def get_batch_planes(self, n_planes: int) -> int:
        rc = lib().mvd_get_batch_planes(self._h, n_planes)
        if rc < 0:
            self._raise(rc, "mvd_get_batch_planes")
        return rc

    def set_update_mode(self, mode: int) -> None:
        """UPDATE_SEQUENTIAL (default) or UPDATE_PRODUCT (the update as printed in PAPER.md:79)."""
        self._raise(lib().mvd_set_update_mode(self._h, mode), "mvd_set_update_mode")

    def set_chunk_planes(self, planes: int) -> None:
        self._raise(lib().mvd_set_chunk_planes(self._h, planes), "mvd_set_chunk_planes")

    def set_resident_streams(self, n: int) -> None:
        self._raise(lib().mvd_set_resident_streams(self._h, n), "mvd_set_resident_streams")

    def set_pipeline_streams(self, n: int) -> None:
        self._raise(lib().mvd_set_pipeline_streams(self._h, n), "mvd_set_pipeline_streams")

    def set_batch_planes(self, planes: int) -> None:
        self._raise(lib().mvd_set_batch_planes(self._h, planes), "mvd_set_batch_planes")

    def launch_count(self) -> int:
        return int(lib().mvd_launch_count(self._h))

    def launch_count_reset(self) -> None:
        lib().mvd_launch_count_reset(self._h)

    def profile_enable(self, on: bool) -> None:
        self._raise(lib().mvd_profile_enable(self._h, int(on)), "mvd_profile_enable")

    def profile_read(self):
        """{kernel class name: (summed ms, launches)} since the last read (synchronises)."""
        ms = (ctypes.c_float * N_KERNEL_CLASSES)()
        n = (_ll * N_KERNEL_CLASSES)()
        self._raise(lib().mvd_profile_read(self._h, ms, n), "mvd_profile_read")
        return {name: (float(ms[k]), int(n[k])) for k, name in enumerate(kernel_class_names())}

    # -- plumbing ----------------------------------------------------------------------------------
    def _raise(self, rc: int, what: str) -> None:
        if rc != MVD_OK:
            raise MvdError(rc, what, lib().mvd_last_cuda_error(self._h))

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def _ptr(x) -> _vp:
    if x is None:
        return _vp(0)
    if isinstance(x, int):
        return _vp(x)
    if isinstance(x, np.ndarray):
        if not x.flags["C_CONTIGUOUS"]:
            raise ValueError("numpy buffer must be C-contiguous")
        return _vp(x.ctypes.data)
    if hasattr(x, "data_ptr"):
        if not x.is_contiguous():
            raise ValueError("tensor must be contiguous")
        return _vp(x.data_ptr())
    raise TypeError(type(x))


def _stream(s) -> _vp:
    if s is None:
        import torch
        return _vp(torch.cuda.current_stream().cuda_stream)
    if isinstance(s, int):
        return _vp(s)
    return _vp(s.cuda_stream)


BP_INDEPENDENT, BP_EFFICIENT_BAYESIAN, BP_OPTIMIZATION1 = 0, 1, 2


def build_backprojectors(variant: int, psfs: np.ndarray) -> np.ndarray:
    """mvd_build_backprojectors: float32 `[V][K][K]` back-projectors of the paper's variants (host, no device)."""
    psfs = np.ascontiguousarray(psfs, dtype=np.float32)
    V, K, _ = psfs.shape
    out = np.empty_like(psfs)
    rc = lib().mvd_build_backprojectors(int(variant), V, psfs.ctypes.data_as(_fp), K, out.ctypes.data_as(_fp))
    if rc != MVD_OK:
        raise MvdError(rc, "mvd_build_backprojectors")
    return out


def deconvolve(views: np.ndarray, psfs: np.ndarray, iterations: int, eps: float = 1e-6,
               path: Optional[int] = None, host: bool = False, chunk_planes: int = 0,
               batch_planes: int = 0, backprojectors: Optional[np.ndarray] = None,
               resident_streams: int = 0, weights: Optional[np.ndarray] = None, out_u16: bool = False,
               padded: bool = False, product: bool = False) -> np.ndarray:
    """Convenience for tests: numpy uint16 `[V][N][H][W]` in, numpy float32 `[N][H][W]` out, through
    mvd_deconvolve_planes (host=False) or mvd_deconvolve_host (host=True, pinned buffers)."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("no CUDA device: libmvd has no CPU fallback")
    views = np.ascontiguousarray(views, dtype=np.uint16)
    V, N, H, W = views.shape
    K = psfs.shape[-1]
    with Mvd(W, H, V, psfs, K, iterations, eps, path, backprojectors, padded) as m:
        if product:
            m.set_update_mode(UPDATE_PRODUCT)
        if chunk_planes:
            m.set_chunk_planes(chunk_planes)
        if batch_planes:
            m.set_batch_planes(batch_planes)
        if resident_streams:
            m.set_resident_streams(resident_streams)
        tv = torch.from_numpy(views.view(np.int16))
        tw = None if weights is None else torch.from_numpy(np.ascontiguousarray(weights, dtype=np.float32))
        odt = torch.int16 if out_u16 else torch.float32
        if host:
            hv = tv.pin_memory()
            hw = None if tw is None else tw.pin_memory()
            ho = torch.empty((N, H, W), dtype=odt).pin_memory()
            if tw is None and not out_u16:
                m.deconvolve_host(hv, ho, N)
            else:
                m.deconvolve_host_ex(hv, ho, N, weights=hw, out_u16=out_u16)
            res = ho.numpy().copy()
        else:
            dv = tv.cuda()
            dw = None if tw is None else tw.cuda()
            do = torch.empty((N, H, W), dtype=odt, device="cuda")
            if tw is None and not out_u16:
                m.deconvolve_planes(dv, do, N)
            else:
                m.deconvolve_planes_ex(dv, do, N, weights=dw, out_u16=out_u16)
            torch.cuda.synchronize()
            res = do.cpu().numpy()
        return res.view(np.uint16) if out_u16 else res
