"""ctypes loader for the fp64 CPU oracle (oracle/mvd_oracle.c).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It never imports the CUDA package, and the CUDA package never imports it.

The shared object is compiled with gcc on the machine that uses it (seconds), keyed by the source
hash and the host's CPU flags, so a copy built on another box is never executed with the wrong ISA.
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mvd_oracle.c")
_CFLAGS = ["-O3", "-march=native", "-ffp-contract=off", "-fno-fast-math", "-std=c11",
           "-shared", "-fPIC", "-pthread"]
_lib: Optional[ctypes.CDLL] = None


def _cpu_key() -> str:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    return line
    except OSError:
        pass
    return "unknown"


def lib_path() -> str:
    with open(_SRC, "rb") as f:
        h = hashlib.sha1(f.read() + _cpu_key().encode() + " ".join(_CFLAGS).encode()).hexdigest()[:12]
    return os.path.join(_HERE, "_build", f"libmvd_oracle_{h}.so")


def build(force: bool = False) -> str:
    """Compile oracle/mvd_oracle.c for this host; returns the .so path."""
    out = lib_path()
    if os.path.exists(out) and not force:
        return out
    os.makedirs(os.path.dirname(out), exist_ok=True)
    tmp = out + f".tmp{os.getpid()}"
    subprocess.check_call(["gcc", *_CFLAGS, "-o", tmp, _SRC, "-lm"])
    os.replace(tmp, out)
    return out


def _load() -> ctypes.CDLL:
    global _lib
    if _lib is not None:
        return _lib
    lib = ctypes.CDLL(build())
    i, d = ctypes.c_int, ctypes.c_double
    fp = ctypes.POINTER(ctypes.c_float)
    dp = ctypes.POINTER(ctypes.c_double)
    up = ctypes.POINTER(ctypes.c_uint16)
    for name in ("mvd_oracle", "mvd_oracle_literal"):
        fn = getattr(lib, name)
        fn.argtypes = [i, i, i, fp, i, i, d, up, dp, i, i]
        fn.restype = i
    lib.mvd_oracle_trace.argtypes = [i, i, i, fp, i, i, d, up, dp, dp]
    lib.mvd_oracle_trace.restype = i
    for name in ("mvd_oracle_blur", "mvd_oracle_backproject",
                 "mvd_oracle_blur_literal", "mvd_oracle_backproject_literal"):
        fn = getattr(lib, name)
        fn.argtypes = [dp, fp, i, i, i, dp]
        fn.restype = None
    _lib = lib
    return lib


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _ptr(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct))


def n_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def deconvolve(views: np.ndarray, psfs: np.ndarray, T: int, eps: float = 1e-6,
               n_threads: Optional[int] = None, literal: bool = False) -> np.ndarray:
    """fp64 `[N][H][W]` = T sequential multi-view RL iterations on every plane.

    views uint16 `[V][N][H][W]`, psfs float32 `[V][K][K]`.  eps is first rounded to fp32 (the C ABI
    of the product takes `float eps`), so both sides clamp at the identical threshold (reading A6).
    """
    views = np.ascontiguousarray(views, dtype=np.uint16)
    psfs = _f32(psfs)
    assert views.ndim == 4 and psfs.ndim == 3 and psfs.shape[0] == views.shape[0]
    V, N, H, W = views.shape
    K = psfs.shape[1]
    assert psfs.shape[2] == K
    out = np.empty((N, H, W), dtype=np.float64)
    nt = n_cores() if n_threads is None else n_threads
    fn = _load().mvd_oracle_literal if literal else _load().mvd_oracle
    rc = fn(W, H, V, _ptr(psfs, ctypes.c_float), K, int(T), float(np.float32(eps)),
            _ptr(views, ctypes.c_uint16), _ptr(out, ctypes.c_double), N, int(nt))
    if rc != 0:
        raise ValueError(f"mvd_oracle rejected its arguments (rc={rc})")
    return out


def trace(views_plane: np.ndarray, psfs: np.ndarray, T: int, eps: float = 1e-6) -> np.ndarray:
    """fp64 `[T*V][H][W]`: psi after every view update of ONE plane (views_plane uint16 `[V][H][W]`)."""
    views_plane = np.ascontiguousarray(views_plane, dtype=np.uint16)
    psfs = _f32(psfs)
    V, H, W = views_plane.shape
    K = psfs.shape[1]
    out = np.empty((H, W), dtype=np.float64)
    tr = np.empty((max(T * V, 1), H, W), dtype=np.float64)
    rc = _load().mvd_oracle_trace(W, H, V, _ptr(psfs, ctypes.c_float), K, int(T),
                                  float(np.float32(eps)), _ptr(views_plane, ctypes.c_uint16),
                                  _ptr(out, ctypes.c_double), _ptr(tr, ctypes.c_double))
    if rc != 0:
        raise ValueError(f"mvd_oracle_trace rejected its arguments (rc={rc})")
    return tr[: T * V]


def _conv(name: str, img: np.ndarray, P: np.ndarray) -> np.ndarray:
    img = np.ascontiguousarray(img, dtype=np.float64)
    P = _f32(P)
    H, W = img.shape
    out = np.empty_like(img)
    getattr(_load(), name)(_ptr(img, ctypes.c_double), _ptr(P, ctypes.c_float), P.shape[0], W, H,
                           _ptr(out, ctypes.c_double))
    return out


def blur(psi, P, literal=False):
    """a1: psi * P (periodic true convolution)."""
    return _conv("mvd_oracle_blur_literal" if literal else "mvd_oracle_blur", psi, P)


def backproject(r, P, literal=False):
    """a3: r * P^* (periodic correlation with P)."""
    return _conv("mvd_oracle_backproject_literal" if literal else "mvd_oracle_backproject", r, P)
