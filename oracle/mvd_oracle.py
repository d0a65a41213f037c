"""ctypes loader for the fp64 CPU oracle (oracle/mvd_oracle.c).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It never imports the CUDA package, and the CUDA package never imports it.

Parity unpinned (no value in the paper fixes the READING; the arithmetic under the reading is pinned in
tests/test_oracle_pins.py): the per-view weights of `deconvolve(weights=)` (reading W1), the zero fill of
`deconvolve_padded` (reading PD1), the variant builders of `backprojectors()` (readings B1-B4).  Everything else --
`deconvolve`, `deconvolve_product`, `blur`, `backproject`, `trace` -- is pinned (P1-P11, PX1-PX4, PP1-PP3).

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
    lib.mvd_oracle_x.argtypes = [i, i, i, fp, i, fp, i, i, d, up, dp, i, i, i]
    lib.mvd_oracle_x.restype = i
    lib.mvd_oracle_w.argtypes = [i, i, i, fp, i, fp, i, i, d, up, fp, dp, i, i, i]
    lib.mvd_oracle_w.restype = i
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
               n_threads: Optional[int] = None, literal: bool = False,
               backprojectors: Optional[np.ndarray] = None,
               weights: Optional[np.ndarray] = None) -> np.ndarray:
    """fp64 `[N][H][W]` = T sequential multi-view RL iterations on every plane.

    views uint16 `[V][N][H][W]`, psfs float32 `[V][K][K]`.  eps is first rounded to fp32 (the C ABI
    of the product takes `float eps`), so both sides clamp at the identical threshold (reading A6).
    backprojectors float32 `[V][KX][KX]` (optional): step a3 is the true convolution r * X_v with these
    kernels instead of the correlation with P_v; None is the Independent variant.
    weights float32 `[V][N][H][W]` in [0, 1] (optional): step a4 becomes psi <- psi . (w_v q + 1 - w_v)
    ("weights"; READING W1, parity unpinned).
    """
    views = np.ascontiguousarray(views, dtype=np.uint16)
    psfs = _f32(psfs)
    assert views.ndim == 4 and psfs.ndim == 3 and psfs.shape[0] == views.shape[0]
    V, N, H, W = views.shape
    K = psfs.shape[1]
    assert psfs.shape[2] == K
    out = np.empty((N, H, W), dtype=np.float64)
    nt = n_cores() if n_threads is None else n_threads
    if weights is not None:
        w = _f32(weights)
        assert w.shape == views.shape
        xs = _f32(backprojectors) if backprojectors is not None else None
        rc = _load().mvd_oracle_w(W, H, V, _ptr(psfs, ctypes.c_float), K,
                                  _ptr(xs, ctypes.c_float) if xs is not None else None,
                                  xs.shape[1] if xs is not None else 0, int(T), float(np.float32(eps)),
                                  _ptr(views, ctypes.c_uint16), _ptr(w, ctypes.c_float),
                                  _ptr(out, ctypes.c_double), N, int(nt), int(bool(literal)))
        if rc != 0:
            raise ValueError(f"mvd_oracle_w rejected its arguments (rc={rc})")
        return out
    if backprojectors is not None:
        xs = _f32(backprojectors)
        assert xs.ndim == 3 and xs.shape[0] == V and xs.shape[1] == xs.shape[2]
        rc = _load().mvd_oracle_x(W, H, V, _ptr(psfs, ctypes.c_float), K, _ptr(xs, ctypes.c_float),
                                  xs.shape[1], int(T), float(np.float32(eps)), _ptr(views, ctypes.c_uint16),
                                  _ptr(out, ctypes.c_double), N, int(nt), int(bool(literal)))
        if rc != 0:
            raise ValueError(f"mvd_oracle_x rejected its arguments (rc={rc})")
        return out
    fn = _load().mvd_oracle_literal if literal else _load().mvd_oracle
    rc = fn(W, H, V, _ptr(psfs, ctypes.c_float), K, int(T), float(np.float32(eps)),
            _ptr(views, ctypes.c_uint16), _ptr(out, ctypes.c_double), N, int(nt))
    if rc != 0:
        raise ValueError(f"mvd_oracle rejected its arguments (rc={rc})")
    return out


def deconvolve_padded(views: np.ndarray, psfs: np.ndarray, T: int, eps: float = 1e-6,
                      n_threads: Optional[int] = None, extra: int = 0,
                      weights: Optional[np.ndarray] = None) -> np.ndarray:
    """The paper's own boundary (Supp. Table 1 caption: the transformed size is "the sum of the
    actual data size and the size of PSF"): every plane of every view is embedded in a plane K - 1 (+ `extra`)
    pixels larger in x and z, the periodic iteration runs on the padded planes, and the result is cropped.
    READING PD1 (the paper does not say what the padding holds; parity of the reading unpinned,
    arithmetic pinned by PD1-PD4): the padding is ZERO.
    Then psi_0 and every later psi are zero in it (the update is multiplicative) and so is r (phi = 0), i.e. the
    result on the plane is the RL iteration with zero boundary conditions -- whatever `extra` is (pin PD1).
    """
    views = np.ascontiguousarray(views, dtype=np.uint16)
    V, N, H, W = views.shape
    K = np.asarray(psfs).shape[1]
    padded = np.zeros((V, N, H + K - 1 + extra, W + K - 1 + extra), dtype=np.uint16)
    padded[:, :, :H, :W] = views
    pw = None
    if weights is not None:      # reading W1 on the padded planes; the weight in the padding is immaterial (psi = 0 there): 0
        pw = np.zeros(padded.shape, dtype=np.float32)
        pw[:, :, :H, :W] = weights
    return np.ascontiguousarray(deconvolve(padded, psfs, T, eps, n_threads, weights=pw)[:, :H, :W])


def deconvolve_product(views: np.ndarray, psfs: np.ndarray, T: int, eps: float = 1e-6,
                       weights: Optional[np.ndarray] = None) -> np.ndarray:
    """The update exactly as PAPER.md:79 prints it (Supp. Note 1): psi^{t+1} = psi^t prod_v (phi_v / (psi^t * P_v)) * P_v^*,
    every view's factor computed from the SAME psi^t (the "simultaneous" form).  north_star's reading (A1) is the
    sequential form of `deconvolve`; this is the other one, offered as an update mode of the library.  Steps a1-a3 are the
    C routines behind `blur` / `backproject`; with weights each factor is w_v q_v + 1 - w_v (reading W1).
    """
    views = np.ascontiguousarray(views, dtype=np.uint16)
    psfs = _f32(psfs)
    V, N, H, W = views.shape
    e32 = float(np.float32(eps))
    out = np.empty((N, H, W), dtype=np.float64)
    for n in range(N):
        phi = views[:, n].astype(np.float64)
        psi = phi.sum(axis=0) / V                                   # a0
        for _ in range(T):
            factor = np.ones_like(psi)
            for v in range(V):
                b = blur(psi, psfs[v])                              # a1, from psi^t for every view
                q = backproject(phi[v] / np.maximum(b, e32), psfs[v])   # a2, a3
                if weights is not None:
                    w = np.asarray(weights[v, n], dtype=np.float64)
                    q = w * q + (1.0 - w)
                factor *= q
            psi = psi * factor                                      # a4, once per iteration
        out[n] = psi
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


# ---------------------------------------------------------------------------------------------
# Back-projectors of Supp. Note 2 section 1, written out from the printed formulas.
# READINGS (the text is garbled and defines none of the operators, B1-B4):
#   B1  "*" is the full (non-periodic) 2D convolution of the small kernels, P^* the flipped PSF;
#   B2  juxtaposition and the product sign are POINTWISE products of kernels laid over a common
#       centre (a kernel is zero outside its support), so X_v lives on P_v^*'s K x K support;
#   B3  W_v is the set of all other views w != v; Optimization I's printed index "v in W_v" is
#       read as "w in W_v";
#   B4  X_v is normalised to sum 1 (constant images then stay a fixed point of the update).
#   Optimization II's printed formula (a product over "v, w in W_v" of P_v^* alone) cannot be
#   recovered from this text and is not built.
# Parity of these READINGS is unpinned (no value in the paper fixes them); what is pinned is their
# arithmetic (tests/test_oracle_pins.py) and, independently, the iteration for ANY given X_v.
# ---------------------------------------------------------------------------------------------
def _full_conv(a: np.ndarray, b: np.ndarray) -> np.ndarray:
    out = np.zeros((a.shape[0] + b.shape[0] - 1, a.shape[1] + b.shape[1] - 1), dtype=np.float64)
    for j in range(b.shape[0]):
        for i in range(b.shape[1]):
            out[j:j + a.shape[0], i:i + a.shape[1]] += b[j, i] * a
    return out


def _centre_crop(a: np.ndarray, K: int) -> np.ndarray:
    oy, ox = (a.shape[0] - K) // 2, (a.shape[1] - K) // 2
    return a[oy:oy + K, ox:ox + K]


def backprojectors(psfs: np.ndarray, variant: str) -> np.ndarray:
    """float32 `[V][K][K]` back-projectors X_v for variant in {"independent", "efficient_bayesian",
    "optimization1"}, fp64 arithmetic, rounded to fp32 at the end."""
    P = np.asarray(psfs, dtype=np.float64)
    V, K, _ = P.shape
    flip = P[:, ::-1, ::-1]
    if variant == "independent":
        return np.ascontiguousarray(flip, dtype=np.float32)         # PAPER.md:104, not normalised: X = P_v^*
    out = np.empty_like(P)
    for v in range(V):
        X = flip[v].copy()
        for w in range(V):
            if w == v:
                continue
            if variant == "efficient_bayesian":                     # PAPER.md:108  P_v^* * P_w * P_w^*
                f = _full_conv(_full_conv(flip[v], P[w]), flip[w])
            elif variant == "optimization1":                        # PAPER.md:112  P_v^* * P_w
                f = _full_conv(flip[v], P[w])
            else:
                raise ValueError(f"unknown variant {variant!r}")
            X = X * _centre_crop(f, K)
        out[v] = X / X.sum()
    return np.ascontiguousarray(out, dtype=np.float32)
