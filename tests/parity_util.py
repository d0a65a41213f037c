"""Tolerance bookkeeping of the GPU-vs-oracle parity tests.

north_star: relative L2 <= 1e-4 and max relative error <= 1e-3 on pixels above 1 % of max, after all
iterations.  Both are evaluated per plane (threshold from that plane's own maximum) and pooled over
all checked planes; a case passes only if every figure is within its bar.
"""
import numpy as np

REL_L2_BAR = 1e-4
MAX_REL_BAR = 1e-3


def errors(gpu: np.ndarray, oracle: np.ndarray):
    """(worst per-plane rel L2, pooled rel L2, worst max-rel-err over bright pixels)."""
    g = np.asarray(gpu, dtype=np.float64)
    o = np.asarray(oracle, dtype=np.float64)
    assert g.shape == o.shape and g.ndim == 3
    assert np.isfinite(g).all(), "GPU output has non-finite values"
    d = g - o
    num = (d ** 2).sum(axis=(1, 2))
    den = (o ** 2).sum(axis=(1, 2))
    per_plane = np.sqrt(num / np.maximum(den, 1e-300))
    pooled = float(np.sqrt(num.sum() / max(den.sum(), 1e-300)))
    worst_rel = 0.0
    for p in range(o.shape[0]):
        m = o[p].max()
        if m <= 0:
            continue
        bright = o[p] > 0.01 * m
        worst_rel = max(worst_rel, float((np.abs(d[p][bright]) / o[p][bright]).max()))
    return float(per_plane.max()), pooled, worst_rel


def assert_parity(gpu, oracle, what=""):
    l2_plane, l2_pool, mx = errors(gpu, oracle)
    assert l2_plane <= REL_L2_BAR and l2_pool <= REL_L2_BAR and mx <= MAX_REL_BAR, (
        f"{what}: rel L2 per-plane {l2_plane:.3e} pooled {l2_pool:.3e} (bar {REL_L2_BAR}), "
        f"max rel err {mx:.3e} (bar {MAX_REL_BAR})")
    return l2_plane, l2_pool, mx
