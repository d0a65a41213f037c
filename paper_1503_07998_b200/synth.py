"""Seeded synthetic light-sheet-like inputs for plane-wise multi-view RL deconvolution.

This module is the ONLY code shared between the CUDA path and the CPU oracle.  It holds none of
the method's arithmetic (no RL update, no blur/ratio/back-projection of an estimate): it only
fabricates what a microscope would have delivered -- registered uint16 views of a phantom and the
per-view 2D PSFs -- with the structure of the paper's data (PAPER.md:39 nuclei-like blobs, :87
uint16 camera counts, :43/:199 anisotropic PSFs, sigma_lateral 1.5-2.5 px, sigma_axial 5-10 px).
The recipe is SURVEY.md section 8(d) / BASELINE.json `configs`; DESIGN.md restates it.

Everything is addressable per plane (`views_plane`) so that any plane of a 13 GB stack can be
produced alone, identically, on either box.

Layouts (same as include/mvd.h): PSFs float32 `[V][K][K]` = `[view][z][x]`, x fastest;
views uint16 `[V][N][H][W]` = `[view][plane][z][x]`.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Iterable, Optional, Sequence

import numpy as np

SEED = 15030799  # arXiv id 1503.07998, digits run together
EPS = np.float32(1e-6)
BLOB_HALF = 12  # rendered half-window of a blob: 4 * sigma_max


# ----------------------------------------------------------------------------------------------
# PSF builders (fp64, normalised to sum 1, then rounded to fp32)
# ----------------------------------------------------------------------------------------------
def _normalise(p: np.ndarray) -> np.ndarray:
    p = np.asarray(p, dtype=np.float64)
    return p / p.sum()


def gaussian_psf64(K: int, sigma_x: float, sigma_z: float) -> np.ndarray:
    """Axis-aligned anisotropic Gaussian on a K x K grid, `[z][x]`, fp64, sum 1."""
    c = (K - 1) // 2
    u = np.arange(K, dtype=np.float64) - c
    gz = np.exp(-(u ** 2) / (2.0 * sigma_z ** 2))
    gx = np.exp(-(u ** 2) / (2.0 * sigma_x ** 2))
    return _normalise(gz[:, None] * gx[None, :])


def ring_psf64(K: int, radius: float, sigma_r: float) -> np.ndarray:
    """Centred ring with a Gaussian radial profile, sum 1 (config 3's weak side lobe)."""
    c = (K - 1) // 2
    u = np.arange(K, dtype=np.float64) - c
    rr = np.sqrt(u[:, None] ** 2 + u[None, :] ** 2)
    return _normalise(np.exp(-((rr - radius) ** 2) / (2.0 * sigma_r ** 2)))


def rotated_psf64(base: np.ndarray, theta_deg: float) -> np.ndarray:
    """Rotate `base` about its centre by theta (bilinear resampling, zero outside), sum 1."""
    K = base.shape[0]
    c = (K - 1) / 2.0
    th = np.deg2rad(theta_deg)
    ct, st = np.cos(th), np.sin(th)
    jj, ii = np.meshgrid(np.arange(K, dtype=np.float64) - c,
                         np.arange(K, dtype=np.float64) - c, indexing="ij")
    # output sample (z=jj, x=ii) reads the base at the position rotated by -theta
    xs = ct * ii + st * jj + c
    zs = -st * ii + ct * jj + c
    x0 = np.floor(xs).astype(np.int64)
    z0 = np.floor(zs).astype(np.int64)
    fx = xs - x0
    fz = zs - z0
    out = np.zeros_like(base, dtype=np.float64)
    for dz, wz in ((0, 1.0 - fz), (1, fz)):
        for dx, wx in ((0, 1.0 - fx), (1, fx)):
            zz = z0 + dz
            xx = x0 + dx
            ok = (zz >= 0) & (zz < K) & (xx >= 0) & (xx < K)
            val = np.where(ok, base[np.clip(zz, 0, K - 1), np.clip(xx, 0, K - 1)], 0.0)
            out += wz * wx * val
    out[np.abs(out) < 1e-300] = 0.0
    return _normalise(out)


def random_psf(K: int, rng: np.random.Generator, sparsity: float = 0.0) -> np.ndarray:
    """Random ASYMMETRIC non-negative PSF, sum 1, fp32 (for parity cases the configs lack)."""
    p = rng.random((K, K))
    if sparsity > 0.0:
        p = p * (rng.random((K, K)) >= sparsity)
        if p.sum() == 0.0:
            p[0, 0] = 1.0
    # a smooth asymmetric envelope so the PSF is not white noise
    c = (K - 1) / 2.0
    u = np.arange(K, dtype=np.float64)
    env = np.exp(-((u[:, None] - 0.6 * c) ** 2) / (2.0 * (0.35 * K) ** 2)
                 - ((u[None, :] - 1.3 * c) ** 2) / (2.0 * (0.2 * K + 0.5) ** 2))
    return _normalise(p * env).astype(np.float32)


def delta_psf(K: int, dz: int = 0, dx: int = 0) -> np.ndarray:
    """P[c+dz][c+dx] = 1: convolving with it shifts by (dz, dx)."""
    c = (K - 1) // 2
    p = np.zeros((K, K), dtype=np.float32)
    p[c + dz, c + dx] = 1.0
    return p


# ----------------------------------------------------------------------------------------------
# Configs (BASELINE.json `configs`, SURVEY.md section 8 size table)
# ----------------------------------------------------------------------------------------------
@dataclass(frozen=True)
class Config:
    cid: int          # seeds the RNG streams
    V: int            # views
    N: int            # planes
    W: int            # plane_w (x, fastest)
    H: int            # plane_h (z)
    K: int            # psf_size (odd)
    T: int            # RL iterations
    n_blobs: int
    eps: float = float(EPS)
    name: str = ""

    @property
    def voxels(self) -> int:
        return self.N * self.W * self.H

    @property
    def units(self) -> int:
        """voxel-view-iterations: the numerator of the Mvoxel/s metric."""
        return self.voxels * self.V * self.T

    def with_planes(self, n: int) -> "Config":
        return Config(self.cid, self.V, n, self.W, self.H, self.K, self.T, self.n_blobs,
                      self.eps, self.name)


_BLOB_DENSITY = 20000.0 / (512 * 512 * 256)  # config 2's density, kept for configs 3-5

CONFIGS = {
    1: Config(1, 2, 8, 64, 64, 9, 10, 50, name="config1 2v 8x64x64 K9 T10"),
    2: Config(2, 2, 512, 512, 256, 21, 10, 20000, name="config2 2v 512x512x256 K21 T10"),
    3: Config(3, 4, 1024, 1024, 512, 31, 10, int(round(_BLOB_DENSITY * 1024 * 1024 * 512)),
              name="config3 4v 1024x1024x512 K31 T10"),
    4: Config(4, 2, 2048, 2048, 800, 41, 10, int(round(_BLOB_DENSITY * 2048 * 2048 * 800)),
              name="config4 2v 2048x2048x800 K41 T10"),
    5: Config(5, 6, 256, 1024, 1024, 51, 20, int(round(_BLOB_DENSITY * 256 * 1024 * 1024)),
              name="config5 6v 256x1024x1024 K51 T20"),
}


def config(cid: int) -> Config:
    return CONFIGS[cid]


def config_psfs(cid: int) -> np.ndarray:
    """fp32 `[V][K][K]` PSFs of a BASELINE.json config."""
    cfg = CONFIGS[cid]
    K = cfg.K
    if cid == 1:
        ps = [gaussian_psf64(K, 1.0, 3.0), gaussian_psf64(K, 3.0, 1.0)]
    elif cid == 2:
        ps = [gaussian_psf64(K, 1.5, 5.0), gaussian_psf64(K, 5.0, 1.5)]
    elif cid == 3:
        g = gaussian_psf64(K, 2.0, 7.0)
        ring = ring_psf64(K, 10.0, 1.0)
        a = _normalise(0.95 * g + 0.05 * ring)
        ps = [a, a.T.copy(), a, a.T.copy()]          # 0 / 90 / 180 / 270 degrees
    elif cid == 4:
        ps = [gaussian_psf64(K, 2.5, 9.0), gaussian_psf64(K, 9.0, 2.5)]
    elif cid == 5:
        base = gaussian_psf64(K, 2.0, 10.0)
        ps = [rotated_psf64(base, 60.0 * v) for v in range(6)]
    else:
        raise KeyError(cid)
    out = np.stack(ps).astype(np.float32)
    assert out.shape == (cfg.V, K, K)
    return out


# ----------------------------------------------------------------------------------------------
# Phantom and views
# ----------------------------------------------------------------------------------------------
@dataclass
class Blobs:
    x: np.ndarray
    y: np.ndarray  # plane axis
    z: np.ndarray
    sigma: np.ndarray
    amp: np.ndarray
    order: np.ndarray = field(default=None)  # type: ignore[assignment]


_blob_cache: dict = {}


def blobs_for(cfg: Config, n_planes_volume: Optional[int] = None) -> Blobs:
    """The blob list of a config: centres uniform in the volume, sigma U[1,3], amplitude U[100,1000]."""
    nvol = cfg.N if n_planes_volume is None else n_planes_volume
    key = (cfg.cid, cfg.W, cfg.H, nvol, cfg.n_blobs)
    if key in _blob_cache:
        return _blob_cache[key]
    rng = np.random.default_rng([SEED, cfg.cid])
    n = cfg.n_blobs
    x = rng.uniform(0.0, cfg.W, n)
    y = rng.uniform(0.0, nvol, n)
    z = rng.uniform(0.0, cfg.H, n)
    sigma = rng.uniform(1.0, 3.0, n)
    amp = rng.uniform(100.0, 1000.0, n)
    order = np.argsort(y, kind="stable")
    b = Blobs(x[order], y[order], z[order], sigma[order], amp[order], order)
    _blob_cache[key] = b
    return b


def phantom_plane(cfg: Config, p: int, blobs: Optional[Blobs] = None) -> np.ndarray:
    """fp64 `[H][W]` slice y = p of the blob phantom (background 10, periodic in x and z)."""
    b = blobs_for(cfg) if blobs is None else blobs
    W, H = cfg.W, cfg.H
    plane = np.full((H, W), 10.0, dtype=np.float64)
    lo = np.searchsorted(b.y, p - BLOB_HALF, side="left")
    hi = np.searchsorted(b.y, p + BLOB_HALF, side="right")
    if hi <= lo:
        return plane
    sl = slice(lo, hi)
    dy = b.y[sl] - p
    keep = np.abs(dy) <= 4.0 * b.sigma[sl]
    if not keep.any():
        return plane
    xc, zc, sg, am, dy = b.x[sl][keep], b.z[sl][keep], b.sigma[sl][keep], b.amp[sl][keep], dy[keep]
    d = np.arange(-BLOB_HALF, BLOB_HALF + 1)
    xi = np.floor(xc).astype(np.int64)[:, None] + d[None, :]          # (nb, 25)
    zi = np.floor(zc).astype(np.int64)[:, None] + d[None, :]
    inv = 1.0 / (2.0 * sg ** 2)
    gx = np.exp(-((xi - xc[:, None]) ** 2) * inv[:, None])
    gz = np.exp(-((zi - zc[:, None]) ** 2) * inv[:, None])
    ay = am * np.exp(-(dy ** 2) * inv)
    contrib = ay[:, None, None] * gz[:, :, None] * gx[:, None, :]     # (nb, 25, 25)
    zz = np.broadcast_to((zi % H)[:, :, None], contrib.shape)
    xx = np.broadcast_to((xi % W)[:, None, :], contrib.shape)
    np.add.at(plane, (zz.ravel(), xx.ravel()), contrib.ravel())
    return plane


def _embed_psf_periodic(P: np.ndarray, H: int, W: int) -> np.ndarray:
    """K x K PSF placed on an H x W periodic grid with its centre at (0, 0) (taps alias if K > H, W)."""
    K = P.shape[0]
    c = (K - 1) // 2
    g = np.zeros((H, W), dtype=np.float64)
    jj = (np.arange(K) - c) % H
    ii = (np.arange(K) - c) % W
    np.add.at(g, (np.repeat(jj, K), np.tile(ii, K)), np.asarray(P, dtype=np.float64).ravel())
    return g


def simulate_view(truth: np.ndarray, P: np.ndarray, rng: np.random.Generator) -> np.ndarray:
    """What the camera records: Poisson(truth (*) P, periodic), clipped to uint16 (input synthesis only)."""
    H, W = truth.shape
    spec = np.fft.rfft2(truth) * np.fft.rfft2(_embed_psf_periodic(P, H, W))
    lam = np.fft.irfft2(spec, s=(H, W))
    lam = np.clip(lam, 0.0, None)
    return np.clip(rng.poisson(lam), 0, 65535).astype(np.uint16)


def views_plane(cfg: Config, p: int, psfs: Optional[np.ndarray] = None) -> np.ndarray:
    """uint16 `[V][H][W]`: all views of plane p of a BASELINE.json config."""
    psfs = config_psfs(cfg.cid) if psfs is None else psfs
    truth = phantom_plane(cfg, p)
    out = np.empty((cfg.V, cfg.H, cfg.W), dtype=np.uint16)
    for v in range(cfg.V):
        rng = np.random.default_rng([SEED, cfg.cid, p, v])
        out[v] = simulate_view(truth, psfs[v], rng)
    return out


def views(cfg: Config, planes: Optional[Iterable[int]] = None,
          psfs: Optional[np.ndarray] = None, out: Optional[np.ndarray] = None) -> np.ndarray:
    """uint16 `[V][n][H][W]` for the given planes (default: all cfg.N planes)."""
    planes = list(range(cfg.N)) if planes is None else list(planes)
    psfs = config_psfs(cfg.cid) if psfs is None else psfs
    if out is None:
        out = np.empty((cfg.V, len(planes), cfg.H, cfg.W), dtype=np.uint16)
    for k, p in enumerate(planes):
        out[:, k] = views_plane(cfg, p, psfs)
    return out


# ----------------------------------------------------------------------------------------------
# Free-form problems for parity / edge cases that the five configs do not provide
# ----------------------------------------------------------------------------------------------
@dataclass
class Problem:
    psfs: np.ndarray    # float32 [V][K][K]
    views: np.ndarray   # uint16  [V][N][H][W]
    T: int
    eps: float = float(EPS)

    @property
    def V(self): return self.views.shape[0]
    @property
    def N(self): return self.views.shape[1]
    @property
    def H(self): return self.views.shape[2]
    @property
    def W(self): return self.views.shape[3]
    @property
    def K(self): return self.psfs.shape[1]


def make_problem(V: int, N: int, W: int, H: int, K: int, T: int, seed: int,
                 psf: str = "random", n_blobs: Optional[int] = None,
                 background: float = 10.0) -> Problem:
    """A small seeded problem: blob phantom -> simulated uint16 views, with a chosen PSF family.

    psf: "random" (asymmetric, the case the configs lack), "gauss" (anisotropic, alternating axes),
         "sparse" (asymmetric with ~70 % zero taps).
    """
    rng = np.random.default_rng([SEED, 1000 + seed])
    if psf == "random":
        psfs = np.stack([random_psf(K, rng) for _ in range(V)])
    elif psf == "sparse":
        psfs = np.stack([random_psf(K, rng, sparsity=0.7) for _ in range(V)])
    elif psf == "gauss":
        s_lat, s_ax = max(0.6, K / 14.0), max(1.0, K / 4.5)
        psfs = np.stack([gaussian_psf64(K, *( (s_lat, s_ax) if v % 2 == 0 else (s_ax, s_lat))).astype(np.float32)
                         for v in range(V)])
    else:
        raise ValueError(psf)
    nb = max(1, int(round(3e-3 * W * H))) if n_blobs is None else n_blobs
    vs = np.empty((V, N, H, W), dtype=np.uint16)
    d = np.arange(-BLOB_HALF, BLOB_HALF + 1)
    for p in range(N):
        truth = np.full((H, W), background, dtype=np.float64)
        xc = rng.uniform(0, W, nb); zc = rng.uniform(0, H, nb)
        sg = rng.uniform(1.0, 3.0, nb); am = rng.uniform(100.0, 1000.0, nb)
        xi = np.floor(xc).astype(np.int64)[:, None] + d[None, :]
        zi = np.floor(zc).astype(np.int64)[:, None] + d[None, :]
        inv = 1.0 / (2.0 * sg ** 2)
        gx = np.exp(-((xi - xc[:, None]) ** 2) * inv[:, None])
        gz = np.exp(-((zi - zc[:, None]) ** 2) * inv[:, None])
        contrib = am[:, None, None] * gz[:, :, None] * gx[:, None, :]
        zz = np.broadcast_to((zi % H)[:, :, None], contrib.shape)
        xx = np.broadcast_to((xi % W)[:, None, :], contrib.shape)
        np.add.at(truth, (zz.ravel(), xx.ravel()), contrib.ravel())
        for v in range(V):
            vs[v, p] = simulate_view(truth, psfs[v], rng)
    return Problem(psfs=psfs.astype(np.float32), views=vs, T=T)


def random_views(V: int, N: int, W: int, H: int, seed: int, lo: int = 1, hi: int = 4000) -> np.ndarray:
    """Plain uniform random uint16 views in [lo, hi) (for invariants that need no structure)."""
    rng = np.random.default_rng([SEED, 2000 + seed])
    return rng.integers(lo, hi, size=(V, N, H, W), dtype=np.uint16)


def parity_planes(cfg: Config, n_random: int = 8, batch: Optional[int] = None) -> Sequence[int]:
    """Fixed plane subset for configs too big for a full-volume oracle run."""
    rng = np.random.default_rng([SEED, cfg.cid, 777])
    s = {0, cfg.N - 1, cfg.N // 2}
    if batch:
        for b in (batch, 2 * batch):
            for q in (b - 1, b):
                if 0 <= q < cfg.N:
                    s.add(q)
    s.update(int(q) for q in rng.integers(0, cfg.N, n_random))
    return sorted(s)
