"""Writes tests/golden/config{3,4,5}_samples.json: fp64 oracle outputs of a few full-size planes.

    python tests/golden/make_golden.py [cid ...]

Calls ONLY oracle/ and the seeded input generator (paper_1503_07998_b200.synth holds no method
arithmetic); nothing here touches the CUDA path.  Configs 3-5 of BASELINE.json are too large for a
live oracle run inside the test suite (14 s / 29 s / 231 s per plane per core),
so the GPU parity tests compare against these stored planes: per plane, the oracle value at 2048
seeded pixel positions plus the plane's sum, maximum and sum of squares.

What the values are: psi after T sequential multi-view RL iterations (readings A1-A7 of
DESIGN.md) of plane p of the config's seeded synthetic stack.
"""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import mvd_oracle  # noqa: E402
from paper_1503_07998_b200 import synth  # noqa: E402

N_SAMPLES = 2048


def golden_planes(cfg):
    return [cfg.N // 2, cfg.N - 1]


def sample_positions(cfg, p):
    rng = np.random.default_rng([synth.SEED, cfg.cid, p, 4242])
    return rng.integers(0, cfg.H * cfg.W, N_SAMPLES)


def make(cid: int) -> str:
    cfg = synth.config(cid)
    psfs = synth.config_psfs(cid)
    planes = golden_planes(cfg)
    views = synth.views(cfg, planes, psfs)
    t0 = time.time()
    out = mvd_oracle.deconvolve(views, psfs, cfg.T, cfg.eps, n_threads=len(planes))
    dt = time.time() - t0
    rec = {"config": cid, "name": cfg.name, "T": cfg.T, "eps": cfg.eps, "oracle_seconds": round(dt, 1),
           "what": "fp64 oracle psi after T iterations at sampled pixels (flat index y*W+x)", "planes": []}
    for k, p in enumerate(planes):
        pos = sample_positions(cfg, p)
        flat = out[k].ravel()
        rec["planes"].append({
            "plane": int(p), "sum": float(flat.sum()), "max": float(flat.max()),
            "sumsq": float((flat ** 2).sum()),
            "view_sums": [int(views[v, k].astype(np.int64).sum()) for v in range(cfg.V)],
            "pos": [int(q) for q in pos], "val": [float(flat[q]) for q in pos]})
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), f"config{cid}_samples.json")
    with open(path, "w") as f:
        json.dump(rec, f)
    return path


if __name__ == "__main__":
    for cid in ([int(a) for a in sys.argv[1:]] or [3, 4, 5]):
        print(make(cid))
