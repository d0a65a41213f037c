"""Writes the stored oracle values of BASELINE.json's configs 3-5 (full-size planes):

    tests/golden/config{3,4,5}_samples.json   sampled pixels + sums of two planes (middle, last)
    tests/golden/config{3,4,5}_planes.npz     WHOLE planes, fp64 oracle output rounded to fp32, of
                                              planes {0, B-1, B, N/2, N-1} (B = the pipeline's batch)

    python tests/golden/make_golden.py [--samples | --planes] [cid ...]      (default: both, 3 4 5)

Calls ONLY oracle/ and the seeded input generator (paper_1503_07998_b200.synth holds no method
arithmetic); nothing here touches the CUDA path.  Configs 3-5 of BASELINE.json are too large for a
live oracle run inside the test suite (14 s / 29 s / 231 s per plane per core),
so the GPU parity tests compare against these stored planes: per plane, the oracle value at 2048
seeded pixel positions plus the plane's sum, maximum and sum of squares (JSON), and element by element
against whole stored planes (npz; 2-6 MB per plane): first, middle and last plane of the stack and the two
planes on either side of the first batch boundary of the library's 3-stream pipeline.

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


# planes per pipeline batch of libmvd's default policy for the config (csrc/mvd_api.cu default_batch: ~64 MiB
# of uint16 input per batch); the GPU test asks the library for the value in force and, if it differs,
# places the stored planes at the real boundary
PIPELINE_BATCH = {3: 16, 4: 10, 5: 6}


def whole_planes(cfg):
    b = PIPELINE_BATCH[cfg.cid]
    return [0, b - 1, b, cfg.N // 2, cfg.N - 1]


def make_planes(cid: int) -> str:
    cfg = synth.config(cid)
    psfs = synth.config_psfs(cid)
    planes = whole_planes(cfg)
    views = synth.views(cfg, planes, psfs)
    t0 = time.time()
    out = mvd_oracle.deconvolve(views, psfs, cfg.T, cfg.eps, n_threads=len(planes))
    dt = time.time() - t0
    arrays = {f"plane_{p}": out[k].astype(np.float32) for k, p in enumerate(planes)}
    arrays["planes"] = np.array(planes, dtype=np.int64)
    arrays["pipeline_batch"] = np.array(PIPELINE_BATCH[cid], dtype=np.int64)
    arrays["view_sums"] = np.array([[int(views[v, k].astype(np.int64).sum()) for v in range(cfg.V)]
                                    for k in range(len(planes))], dtype=np.int64)
    arrays["oracle_seconds"] = np.array(round(dt, 1))
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), f"config{cid}_planes.npz")
    np.savez_compressed(path, **arrays)
    return path


if __name__ == "__main__":
    args = sys.argv[1:]
    do_samples = "--planes" not in args
    do_planes = "--samples" not in args
    for cid in ([int(a) for a in args if not a.startswith("--")] or [3, 4, 5]):
        if do_samples:
            print(make(cid))
        if do_planes:
            print(make_planes(cid))
