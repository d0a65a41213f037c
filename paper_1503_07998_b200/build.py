"""Build libmvd.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1503_07998_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so lands next to this file so that it travels with the
source tree; nothing is installed into site-packages.
"""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(_HERE), "include")
LIB = os.path.join(_HERE, "libmvd.so")
_STAMP = os.path.join(_HERE, "csrc", ".build_stamp")
SOURCES = ["mvd_api.cu", "mvd_direct.cu", "mvd_sep.cu", "mvd_files.cu", "mvd_fft.cu", "mvd_fft_inst_small.cu", "mvd_fft_inst_mid.cu",
           "mvd_fft_inst_large.cu", "mvd_fft_inst_v2.cu", "mvd_fft_inst_v2b.cu", "mvd_fft_inst_more_a.cu", "mvd_fft_inst_more_b.cu", "mvd_peak.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC,-O2,-fvisibility=hidden",
              "-Xptxas", "-v", "-shared", "-cudart", "static"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _digest() -> str:
    h = hashlib.sha1(" ".join(NVCC_FLAGS).encode())
    for root in (CSRC, INCLUDE):
        for name in sorted(os.listdir(root)):
            if name.endswith((".cu", ".cuh", ".h")):
                with open(os.path.join(root, name), "rb") as f:
                    h.update(name.encode())
                    h.update(f.read())
    return h.hexdigest()


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if the sources changed; returns the path of libmvd.so."""
    dig = _digest()
    if not force and os.path.exists(LIB) and os.path.exists(_STAMP):
        with open(_STAMP) as f:
            if f.read().strip() == dig:
                return LIB
    flags = list(NVCC_FLAGS)
    objs = []
    procs = []
    for src in SOURCES:
        obj = os.path.join(CSRC, src[:-3] + ".o")
        cmd = [_nvcc(), *[f for f in flags if f not in ("-shared",)], "-c", "-I", INCLUDE,
               "-o", obj, os.path.join(CSRC, src)]
        cmd = [c for c in cmd]
        # -cudart static belongs to the link step only
        while "-cudart" in cmd:
            k = cmd.index("-cudart")
            del cmd[k:k + 2]
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    log = []
    for src, p in procs:
        out, _ = p.communicate()
        log.append(out)
        if p.returncode != 0:
            sys.stderr.write(out)
            raise RuntimeError(f"nvcc failed on {src}")
    link = [_nvcc(), "-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a",
            "-Xcompiler", "-fPIC", "-o", LIB + ".tmp", *objs]
    subprocess.check_call(link)
    os.replace(LIB + ".tmp", LIB)
    with open(_STAMP, "w") as f:
        f.write(dig)
    with open(os.path.join(CSRC, ".ptxas.log"), "w") as f:
        f.write("\n".join(log))
    if verbose:
        sys.stdout.write("\n".join(log))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
