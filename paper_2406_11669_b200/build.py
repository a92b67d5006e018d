"""Build step of the CUDA library: nvcc -> paper_2406_11669_b200/libgrmhd.so (in-tree).

sm_100a only (no multi-arch dispatch).  The runtime is linked statically so the library
loads on a box without a GPU (symbol checks) and fails at the first CUDA call instead.
"""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libgrmhd.so")
SOURCES = ["grmhd.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def _deps():
    out = [os.path.join(_HERE, "..", "include", "grmhd.h")]
    for f in os.listdir(CSRC):
        if f.endswith((".cu", ".cuh", ".h")):
            out.append(os.path.join(CSRC, f))
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    stale = (not os.path.exists(LIB)) or any(
        os.path.getmtime(LIB) < os.path.getmtime(p) for p in _deps())
    if force or stale:
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        # GRMHD_NVCC_EXTRA: extra nvcc flags (e.g. "-DFT_NSLOTS=2") for tuning sweeps of the
        # compile-time parameters the kernels expose
        extra = os.environ.get("GRMHD_NVCC_EXTRA", "").split()
        cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + \
              ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
