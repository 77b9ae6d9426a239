"""Build liblrdmc.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2508_12033_b200.build [--force]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblrdmc.so")
SOURCES = ["lrdmc.cu", "lrdmc_aux.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC", "-shared"]


def _deps():
    out = [os.path.join(HERE, "..", "include", "lrdmc.h")]
    for f in os.listdir(CSRC):
        if f.endswith((".cu", ".cuh", ".h")):
            out.append(os.path.join(CSRC, f))
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    stale = force or not os.path.exists(LIB) or any(os.path.getmtime(d) > os.path.getmtime(LIB) for d in _deps())
    if stale:
        nvcc = os.environ.get("NVCC", "nvcc")
        extra = os.environ.get("LRDMC_NVCC_EXTRA", "").split()       # tuning knobs, e.g. "-DLRDMC_WPB=16 -DLRDMC_MINB=1"
        cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
