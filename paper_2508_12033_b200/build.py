"""Build liblrdmc.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2508_12033_b200.build [--force] [-v]

Translation units (compiled in parallel, then linked): lrdmc.cu (C-ABI, host logic, rebuild / reconfigure / reduction kernels),
lrdmc_aux.cu (estimators over generations, host-buffer driver, test hooks), comb_static.cu (the allocation-free comb) and kernels.cu ten times -- the walker kernels
{lattice only, + non-local pseudopotential slots, + three-body Jastrow, + both, lattice only as a listed sweep} x {warp-per-walker, team}.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblrdmc.so")
PROBE_LIB = os.path.join(HERE, "liblrdmc_probe.so")      # include/lrdmc_probe.h: FP64 peak micro-benchmarks (bench.py only)
OBJDIR = os.path.join(HERE, "build")
# (source, object name, extra defines)
UNITS = [("lrdmc.cu", "lrdmc.o", []), ("lrdmc_aux.cu", "lrdmc_aux.o", []), ("comb_static.cu", "comb_static.o", [])] + [
    ("kernels.cu", f"kernels_e{ext}_{'team' if team else 'warp'}.o", [f"-DLRDMC_EXT={ext}", f"-DLRDMC_TEAM_TU={team}"])
    for ext in (0, 1, 2, 3, 4) for team in (0, 1)]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC"]


def _deps():
    out = [os.path.join(HERE, "..", "include", "lrdmc.h"), os.path.abspath(__file__)]
    for f in os.listdir(CSRC):
        if f.endswith((".cu", ".cuh", ".h")):
            out.append(os.path.join(CSRC, f))
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    stale = force or not os.path.exists(LIB) or any(os.path.getmtime(d) > os.path.getmtime(LIB) for d in _deps())
    if stale:
        nvcc = os.environ.get("NVCC", "nvcc")
        extra = os.environ.get("LRDMC_NVCC_EXTRA", "").split()       # tuning knobs, e.g. "-DLRDMC_WPB=16 -DLRDMC_MINB=1"
        os.makedirs(OBJDIR, exist_ok=True)
        procs = []
        for src, obj, defs in UNITS:
            cmd = [nvcc] + NVCC_FLAGS + extra + defs + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", os.path.join(OBJDIR, obj), os.path.join(CSRC, src)]
            procs.append((cmd, subprocess.Popen(cmd)))
        failed = [cmd for cmd, p in procs if p.wait() != 0]
        if failed:
            raise subprocess.CalledProcessError(1, failed[0])
        subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + [os.path.join(OBJDIR, o) for _, o, _ in UNITS], check=True)
    probe_src = os.path.join(CSRC, "probe.cu")
    if force or not os.path.exists(PROBE_LIB) or any(os.path.getmtime(d) > os.path.getmtime(PROBE_LIB) for d in (probe_src, os.path.join(CSRC, "peaks.cuh"))):
        subprocess.run([os.environ.get("NVCC", "nvcc")] + NVCC_FLAGS + ["-shared", "-o", PROBE_LIB, probe_src], check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
