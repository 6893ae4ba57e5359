"""Builds libsdm_b200.so (the C-ABI library of include/sdm.h) in-tree with nvcc for sm_100a.

    python -m paper_2103_17238_b200._build [--force] [--verbose]

-fmad=false: no FMA contraction anywhere (the pair probability and the volume update must round
exactly like the written operation order; the kernels also use __dmul_rn/__dadd_rn explicitly).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "libsdm_b200.so")
SOURCES = ["sdm_api.cu", "sdm_hist.cu", "sdm_sort.cu", "sdm_pair.cu", "sdm_cellsort.cu", "sdm_compact.cu", "sdm_spectrum.cu", "sdm_displace.cu"]
HEADERS = ["sdm_device.cuh", "sdm_internal.h", "sdm_pair.cuh", os.path.join("..", "..", "include", "sdm.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-fmad=false",
    "-Xcompiler", "-fPIC", "-shared", "--cudart=static",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(OUT):
        return True
    t = os.path.getmtime(OUT)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        cmd = [_nvcc(), *NVCC_FLAGS, *os.environ.get("SDM_NVCC_EXTRA", "").split()]
        if verbose:
            cmd += ["-Xptxas", "-v"]
        cmd += [os.path.join(CSRC, s) for s in SOURCES] + ["-o", OUT]
        subprocess.run(cmd, check=True)
    return OUT  # SDM_NVCC_EXTRA: extra nvcc flags for tuning experiments (e.g. -DSDM_CF_WARPS=8)


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
