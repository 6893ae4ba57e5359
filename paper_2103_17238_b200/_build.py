"""Builds libsdm_b200.so (the C-ABI library of include/sdm.h) in-tree with nvcc for sm_100a.

    python -m paper_2103_17238_b200._build [--force] [--verbose]

Every translation unit is compiled to its own object (in parallel; only the stale ones) and the objects are
linked into the shared library.  -fmad=false: no FMA contraction anywhere (the pair probability and the volume
update must round exactly like the written operation order; the kernels also use __dmul_rn/__dadd_rn explicitly).
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
OUT = os.path.join(HERE, "libsdm_b200.so")
SOURCES = ["sdm_api.cu", "sdm_hist.cu", "sdm_sort.cu", "sdm_pair.cu", "sdm_cellsort.cu", "sdm_compact.cu",
           "sdm_spectrum.cu", "sdm_displace.cu", "sdm_box.cu", "sdm_bucket.cu", "sdm_noalloc.cu"]
HEADERS = ["sdm_device.cuh", "sdm_internal.h", "sdm_pair.cuh", os.path.join("..", "..", "include", "sdm.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-fmad=false",
    "-Xcompiler", "-fPIC",
]
LINK_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "--cudart=static", "-Xcompiler", "-fPIC"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def _obj(src: str) -> str:
    return os.path.join(OBJ, os.path.splitext(src)[0] + ".o")


def _stale(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def _common_deps():
    return [os.path.join(CSRC, h) for h in HEADERS] + [os.path.abspath(__file__)]


def needs_build() -> bool:
    return _stale(OUT, [os.path.join(CSRC, s) for s in SOURCES] + _common_deps())


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or needs_build()):
        return OUT
    os.makedirs(OBJ, exist_ok=True)
    nvcc = _nvcc()
    common = _common_deps()
    todo = [s for s in SOURCES if force or _stale(_obj(s), [os.path.join(CSRC, s)] + common)]

    def compile_one(src: str) -> None:
        cmd = [nvcc, *NVCC_FLAGS]
        if verbose:
            cmd += ["-Xptxas", "-v"]
        cmd += ["-c", os.path.join(CSRC, src), "-o", _obj(src)]
        subprocess.run(cmd, check=True)

    with ThreadPoolExecutor(max_workers=min(len(todo), os.cpu_count() or 1) or 1) as pool:
        list(pool.map(compile_one, todo))
    subprocess.run([nvcc, *LINK_FLAGS, *[_obj(s) for s in SOURCES], "-o", OUT], check=True)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
