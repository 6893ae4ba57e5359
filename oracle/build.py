"""Build the oracle shared library (test infrastructure, not the product).

    python oracle/build.py

g++ -O2 -ffp-contract=off -fno-fast-math: no FMA contraction, IEEE fp64 in the written order
(SURVEY.md section 7 step 0).  The output, oracle/liboracle_sdm.so, is git-ignored.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sdm_oracle.cpp")
OUT = os.path.join(HERE, "liboracle_sdm.so")

FLAGS = [
    "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fno-unsafe-math-optimizations",
    "-mno-fma", "-shared", "-fPIC", "-Wall", "-Wextra",
]


def needs_build() -> bool:
    return (not os.path.exists(OUT)) or os.path.getmtime(OUT) < os.path.getmtime(SRC)


def build(force: bool = False) -> str:
    if force or needs_build():
        cmd = ["g++", *FLAGS, SRC, "-o", OUT]
        subprocess.run(cmd, check=True)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
