"""Compile the C oracle (test infrastructure) with gcc.  `python -m oracle.build`.

Building the checker is not using it: __graft_entry__.build() calls this too.
Flags: no FMA contraction (every fused multiply-add in the oracle is an explicit
fmaf), rounding-mode changes respected (-frounding-math), OpenMP for the outer
particle loop only.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "liboracle.so")
SRCS = [os.path.join(HERE, "neighbors.c"), os.path.join(HERE, "neighbors_f64.c"), os.path.join(HERE, "tree.c")]
CFLAGS = ["-O2", "-fopenmp", "-ffp-contract=off", "-frounding-math", "-fno-fast-math",
          "-shared", "-fPIC", "-Wall", "-Wno-unknown-pragmas"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in SRCS)


def build(force: bool = False) -> str:
    if force or needs_build():
        cmd = ["gcc", *CFLAGS, "-o", LIB, *SRCS, "-lm"]
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
