"""Build the CPU oracle shared library (test infrastructure; see gp_oracle.c header).

-ffp-contract=off : no fused multiply-add unless the source writes fmaf (contract C0).
-mfma             : fmaf() becomes one vfmadd instruction instead of a libm call.
No -march=native: the library is built here and also travels to the GPU box.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "gp_oracle.c")
SRCS = [SRC, os.path.join(HERE, "gp_sim_oracle.c")]      # renderer; dynamics + vectorised observation (NEXT-4)
LIB = os.path.join(HERE, "libgp_oracle.so")
CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-mfma", "-std=c99",
          "-Wall", "-Wextra", "-shared", "-fPIC"]


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and all(os.path.getmtime(LIB) >= os.path.getmtime(x) for x in SRCS)):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.check_call(["gcc", *CFLAGS, *SRCS, "-o", tmp, "-lm"])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
