"""Build oracle/liboracle.so from the plain-C oracle sources (gcc only; no CUDA, no product code).

    python -m oracle.build

Flags follow SURVEY.md §8(c): -O2 -fopenmp -ffp-contract=off, no -ffast-math, no -mfma (glibc's
fmaf() picks the hardware FMA at run time; a software fmaf gives the same bits)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["fma_chain.c", "gemm_rows.c"]
LIB = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    srcs = [os.path.join(HERE, s) for s in SOURCES]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(s) for s in srcs):
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB] + srcs + ["-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
