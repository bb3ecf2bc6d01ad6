"""Builds the CPU oracle (oracle/spd_oracle.c -> oracle/libspd_oracle.so) with gcc.

Building the checker is not using it: __graft_entry__.build() calls this; the product path never
loads the result.  Flags: -O3, AVX2+FMA baseline (x86-64-v3, so the .so built on one box runs on
another), OpenMP over GEMV rows, no fp contraction and no fast-math so the arithmetic is IEEE-strict
and identical wherever it is compiled.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = [os.path.join(HERE, "spd_oracle.c")]
HDR = [os.path.join(HERE, "spd_oracle.h")]
LIB = os.path.join(HERE, "libspd_oracle.so")


def build(force: bool = False) -> str:
    newest = max(os.path.getmtime(p) for p in SRC + HDR)
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    cmd = ["gcc", "-std=c11", "-O3", "-march=x86-64-v3", "-ffp-contract=off", "-fno-fast-math",
           "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", LIB] + SRC + ["-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
