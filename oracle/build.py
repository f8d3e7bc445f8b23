"""Compile the fp64 C++ oracle into oracle/libra_mppi_oracle.so (g++ only; no CUDA)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ra_mppi_oracle.cpp")
HDR = os.path.join(HERE, "ra_mppi_oracle.h")
LIB = os.path.join(HERE, "libra_mppi_oracle.so")


def build(force: bool = False) -> str:
    newest = max(os.path.getmtime(SRC), os.path.getmtime(HDR))
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    # -ffp-contract=off: no FMA contraction, so the arithmetic is the source's, operation by operation
    cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-ffp-contract=off", "-pthread",
           "-Wall", "-Wextra", "-o", LIB, SRC]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
