"""Compile the oracle (test infrastructure) with g++.  `python -m oracle.build`."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "magnus_oracle.cpp")
LIB = os.path.join(HERE, "libmagnus_oracle.so")

# No -ffast-math, no -march=native (no FMA contraction): plain IEEE double.
# -fcx-limited-range only drops the inf/NaN recovery of complex multiplication
# (the arithmetic on finite values is the textbook (ac-bd, ad+bc)).
FLAGS = ["-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
         "-fcx-limited-range", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["g++", *FLAGS, SRC, "-o", LIB, "-lquadmath"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
