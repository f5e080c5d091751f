"""Build the CPU oracle shared library (test infrastructure; see lqcd_oracle.cpp header).

    python -m oracle.build        # -> oracle/liblqcd_oracle.so

Plain g++ -O2 with OpenMP; no -ffast-math, no -march flags (the oracle is not tuned)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "lqcd_oracle.cpp")
LIB = os.path.join(HERE, "liblqcd_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
