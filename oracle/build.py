"""Build the CPU oracle shared library (test infrastructure; see lqcd_oracle.cpp header).

    python -m oracle.build        # -> oracle/liblqcd_oracle.so

Plain g++ -O2 with OpenMP; no -ffast-math, no -march flags (the oracle is not tuned).  Rebuilt when the source
differs from the one the library was built from (hash stored beside it; copies of the tree do not keep mtimes)."""
from __future__ import annotations

import fcntl
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "lqcd_oracle.cpp")
LIB = os.path.join(HERE, "liblqcd_oracle.so")
STAMP = LIB + ".srchash"
CMD = ["g++", "-std=c++17", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra"]


def _hash() -> str:
    with open(SRC, "rb") as fh:
        return hashlib.sha256(" ".join(CMD).encode() + fh.read()).hexdigest()


def _up_to_date() -> bool:
    if not (os.path.exists(LIB) and os.path.exists(STAMP)):
        return False
    with open(STAMP) as fh:
        return fh.read().strip() == _hash()


def build(force: bool = False) -> str:
    if not force and _up_to_date():
        return LIB
    with open(LIB + ".lock", "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        if force or not _up_to_date():
            tmp = LIB + f".tmp{os.getpid()}"
            subprocess.run(CMD + ["-o", tmp, SRC], check=True)
            os.replace(tmp, LIB)
            with open(STAMP, "w") as fh:
                fh.write(_hash() + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
