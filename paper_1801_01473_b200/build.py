"""Build the CUDA library for sm_100a, in tree:  python -m paper_1801_01473_b200.build

    paper_1801_01473_b200/liblqcd_b200.so      (git-ignored; travels to the GPU box with gpurun)

nvcc cross-compiles without a GPU.  -lineinfo keeps the ncu source page usable.

``build()`` is called by every ``load_library()``: it returns at once when the library was built from the sources
as they are now.  "As they are now" is decided by a hash of the sources stored beside the library
(``liblqcd_b200.so.srchash``), not by modification times, which a copy of the tree (gpurun) does not preserve."""
from __future__ import annotations

import fcntl
import glob
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblqcd_b200.so")
STAMP = LIB + ".srchash"
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared",
    "-cudart", "shared",
]


def sources() -> list[str]:
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps() -> list[str]:
    root = os.path.dirname(HERE)
    return sorted(sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.h"))
                  + glob.glob(os.path.join(root, "include", "*.h")))


def source_hash(extra: list[str] | None = None) -> str:
    h = hashlib.sha256()
    h.update(" ".join(FLAGS + (extra or [])).encode())
    for path in _deps():
        h.update(os.path.basename(path).encode())
        with open(path, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def up_to_date(extra: list[str] | None = None) -> bool:
    if not (os.path.exists(LIB) and os.path.exists(STAMP)):
        return False
    with open(STAMP) as fh:
        return fh.read().strip() == source_hash(extra)


def build(force: bool = False, verbose: bool = False, extra: list[str] | None = None) -> str:
    if not force and up_to_date(extra):
        return LIB
    with open(LIB + ".lock", "w") as lock:          # one builder at a time (several ranks may import at once)
        fcntl.flock(lock, fcntl.LOCK_EX)
        if force or not up_to_date(extra):
            tmp = LIB + f".tmp{os.getpid()}"
            cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + (extra or []) + ["-o", tmp] + sources()
            subprocess.run(cmd, check=True)
            os.replace(tmp, LIB)
            with open(STAMP, "w") as fh:
                fh.write(source_hash(extra) + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
