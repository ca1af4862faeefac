"""In-tree build of libfitrig.so (hand-written CUDA for sm_100a + the C-ABI of include/fitrig.h).

    python -m paper_2509_21754_b200.build [--force]

nvcc cross-compiles without a GPU.  The library links cudart statically and resolves the one driver
symbol it needs (cuTensorMapEncodeTiled) at run time, so it loads on a machine without a CUDA driver
(the CPU test tier checks its exported symbols there).
"""
from __future__ import annotations

import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libfitrig.so")
SOURCES = [os.path.join(CSRC, "fitrig.cu"), os.path.join(CSRC, "plan.cpp")]
DEPS = SOURCES + [os.path.join(CSRC, "kernels.cuh"), os.path.join(CSRC, "plan.h"),
                  os.path.join(ROOT, "include", "fitrig.h")]

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared",
    "-I" + os.path.join(ROOT, "include"), "-I" + CSRC,
]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


STAMP = LIB + ".srchash"  # hash of the sources the library was built from (file times do not survive a copy)


def source_hash() -> str:
    import hashlib
    h = hashlib.sha256()
    for d in DEPS:
        with open(d, "rb") as f:
            h.update(f.read())
    h.update(" ".join(NVCC_FLAGS).replace(ROOT, ".").encode())  # (the checkout's path is not part of the build)
    return h.hexdigest()


def stale() -> bool:
    if not os.path.exists(LIB) or not os.path.exists(STAMP):
        return True
    with open(STAMP) as f:
        return f.read().strip() != source_hash()


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = [nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
        subprocess.run(cmd, check=True)
        os.replace(tmp, LIB)
        with open(STAMP, "w") as f:
            f.write(source_hash() + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
