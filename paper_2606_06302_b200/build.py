"""Builds libtangram.so (host planners + CUDA kernels, C ABI of include/tangram.h) in-tree with nvcc
for sm_100a.  `python -m paper_2606_06302_b200.build` or build() from __graft_entry__."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtangram.so")
SOURCES = [os.path.join(CSRC, "tangram_decode.cu"), os.path.join(CSRC, "tangram_compact.cu"),
           os.path.join(CSRC, "tangram_host.cpp")]
HEADERS = [os.path.join(ROOT, "include", "tangram.h"), os.path.join(CSRC, "tangram_internal.h")]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    cmd = [nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
           "-Xcompiler", "-fPIC,-ffp-contract=off,-fopenmp", "-Xptxas", "-v" if verbose else "-O3",
           "-shared", "-lgomp", "-o", LIB, "-I", os.path.join(ROOT, "include"), "-I", CSRC] + SOURCES
    if verbose:
        print(" ".join(cmd))
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose="-v" in sys.argv)
    print(LIB)
