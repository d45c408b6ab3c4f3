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
SPIN_LIB = os.path.join(HERE, "libtangram_spin.so")     # debug build: bounded device spin loops (tangram_internal.h)
SPIN_LIMIT_DEFAULT = 4_000_000                           # polls; a few seconds of spinning on B200
SOURCES = [os.path.join(CSRC, "tangram_decode.cu"), os.path.join(CSRC, "tangram_compact.cu"),
           os.path.join(CSRC, "tangram_host.cpp")]
HEADERS = [os.path.join(ROOT, "include", "tangram.h"), os.path.join(CSRC, "tangram_internal.h")]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def stale(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(f) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False, spin_limit: int = 0) -> str:
    """spin_limit = 0: libtangram.so, the product.  spin_limit = N > 0: libtangram_spin.so, the same sources with
    -DTANGRAM_SPIN_LIMIT=N (every cross-CTA spin loop traps after N polls); load it with TANGRAM_LIB=<path>."""
    lib = SPIN_LIB if spin_limit > 0 else LIB
    if not force and not stale(lib):
        return lib
    cmd = [nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
           "-Xcompiler", "-fPIC,-ffp-contract=off,-fopenmp", "-Xptxas", "-v" if verbose else "-O3",
           "-shared", "-lgomp", "-o", lib, "-I", os.path.join(ROOT, "include"), "-I", CSRC] + SOURCES
    if spin_limit > 0:
        cmd.insert(1, f"-DTANGRAM_SPIN_LIMIT={int(spin_limit)}")
    if verbose:
        print(" ".join(cmd))
    subprocess.check_call(cmd)
    return lib


if __name__ == "__main__":
    n = int(sys.argv[sys.argv.index("--spin-limit") + 1]) if "--spin-limit" in sys.argv else 0
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, spin_limit=n))
