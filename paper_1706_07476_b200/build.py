"""Builds libmonteray.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1706_07476_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The shared object lands next to this file so that it
travels with the repo snapshot to the GPU box (it is git-ignored, not gpurun-ignored).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmonteray.so")
SOURCES = [os.path.join(CSRC, "monteray.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "mr_device.cuh"), os.path.join(CSRC, "mr_sort.cuh"), os.path.join(CSRC, "mr_defer.cuh"), os.path.join(CSRC, "mr_tiled.cuh"), os.path.join(CSRC, "mr_microbench.cuh"), os.path.join(ROOT, "include", "monteray.h")]

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-lineinfo",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-Xcompiler", "-fPIC,-fvisibility=hidden", "-shared",
    "--cudart", "static",
]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def up_to_date() -> bool:
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    return all(os.path.getmtime(d) <= t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and up_to_date():
        return LIB
    tmp = LIB + f".{os.getpid()}.tmp"
    cmd = [nvcc_path()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
    if verbose:
        print(" ".join(cmd), flush=True)
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
