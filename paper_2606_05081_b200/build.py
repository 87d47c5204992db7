"""Compile the C-ABI library ``libblest.so`` in-tree with nvcc for sm_100a.

    python -m paper_2606_05081_b200.build [--force]

nvcc cross-compiles without a GPU; the .so is git-ignored but travels to the GPU box with the snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libblest.so")
SOURCES = ["api.cu", "bfs_lazy.cu", "bfs_eager.cu", "msbfs_kernels.cu", "microbench.cu", "host_graph.cpp"]
HEADERS = ["device_common.cuh", "bfs_kernels.cuh", "host_graph.h", os.path.join("..", "..", "include", "blest.h")]
NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC,-fopenmp,-O3", "-shared", "-cudart", "static", "-lgomp",
]


LIB_DEBUG = os.path.join(HERE, "libblest_debug.so")


def _stale(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or _stale():
        nvcc = os.environ.get("NVCC", "nvcc")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + [os.path.join(CSRC, f) for f in SOURCES]
        subprocess.check_call(cmd)
    return LIB


def build_debug(force: bool = False) -> str:
    """libblest_debug.so: the same sources with -DBLEST_DEBUG (device-side bounds asserts on every index)."""
    if force or _stale(LIB_DEBUG):
        nvcc = os.environ.get("NVCC", "nvcc")
        subprocess.check_call([nvcc] + NVCC_FLAGS + ["-DBLEST_DEBUG", "-o", LIB_DEBUG] + [os.path.join(CSRC, f) for f in SOURCES])
    return LIB_DEBUG


if __name__ == "__main__":
    if "--debug" in sys.argv:
        print(build_debug(force="--force" in sys.argv))
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
