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


def _compile_and_link(lib: str, tag: str, extra: list, verbose: bool = False) -> None:
    """One object per source, compiled in parallel (only the stale ones), then one link.  Objects live in build/<tag>/
    (git-ignored)."""
    from concurrent.futures import ThreadPoolExecutor

    nvcc = os.environ.get("NVCC", "nvcc")
    objdir = os.path.join(HERE, "build", tag)
    os.makedirs(objdir, exist_ok=True)
    hdr_t = max(os.path.getmtime(os.path.join(CSRC, f)) for f in HEADERS)
    compile_flags = [f for f in NVCC_FLAGS if f not in ("-shared", "-lgomp")]
    i = compile_flags.index("-cudart")
    del compile_flags[i:i + 2]

    def one(src: str) -> str:
        obj = os.path.join(objdir, os.path.splitext(src)[0] + ".o")
        path = os.path.join(CSRC, src)
        if not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(path), hdr_t):
            subprocess.check_call([nvcc] + compile_flags + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, path])
        return obj

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(one, SOURCES))
    subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static", "-Xcompiler", "-fPIC,-fopenmp",
                           "-lgomp", "-o", lib] + objs)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or _stale():
        _compile_and_link(LIB, "release", [], verbose)
    return LIB


def build_debug(force: bool = False) -> str:
    """libblest_debug.so: the same sources with -DBLEST_DEBUG (device-side bounds asserts on every index)."""
    if force or _stale(LIB_DEBUG):
        _compile_and_link(LIB_DEBUG, "debug", ["-DBLEST_DEBUG"])
    return LIB_DEBUG


if __name__ == "__main__":
    if "--debug" in sys.argv:
        print(build_debug(force="--force" in sys.argv))
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
