"""CPU ORACLE -- TEST INFRASTRUCTURE ONLY (see bfs_oracle.c for the full header and citations).

Thin ctypes access to ``bfs_oracle.c`` (plain C, gcc): queue BFS -> int32 levels (-1 unreachable),
uint64 farness, uint32 reach, fp64 closeness.  Independent of the CUDA path: imports nothing from
``paper_2606_05081_b200`` and shares no code with it.  Only ``tests/``, ``__graft_entry__.smoke()``
and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bfs_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

_u32p = ctypes.POINTER(ctypes.c_uint32)
_i32p = ctypes.POINTER(ctypes.c_int32)
_u64p = ctypes.POINTER(ctypes.c_uint64)
_f64p = ctypes.POINTER(ctypes.c_double)


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp bfs_oracle.c -> liboracle.so (as it stands; never tuned)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC])
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        L.oracle_bfs.argtypes = [ctypes.c_uint32, _u32p, _u32p, ctypes.c_uint32, _i32p]
        L.oracle_bfs.restype = ctypes.c_int
        L.oracle_msbfs.argtypes = [ctypes.c_uint32, _u32p, _u32p, _u32p, ctypes.c_uint32, _i32p]
        L.oracle_msbfs.restype = ctypes.c_int
        L.oracle_farness.argtypes = [ctypes.c_uint32, _i32p, _u64p, _u32p]
        L.oracle_farness.restype = None
        L.oracle_closeness_value.argtypes = [ctypes.c_uint32, ctypes.c_uint64]
        L.oracle_closeness_value.restype = ctypes.c_double
        L.oracle_closeness.argtypes = [ctypes.c_uint32, _u32p, _u32p, _u32p, ctypes.c_uint64,
                                       _u64p, _u32p, _f64p, ctypes.c_int]
        L.oracle_closeness.restype = ctypes.c_int
        L.oracle_component_edges.argtypes = [ctypes.c_uint32, _u32p, _i32p]
        L.oracle_component_edges.restype = ctypes.c_uint64
        _lib = L
    return _lib


def _csr(rowptr, colidx):
    rowptr = np.ascontiguousarray(rowptr, dtype=np.uint32)
    colidx = np.ascontiguousarray(colidx, dtype=np.uint32)
    if colidx.size == 0:  # keep a valid pointer for empty graphs
        colidx = np.zeros(1, dtype=np.uint32)
    return rowptr, colidx


def bfs(n, rowptr, colidx, src) -> np.ndarray:
    """int32 levels from ``src`` (-1 = unreachable).  PAPER.md:38-44."""
    rowptr, colidx = _csr(rowptr, colidx)
    level = np.empty(n, dtype=np.int32)
    rc = _load().oracle_bfs(n, rowptr.ctypes.data_as(_u32p), colidx.ctypes.data_as(_u32p), int(src),
                            level.ctypes.data_as(_i32p))
    if rc:
        raise ValueError(f"oracle_bfs failed ({rc})")
    return level


def msbfs(n, rowptr, colidx, srcs) -> np.ndarray:
    """int32[k, n]: row b = levels from srcs[b].  PAPER.md:504."""
    rowptr, colidx = _csr(rowptr, colidx)
    srcs = np.ascontiguousarray(srcs, dtype=np.uint32)
    out = np.empty((srcs.size, n), dtype=np.int32)
    if srcs.size:
        rc = _load().oracle_msbfs(n, rowptr.ctypes.data_as(_u32p), colidx.ctypes.data_as(_u32p),
                                  srcs.ctypes.data_as(_u32p), srcs.size, out.ctypes.data_as(_i32p))
        if rc:
            raise ValueError(f"oracle_msbfs failed ({rc})")
    return out


def farness(level) -> tuple[int, int]:
    """(far, reach) of one level array.  PAPER.md Eq. 7."""
    level = np.ascontiguousarray(level, dtype=np.int32)
    far, reach = ctypes.c_uint64(0), ctypes.c_uint32(0)
    _load().oracle_farness(level.size, level.ctypes.data_as(_i32p), ctypes.byref(far), ctypes.byref(reach))
    return int(far.value), int(reach.value)


def closeness_value(reach: int, far: int) -> float:
    return float(_load().oracle_closeness_value(int(reach), int(far)))


def closeness(n, rowptr, colidx, srcs=None, nthreads: int = 0):
    """(far uint64[k], reach uint32[k], cc float64[k], threads_used).  srcs=None: every vertex."""
    rowptr, colidx = _csr(rowptr, colidx)
    if srcs is None:
        k, sp = n, None
    else:
        srcs = np.ascontiguousarray(srcs, dtype=np.uint32)
        k, sp = srcs.size, srcs.ctypes.data_as(_u32p)
    far = np.zeros(k, dtype=np.uint64)
    reach = np.zeros(k, dtype=np.uint32)
    cc = np.zeros(k, dtype=np.float64)
    used = 1
    if k:
        used = _load().oracle_closeness(n, rowptr.ctypes.data_as(_u32p), colidx.ctypes.data_as(_u32p), sp, k,
                                        far.ctypes.data_as(_u64p), reach.ctypes.data_as(_u32p),
                                        cc.ctypes.data_as(_f64p), int(nthreads))
        if used < 0:
            raise ValueError("oracle_closeness failed")
    return far, reach, cc, used


def component_edges(rowptr, level) -> int:
    """Undirected edges of the source's component (TEPS numerator, BASELINE.json)."""
    rowptr = np.ascontiguousarray(rowptr, dtype=np.uint32)
    level = np.ascontiguousarray(level, dtype=np.int32)
    return int(_load().oracle_component_edges(level.size, rowptr.ctypes.data_as(_u32p),
                                              level.ctypes.data_as(_i32p)))
