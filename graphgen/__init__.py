"""Seeded synthetic graph generators shared by the oracle's tests and the CUDA path's tests/bench.

Input plumbing only -- none of the method's arithmetic lives here (no BFS, no BVSS, no bitmaps).
Every generator returns a *symmetric, sorted, loop-free, duplicate-free uint32 CSR* ``(n, rowptr,
colidx)`` as numpy arrays, the input format of BASELINE.json's configs.  The heavy lifting is in
``gen.cpp`` (OpenMP, counter-based hash => output independent of the thread count); the tiny
closed-form graphs used by the pins (path, cycle, star, ...) are assembled here with numpy.

The recipe for each BASELINE.json config (sizes, seeds, distributions) is ``CONFIGS`` below and is
restated in DESIGN.md "Input recipe".
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen.cpp")
_LIB = os.path.join(_HERE, "libgraphgen.so")
_lib = None

# Seeds fixed once: graph seed S_i = 260605081 + 10*i, sources S_i + 1, relabel S_i + 2.
BASE_SEED = 260605081
RMAT_ABC = (0.57, 0.19, 0.19)


def build(force: bool = False) -> str:
    """Compile gen.cpp -> libgraphgen.so (g++ -O3 -fopenmp) when missing or stale."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["g++", "-O3", "-march=x86-64-v2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC]
        )
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        u32p, u64, dbl = ctypes.POINTER(ctypes.c_uint32), ctypes.c_uint64, ctypes.c_double
        L.gg_rmat_edges.argtypes = [ctypes.c_int, u64, u64, dbl, dbl, dbl, u32p, u32p, u32p]
        L.gg_rmat_edges.restype = None
        L.gg_random_perm.argtypes = [ctypes.c_uint32, u64, u32p]
        L.gg_random_perm.restype = None
        L.gg_grid_edges.argtypes = [ctypes.c_uint32, ctypes.c_uint32, dbl, u64, u32p, u32p]
        L.gg_grid_edges.restype = u64
        L.gg_gnm_edges.argtypes = [ctypes.c_uint32, u64, u64, u32p, u32p]
        L.gg_gnm_edges.restype = None
        L.gg_edges_to_csr.argtypes = [ctypes.c_uint32, u64, u32p, u32p, u32p, u32p]
        L.gg_edges_to_csr.restype = u64
        L.gg_num_threads.restype = ctypes.c_int
        _lib = L
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_uint32))


def from_edges(n: int, src, dst):
    """Symmetric CSR from an arbitrary edge list (loops dropped, reverse edges added, deduplicated)."""
    L = _load()
    src = np.ascontiguousarray(src, dtype=np.uint32)
    dst = np.ascontiguousarray(dst, dtype=np.uint32)
    assert src.shape == dst.shape and src.ndim == 1
    if src.size and (int(src.max()) >= n or int(dst.max()) >= n):
        raise ValueError("endpoint out of range")
    m = int(src.size)
    rowptr = np.zeros(n + 1, dtype=np.uint32)
    colidx = np.empty(max(2 * m, 1), dtype=np.uint32)
    nnz = L.gg_edges_to_csr(n, m, _p(src), _p(dst), _p(rowptr), _p(colidx))
    if nnz == 2**64 - 1:
        raise OverflowError("nnz does not fit uint32")
    return n, rowptr, colidx[: int(nnz)]


def from_directed_edges(n: int, src, dst):
    """DIRECTED CSR from an edge list src -> dst: row u = sorted out-neighbours of u, loops dropped, duplicates merged.
    (numpy; the directed test graphs are small.)"""
    src = np.asarray(src, dtype=np.int64)
    dst = np.asarray(dst, dtype=np.int64)
    keep = src != dst
    key = np.unique(src[keep] * n + dst[keep])
    rows = key // n
    rowptr = np.zeros(n + 1, dtype=np.int64)
    np.add.at(rowptr, rows + 1, 1)
    return n, np.cumsum(rowptr).astype(np.uint32), (key % n).astype(np.uint32)


def rmat_directed(scale: int, edge_factor: int, seed: int, abc=RMAT_ABC):
    """The RMAT draws of `rmat` kept as DIRECTED edges (not symmetrised): GAP-twitter / GAP-web are directed."""
    L = _load()
    n = 1 << scale
    m = edge_factor << scale
    src = np.empty(m, dtype=np.uint32)
    dst = np.empty(m, dtype=np.uint32)
    perm = np.empty(n, dtype=np.uint32)
    L.gg_random_perm(n, seed + 2, _p(perm))
    L.gg_rmat_edges(scale, m, seed, abc[0], abc[1], abc[2], _p(perm), _p(src), _p(dst))
    return from_directed_edges(n, src, dst)


def rmat(scale: int, edge_factor: int, seed: int, abc=RMAT_ABC, relabel: bool = True):
    """Graph500-style RMAT: edge_factor * 2**scale draws, then (optionally) a seeded random relabelling
    of the vertex ids so that the natural order is not accidentally degree-sorted."""
    L = _load()
    n = 1 << scale
    m = edge_factor << scale
    src = np.empty(m, dtype=np.uint32)
    dst = np.empty(m, dtype=np.uint32)
    perm = None
    if relabel:
        perm = np.empty(n, dtype=np.uint32)
        L.gg_random_perm(n, seed + 2, _p(perm))
    L.gg_rmat_edges(scale, m, seed, abc[0], abc[1], abc[2], _p(perm) if relabel else None, _p(src), _p(dst))
    return from_edges(n, src, dst)


def grid2d(rows: int, cols: int, delete_frac: float = 0.0, seed: int = 0):
    """rows x cols 4-connected lattice, id = r*cols + c; every lattice edge is deleted independently
    with probability delete_frac (Bernoulli per edge, seeded)."""
    L = _load()
    cap = rows * (cols - 1) + (rows - 1) * cols
    src = np.empty(max(cap, 1), dtype=np.uint32)
    dst = np.empty(max(cap, 1), dtype=np.uint32)
    kept = int(L.gg_grid_edges(rows, cols, float(delete_frac), seed, _p(src), _p(dst)))
    return from_edges(rows * cols, src[:kept], dst[:kept])


def gnm(n: int, m: int, seed: int):
    """Uniform random multigraph G(n, m) with i.i.d. endpoints, then symmetrised and deduplicated."""
    L = _load()
    src = np.empty(m, dtype=np.uint32)
    dst = np.empty(m, dtype=np.uint32)
    L.gg_gnm_edges(n, m, seed, _p(src), _p(dst))
    return from_edges(n, src, dst)


# ---- small closed-form graphs (pins) -------------------------------------------------------------
def path(n: int):
    i = np.arange(max(n - 1, 0), dtype=np.uint32)
    return from_edges(n, i, i + 1)


def cycle(n: int):
    i = np.arange(n, dtype=np.uint32)
    return from_edges(n, i, (i + 1) % n)


def star(n: int, centre: int = 0):
    leaves = np.array([v for v in range(n) if v != centre], dtype=np.uint32)
    return from_edges(n, np.full(leaves.size, centre, dtype=np.uint32), leaves)


def complete(n: int):
    u, v = np.triu_indices(n, k=1)
    return from_edges(n, u.astype(np.uint32), v.astype(np.uint32))


def binary_tree(n: int):
    """Complete binary tree in heap order: parent(i) = (i-1)//2."""
    i = np.arange(1, n, dtype=np.uint32)
    return from_edges(n, (i - 1) // 2, i)


def empty(n: int):
    return from_edges(n, np.empty(0, np.uint32), np.empty(0, np.uint32))


def disjoint_union(*graphs):
    """Vertex-disjoint union; ids of graph k are shifted by the sizes of graphs 0..k-1."""
    n_tot, rps, cis, off_v, off_e = 0, [np.zeros(1, np.uint32)], [], 0, 0
    for n, rp, ci in graphs:
        rps.append(rp[1:].astype(np.uint64) + off_e)
        cis.append(ci.astype(np.uint64) + off_v)
        off_v += n
        off_e += int(rp[-1])
        n_tot += n
    rowptr = np.concatenate(rps).astype(np.uint32)
    colidx = np.concatenate(cis).astype(np.uint32) if cis else np.empty(0, np.uint32)
    return n_tot, rowptr, colidx


def random_graph(n: int, m: int, seed: int):
    """Small G(n,m) used by the brute-force pins (same generator as config 3)."""
    return gnm(n, m, seed) if m > 0 else empty(n)


def degrees(rowptr: np.ndarray) -> np.ndarray:
    return np.diff(rowptr.astype(np.int64))


def pick_sources(rowptr: np.ndarray, k: int, seed: int, nonzero_degree: bool = True) -> np.ndarray:
    """k distinct seeded sources, optionally restricted to vertices of non-zero degree."""
    deg = degrees(rowptr)
    cand = np.flatnonzero(deg > 0) if nonzero_degree else np.arange(deg.size)
    rng = np.random.Generator(np.random.PCG64(seed))
    k = min(k, cand.size)
    return np.sort(rng.choice(cand, size=k, replace=False)).astype(np.uint32)


def num_threads() -> int:
    return int(_load().gg_num_threads())


# ---- BASELINE.json configs -----------------------------------------------------------------------
CONFIGS = {
    # name: (description, builder, n_sources)
    "c1_rmat16": dict(kind="rmat", scale=16, edge_factor=16, seed=BASE_SEED + 10, n_sources=64),
    "c2_grid4096": dict(kind="grid", rows=4096, cols=4096, delete_frac=0.05, seed=BASE_SEED + 20, n_sources=16),
    "c3_gnm25": dict(kind="gnm", n=1 << 25, m=1 << 27, seed=BASE_SEED + 30, n_sources=16),
    "c4_rmat24": dict(kind="rmat", scale=24, edge_factor=32, seed=BASE_SEED + 40, n_sources=64),
    "c5_rmat18": dict(kind="rmat", scale=18, edge_factor=16, seed=BASE_SEED + 50, n_sources=0),
}


def make_config(name: str, shrink: int = 0):
    """Build the CSR of a BASELINE.json config.  ``shrink`` halves the linear size that many times
    (RMAT scale - shrink, grid side >> shrink, G(n,m) n and m >> shrink) for CPU-sized test cases."""
    c = CONFIGS[name]
    if c["kind"] == "rmat":
        return rmat(c["scale"] - shrink, c["edge_factor"], c["seed"])
    if c["kind"] == "grid":
        return grid2d(c["rows"] >> shrink, c["cols"] >> shrink, c["delete_frac"], c["seed"])
    if c["kind"] == "gnm":
        return gnm(c["n"] >> shrink, c["m"] >> shrink, c["seed"])
    raise KeyError(name)


def config_sources(name: str, rowptr: np.ndarray, replica: int = 0) -> np.ndarray:
    """The config's seeded sources.  replica > 0: another draw of the same size from the same population (seed
    S_i + 1 + 1000 * replica) -- the disjoint per-rank work of a multi-GPU weak-scaling run."""
    c = CONFIGS[name]
    k = c["n_sources"]
    srcs = pick_sources(rowptr, k, c["seed"] + 1 + 1000 * replica, nonzero_degree=True) if k else np.empty(0, np.uint32)
    if c["kind"] == "grid":  # corner vertex first (BASELINE.json config 2)
        srcs = np.concatenate([np.zeros(1, np.uint32), srcs])
    return srcs
