"""Thin ctypes binding over the C ABI of ``include/blest.h`` -- argument marshalling only.

Every step of the path (init, contraction, lazy/eager updates, switching, multi-source, closeness) runs in the
CUDA kernels of ``libblest.so``; nothing here computes.  There is NO CPU fallback: if the library cannot be
loaded, or no sm_100 device is present, calls raise.  Outputs may be torch CUDA tensors (their ``data_ptr()`` is
passed) or numpy arrays (host pointers; the library copies device->host on the stream).
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import numpy as np

from . import build as _build

_LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libblest.so")
_lib = None

# status codes (include/blest.h)
OK, EINVAL, ERANGE, EUNSORTED, ENOTSYM, ENOMEM, ECUDA, EUNSUPPORTED, EOVERFLOW = 0, -1, -2, -3, -4, -5, -6, -7, -8

# option values
REORDER = {"none": 0, "rcm": 1, "degree": 2, "jaccard": 3}
KERNEL = {"auto": 0, "eager": 1, "lazy": 2}
SWITCHING = {"auto": 0, "off": 1, "bottom_up": 2, "top_down": 3, "slice": 4, "scripted": 5}
CONTRACTION = {"auto": 0, "alu": 1, "mma_b1": 2, "mma_u8": 3}


class BlestError(RuntimeError):
    def __init__(self, status: int, what: str):
        self.status = status
        super().__init__(f"{what}: {status} ({strerror(status)})")


class _Csr(ctypes.Structure):
    _fields_ = [("n", ctypes.c_uint32), ("nnz", ctypes.c_uint64), ("rowptr", ctypes.c_void_p),
                ("colidx", ctypes.c_void_p), ("on_device", ctypes.c_int), ("directed", ctypes.c_int)]


class _Options(ctypes.Structure):
    _fields_ = [("reorder", ctypes.c_int), ("builder", ctypes.c_int), ("validate", ctypes.c_int),
                ("kernel", ctypes.c_int), ("switching", ctypes.c_int), ("contraction", ctypes.c_int),
                ("kappa", ctypes.c_int), ("trace", ctypes.c_int), ("eta", ctypes.c_float), ("gamma", ctypes.c_float),
                ("persist_l2", ctypes.c_int), ("prune_components", ctypes.c_int), ("queue_capacity", ctypes.c_uint32),
                ("tune", ctypes.c_int * 4), ("reserved", ctypes.c_int * 6)]


class _Info(ctypes.Structure):
    _fields_ = [("n", ctypes.c_uint32), ("nnz", ctypes.c_uint64), ("n_slice_sets", ctypes.c_uint32),
                ("n_vss", ctypes.c_uint32), ("n_slices", ctypes.c_uint64), ("n_quads", ctypes.c_uint64),
                ("bvss_bytes", ctypes.c_uint64), ("csr_bytes", ctypes.c_uint64), ("workspace_bytes", ctypes.c_uint64),
                ("mask_density", ctypes.c_double), ("u_div", ctypes.c_double), ("reorder_seconds", ctypes.c_double),
                ("build_seconds", ctypes.c_double), ("upload_seconds", ctypes.c_double),
                ("component_seconds", ctypes.c_double), ("kernel_chosen", ctypes.c_int), ("reorder", ctypes.c_int), ("kappa", ctypes.c_int),
                ("num_sms", ctypes.c_int), ("grid_blocks", ctypes.c_int), ("block_threads", ctypes.c_int),
                ("queue_capacity", ctypes.c_uint32), ("n_sweep_words", ctypes.c_uint32)]


class _Trace(ctypes.Structure):
    _fields_ = [("level", ctypes.c_uint32), ("mode", ctypes.c_uint32), ("q_entries", ctypes.c_uint32),
                ("new_vertices", ctypes.c_uint32), ("q_bytes", ctypes.c_uint64), ("bu_scanned", ctypes.c_uint64),
                ("unvisited", ctypes.c_uint32), ("reserved", ctypes.c_uint32), ("t_ns", ctypes.c_uint64),
                ("t_stage1_ns", ctypes.c_uint64)]


TRACE_DTYPE = np.dtype([("level", "<u4"), ("mode", "<u4"), ("q_entries", "<u4"), ("new_vertices", "<u4"),
                        ("q_bytes", "<u8"), ("bu_scanned", "<u8"), ("unvisited", "<u4"), ("reserved", "<u4"),
                        ("t_ns", "<u8"), ("t_stage1_ns", "<u8")])

EXPORTS = ["blest_build", "blest_preprocess_host", "blest_configure", "blest_get_call_stats", "blest_bfs", "blest_msbfs", "blest_closeness", "blest_farness",
           "blest_get_info", "blest_last_status", "blest_farness_partial", "blest_closeness_from_sums", "blest_get_ms_stats", "blest_get_ms_phases", "blest_get_ms_level_trace",
           "blest_l2_microbench", "blest_tcgen05_microbench", "blest_closeness_noalloc", "blest_noalloc_limits", "blest_get_trace", "blest_get_array", "blest_get_vi", "blest_contraction_selftest",
           "blest_mma_microbench", "blest_barrier_microbench", "blest_cluster_microbench", "blest_destroy", "blest_strerror",
           "blest_last_cuda_error"]


def load(build_if_missing: bool = True):
    """dlopen libblest.so (building it with nvcc first when it is missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _LIB_PATH
    if os.environ.get("BLEST_DEBUG_LIB") == "1":  # the bounds-asserting build (tests; python -m ...build --debug)
        path = _build.build_debug() if build_if_missing else _build.LIB_DEBUG
    elif build_if_missing:
        _build.build()
    if not os.path.exists(path):
        raise ImportError(f"{path} is missing: run `python -m paper_2606_05081_b200.build` (no CPU fallback exists)")
    L = ctypes.CDLL(path)
    vp, u32, u64, i32 = ctypes.c_void_p, ctypes.c_uint32, ctypes.c_uint64, ctypes.c_int
    L.blest_build.argtypes = [ctypes.POINTER(_Csr), ctypes.POINTER(_Options), ctypes.POINTER(vp)]
    L.blest_preprocess_host.argtypes = [ctypes.POINTER(_Csr), ctypes.POINTER(_Options), ctypes.POINTER(vp)]
    L.blest_configure.argtypes = [vp, ctypes.POINTER(_Options)]
    L.blest_bfs.argtypes = [vp, u32, vp, vp]
    L.blest_msbfs.argtypes = [vp, vp, u32, vp, vp]
    L.blest_closeness.argtypes = [vp, vp, u64, vp, vp]
    L.blest_farness.argtypes = [vp, vp, u64, vp, vp, vp]
    L.blest_get_info.argtypes = [vp, ctypes.POINTER(_Info)]
    L.blest_last_status.argtypes = [vp]
    L.blest_farness_partial.argtypes = [vp, u32, u32, vp, vp, vp]
    L.blest_closeness_from_sums.argtypes = [vp, vp, u64, vp, vp]
    L.blest_get_ms_stats.argtypes = [vp, ctypes.POINTER(u64)]
    L.blest_get_ms_phases.argtypes = [vp, ctypes.POINTER(u64)]
    L.blest_get_ms_level_trace.argtypes = [vp, ctypes.POINTER(u64), ctypes.c_uint32, ctypes.POINTER(ctypes.c_uint32)]
    L.blest_closeness_noalloc.argtypes = [vp, vp, u32, vp, vp]
    L.blest_noalloc_limits.argtypes = [ctypes.POINTER(u32), ctypes.POINTER(u64), ctypes.POINTER(u64)]
    L.blest_l2_microbench.argtypes = [u64, u32, ctypes.POINTER(ctypes.c_double)]
    L.blest_tcgen05_microbench.argtypes = [u32, u32, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(u64)]
    L.blest_get_trace.argtypes = [vp, vp, u32, ctypes.POINTER(u32)]
    L.blest_get_call_stats.argtypes = [vp, ctypes.POINTER(u64), ctypes.POINTER(u64)]
    L.blest_get_array.argtypes = [vp, i32, vp, u64]
    L.blest_get_vi.argtypes = [u64, u64]
    L.blest_get_vi.restype = u64
    L.blest_contraction_selftest.argtypes = [i32, ctypes.POINTER(u64)]
    L.blest_mma_microbench.argtypes = [i32, u32, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    L.blest_barrier_microbench.argtypes = [u32, ctypes.POINTER(ctypes.c_double)]
    L.blest_cluster_microbench.argtypes = [ctypes.c_int, u32, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    L.blest_destroy.argtypes = [vp]
    L.blest_destroy.restype = None
    L.blest_strerror.argtypes = [i32]
    L.blest_strerror.restype = ctypes.c_char_p
    L.blest_last_cuda_error.restype = i32
    _lib = L
    return L


def strerror(status: int) -> str:
    return load().blest_strerror(int(status)).decode()


def _check(status: int, what: str):
    if status != OK:
        raise BlestError(status, what)


def _ptr(x):
    """Device or host pointer of a torch tensor / numpy array (None -> NULL)."""
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        if not x.flags["C_CONTIGUOUS"]:
            raise ValueError("output arrays must be C-contiguous")
        return ctypes.c_void_p(x.ctypes.data)
    if hasattr(x, "data_ptr"):
        if not x.is_contiguous():
            raise ValueError("output tensors must be contiguous")
        return ctypes.c_void_p(x.data_ptr())
    raise TypeError(type(x))


def _stream(stream):
    if stream is None:
        return None
    return ctypes.c_void_p(int(getattr(stream, "cuda_stream", stream)))


def _options(reorder="none", builder=0, validate=False, kernel="auto", switching="auto", contraction="auto", kappa=64,
             trace=True, eta=0.0, gamma=0.0, bu_mask=0, costs=None, persist_l2=True, prune_components=True,
             queue_capacity=0, tma_tiles=False, ms_pull=True, level_guess=True, ms_lanes=0) -> _Options:
    o = _Options()
    o.reorder = REORDER[reorder] if isinstance(reorder, str) else int(reorder)
    o.builder = int(builder)
    o.validate = int(bool(validate))
    o.kernel = KERNEL[kernel] if isinstance(kernel, str) else int(kernel)
    o.switching = SWITCHING[switching] if isinstance(switching, str) else int(switching)
    o.contraction = CONTRACTION[contraction] if isinstance(contraction, str) else int(contraction)
    o.kappa = int(kappa)
    o.trace = 1 if trace else 2
    o.eta = float(eta)
    o.gamma = float(gamma)
    o.persist_l2 = 0 if persist_l2 else 1
    o.prune_components = 0 if prune_components else 1
    o.queue_capacity = int(queue_capacity)
    o.tune[0] = int(bool(tma_tiles))
    o.tune[1] = 0 if ms_pull else 1
    o.tune[2] = 0 if level_guess else 1
    o.tune[3] = int(ms_lanes)
    o.reserved[0] = int(bu_mask)
    for k, c in enumerate(costs or ()):  # switch cost model overrides, ps per unit (tuning only): td_edge, td_vertex,
        o.reserved[1 + k] = int(round(100 * float(c)))  # bu_vertex, bu_scan, bu_word
    return o


@dataclass
class Info:
    n: int; nnz: int; n_slice_sets: int; n_vss: int; n_slices: int; n_quads: int
    bvss_bytes: int; csr_bytes: int; workspace_bytes: int; mask_density: float; u_div: float
    reorder_seconds: float; build_seconds: float; upload_seconds: float; component_seconds: float
    kernel_chosen: int; reorder: int; kappa: int; num_sms: int; grid_blocks: int; block_threads: int
    queue_capacity: int; n_sweep_words: int


class Graph:
    """Owns one ``blest_handle_t``.  ``Graph(n, rowptr, colidx, reorder=..., ...)`` calls ``blest_build``."""

    def __init__(self, n: int, rowptr, colidx, host_only: bool = False, directed: bool = False, **opts):
        L = load()
        self._h = ctypes.c_void_p()
        on_device = hasattr(rowptr, "data_ptr")
        if on_device:
            rp, ci = rowptr, colidx
            nnz = int(colidx.numel())
        else:
            rp = np.ascontiguousarray(rowptr, dtype=np.uint32)
            ci = np.ascontiguousarray(colidx, dtype=np.uint32)
            nnz = int(ci.size)
        self._keep = (rp, ci)
        csr = _Csr(int(n), nnz, _ptr(rp), _ptr(ci) if nnz else None, int(on_device), int(bool(directed)))
        self._opts = dict(opts)
        o = _options(**opts)
        fn = L.blest_preprocess_host if host_only else L.blest_build
        _check(fn(ctypes.byref(csr), ctypes.byref(o), ctypes.byref(self._h)), "blest_preprocess_host" if host_only else "blest_build")
        self._keep = None
        self.n = int(n)

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            load().blest_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # -- options
    def configure(self, **opts):
        self._opts.update(opts)
        o = _options(**self._opts)
        _check(load().blest_configure(self._h, ctypes.byref(o)), "blest_configure")

    # -- traversal
    def bfs(self, src: int, levels_out, stream=None):
        """blest_bfs: levels_out int32[n] (torch CUDA tensor or numpy array), returned for convenience."""
        _check(load().blest_bfs(self._h, int(src), _ptr(levels_out), _stream(stream)), "blest_bfs")
        return levels_out

    def msbfs(self, srcs, levels_out, stream=None):
        srcs = np.ascontiguousarray(srcs, dtype=np.uint32)
        _check(load().blest_msbfs(self._h, _ptr(srcs), int(srcs.size), _ptr(levels_out), _stream(stream)), "blest_msbfs")
        return levels_out

    def closeness(self, out, srcs=None, stream=None):
        if srcs is None:
            sp, k = None, self.n
        else:
            srcs = np.ascontiguousarray(srcs, dtype=np.uint32)
            sp, k = _ptr(srcs), int(srcs.size)
        _check(load().blest_closeness(self._h, sp, k, _ptr(out), _stream(stream)), "blest_closeness")
        return out

    def farness(self, far_out=None, reach_out=None, srcs=None, stream=None):
        if srcs is None:
            sp, k = None, self.n
        else:
            srcs = np.ascontiguousarray(srcs, dtype=np.uint32)
            sp, k = _ptr(srcs), int(srcs.size)
        _check(load().blest_farness(self._h, sp, k, _ptr(far_out), _ptr(reach_out), _stream(stream)), "blest_farness")
        return far_out, reach_out

    def farness_partial(self, first: int, count: int, far_sum, reach_sum, stream=None):
        """blest_farness_partial: target-side sums over sources [first, first+count) (device tensors, original ids)."""
        _check(load().blest_farness_partial(self._h, int(first), int(count), _ptr(far_sum), _ptr(reach_sum), _stream(stream)),
               "blest_farness_partial")
        return far_sum, reach_sum

    def closeness_noalloc(self, out, srcs_dev, stream=None):
        """blest_closeness_noalloc: srcs_dev a CUDA uint32/int32 tensor, out a CUDA float64 tensor; allocates nothing."""
        k = int(srcs_dev.numel()) if hasattr(srcs_dev, "numel") else int(srcs_dev.size)
        _check(load().blest_closeness_noalloc(self._h, _ptr(srcs_dev), k, _ptr(out), _stream(stream)), "blest_closeness_noalloc")
        return out

    def ms_stats(self) -> dict:
        """Totals of the last multi-source launch (blest_get_ms_stats)."""
        buf = (ctypes.c_uint64 * 8)()
        _check(load().blest_get_ms_stats(self._h, buf), "blest_get_ms_stats")
        keys = ("entries", "quads", "probes", "fresh", "dirty_sets", "levels", "batches", "pull_neighbours")
        return {k: int(buf[i]) for i, k in enumerate(keys)}

    def ms_phases(self) -> dict:
        """Nanoseconds CTA 0 spent per phase of the last multi-source launch (blest_get_ms_phases)."""
        buf = (ctypes.c_uint64 * 8)()
        _check(load().blest_get_ms_phases(self._h, buf), "blest_get_ms_phases")
        keys = ("init_ns", "stage1_ns", "barrier1_ns", "stage2_ns", "barrier2_ns", "pull_rows", "pull_levels")
        return {k: int(buf[i]) for i, k in enumerate(keys)}

    def ms_level_trace(self, max_levels: int = 60) -> list:
        """Per-level records of the first levels of the last multi-source launch (blest_get_ms_level_trace)."""
        buf = (ctypes.c_uint64 * (4 * max_levels))()
        k = ctypes.c_uint32(0)
        _check(load().blest_get_ms_level_trace(self._h, buf, max_levels, ctypes.byref(k)), "blest_get_ms_level_trace")
        return [{"level": int((buf[4 * i] >> 32) & 0x7FFFFFFF), "pull": bool(buf[4 * i] >> 63),
                 "entries": int(buf[4 * i] & 0xFFFFFFFF), "stage1_ns": int(buf[4 * i + 1]),
                 "stage2_ns": int(buf[4 * i + 2]), "enqueued": int(buf[4 * i + 3])} for i in range(k.value)]

    # -- introspection
    def info(self) -> Info:
        i = _Info()
        _check(load().blest_get_info(self._h, ctypes.byref(i)), "blest_get_info")
        return Info(**{f[0]: getattr(i, f[0]) for f in _Info._fields_})

    def last_status(self) -> int:
        """blest_last_status: synchronises, returns and clears the handle's deferred status (OK or EOVERFLOW)."""
        return int(load().blest_last_status(self._h))

    def call_stats(self):
        """(init_ns, levels_ns) of the last bfs call on the lazy kernel."""
        a, b = ctypes.c_uint64(0), ctypes.c_uint64(0)
        _check(load().blest_get_call_stats(self._h, ctypes.byref(a), ctypes.byref(b)), "blest_get_call_stats")
        return int(a.value), int(b.value)

    def trace(self) -> np.ndarray:
        """Per-level records of the last bfs() call (structured array, TRACE_DTYPE).  Synchronises the device."""
        n = ctypes.c_uint32(0)
        _check(load().blest_get_trace(self._h, None, 0, ctypes.byref(n)), "blest_get_trace")
        buf = np.zeros(n.value, dtype=TRACE_DTYPE)
        if n.value:
            _check(load().blest_get_trace(self._h, ctypes.c_void_p(buf.ctypes.data), n.value, ctypes.byref(n)), "blest_get_trace")
        return buf

    _ARRAYS = {"setPtr": 0, "rowIds": 1, "masks": 2, "realPtrs": 3, "virtualToReal": 4, "perm": 5, "iperm": 6,
               "rowptr": 7, "colidx": 8}

    def array(self, name: str) -> np.ndarray:
        i = self.info()
        sizes = {"setPtr": i.n_slice_sets + 1, "rowIds": 4 * i.n_quads, "masks": i.n_quads,
                 "realPtrs": i.n_slice_sets + 1, "virtualToReal": i.n_vss, "perm": i.n, "iperm": i.n,
                 "rowptr": i.n + 1, "colidx": i.nnz}
        out = np.empty(sizes[name], dtype=np.uint32)
        _check(load().blest_get_array(self._h, self._ARRAYS[name], ctypes.c_void_p(out.ctypes.data), out.nbytes), "blest_get_array")
        return out


def get_vi(u: int, rho: int) -> int:
    return int(load().blest_get_vi(int(u), int(rho)))


def contraction_selftest(contraction) -> int:
    c = CONTRACTION[contraction] if isinstance(contraction, str) else int(contraction)
    n = ctypes.c_uint64(0)
    _check(load().blest_contraction_selftest(c, ctypes.byref(n)), "blest_contraction_selftest")
    return int(n.value)


def mma_microbench(kind, iters: int = 4096):
    k = CONTRACTION[kind] if isinstance(kind, str) else int(kind)
    t, ms = ctypes.c_double(0), ctypes.c_double(0)
    _check(load().blest_mma_microbench(k, iters, ctypes.byref(t), ctypes.byref(ms)), "blest_mma_microbench")
    return t.value, ms.value


def closeness_from_sums(far_sum, reach_sum, out, stream=None):
    n = int(out.numel()) if hasattr(out, "numel") else int(out.size)
    _check(load().blest_closeness_from_sums(_ptr(far_sum), _ptr(reach_sum), n, _ptr(out), _stream(stream)),
           "blest_closeness_from_sums")
    return out


def l2_microbench(nbytes: int = 48 << 20, iters: int = 50) -> float:
    """Read + write GB/s of an L2-resident copy in the persistent launch configuration."""
    g = ctypes.c_double(0)
    _check(load().blest_l2_microbench(int(nbytes), int(iters), ctypes.byref(g)), "blest_l2_microbench")
    return g.value


def tcgen05_microbench(iters: int = 2048, n: int = 256):
    """(tera byte-MACs/s, wrong accumulator elements) of tcgen05.mma kind::i8, M = 128, N = n, K = 32."""
    t, bad = ctypes.c_double(0), ctypes.c_uint64(0)
    _check(load().blest_tcgen05_microbench(int(iters), int(n), ctypes.byref(t), ctypes.byref(bad)), "blest_tcgen05_microbench")
    return t.value, int(bad.value)


def noalloc_limits():
    """(max sources per call, max bytes of one state array, max vertices at kappa = 64) of blest_closeness_noalloc."""
    a, b, c = ctypes.c_uint32(0), ctypes.c_uint64(0), ctypes.c_uint64(0)
    _check(load().blest_noalloc_limits(ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)), "blest_noalloc_limits")
    return int(a.value), int(b.value), int(c.value)


def cluster_microbench(cluster_ctas: int = 8, iters: int = 2000):
    """(ns per cluster barrier, ns per dependent distributed-shared-memory load) for one cluster of `cluster_ctas` CTAs."""
    a, b = ctypes.c_double(0.0), ctypes.c_double(0.0)
    _check(load().blest_cluster_microbench(int(cluster_ctas), iters, ctypes.byref(a), ctypes.byref(b)), "blest_cluster_microbench")
    return a.value, b.value


def barrier_microbench(iters: int = 2000) -> float:
    ns = ctypes.c_double(0)
    _check(load().blest_barrier_microbench(iters, ctypes.byref(ns)), "blest_barrier_microbench")
    return ns.value
