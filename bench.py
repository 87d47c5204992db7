#!/usr/bin/env python
"""bench.py -- the measurement contract of this repo.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config c4_rmat24] [--shrink S]
                    [--no-parity] [--no-cpu-baseline] [--no-extra]

One "step" = one pass of the whole hot path (blest_bfs: init -> per-level contraction / switch -> lazy finalisation ->
hand-off, Alg. 2-4) over one batch of synthetic input = single-source BFS from each of the config's seeded
sources, on the resident graph.  The workload at N = 1 is BASELINE.json's headline config, configs[3] (RMAT scale 24,
edge factor 32, degree-sorted before the BVSS build, 64 sources): the config the GTEPS / HBM-roofline metric is quoted
on; it fits one GPU.  blest_build (reorder + BVSS build + upload) is timed separately, as the paper does (Table 7).

Prints ONE JSON line (rank 0).  `value` = GTEPS = (sum over timed BFS calls of the undirected edges of the source's
component, taken from the ORACLE's levels) / device time, inputs resident in HBM.  `e2e` = the same through the C ABI
with a pinned HOST levels_out buffer (device->host copy of the 4n-byte level array inside the timed region; the only
per-call input is the 4-byte source id).  `roofline` is for the persistent traversal kernel (the only kernel of the
step).  Outside the timed region the run checks itself: farness / reach of EVERY timed source and the full level
arrays of four of them against the CPU oracle (`parity_checked`; a mismatch prints the line and exits 1).

The default run (config c4_rmat24, N = 1) also carries, under `config.extra`, the other two components of
BASELINE.json's metric and row A5's own number: multi-source BFS sources/s on config 5 (kappa = 64, its own roofline
against a measured L2 peak, its own oracle baseline and parity sample), the forced BVSS slice path (`switching = off`:
the paper's kernel without Eq. 6) on 8 of the headline sources with its HBM fraction, and the in-repo tensor-pipe /
barrier / L2 microbenchmarks.  `--config c5_rmat18` makes the multi-source measurement the main line.

`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores on a bounded sample.
N > 1 (torchrun): single-source BFS does not shard (replicas only): every rank holds the graph
and traverses from its OWN seeded draw of 64 sources (disjoint work, fixed per rank => weak scaling, no data-path
collective).  Closeness (config 5) partitions the SOURCES over the ranks as the paper does and sums the
partial target-side farness arrays with one NCCL all-reduce (fixed total work => strong scaling).
"""
from __future__ import annotations

import argparse
import concurrent.futures
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import graphgen as gg  # noqa: E402  (seeded input generators: no method arithmetic)

REORDER_FOR = {"c1_rmat16": "none", "c2_grid4096": "none", "c3_gnm25": "none", "c4_rmat24": "degree", "c5_rmat18": "none"}
KERNEL_NAME = "bfs_lazy_kernel / bfs_eager_kernel (persistent cooperative; one launch per blest_bfs)"


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def measured_peaks():
    """HBM GB/s roofline denominator: MEASURED_PEAKS.json (driver-written), else the profiling guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def committed_profile(key: str):
    """Per-launch ncu figures of the committed capture of this workload (profiles/traffic.json), or None."""
    tp = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        return json.load(open(tp)).get(key)
    except Exception:
        return None


def load_graph(name: str, shrink: int, rank: int, world: int):
    """Rank 0 generates (seeded); with several ranks the CSR is handed over through /dev/shm."""
    if world == 1:
        return gg.make_config(name, shrink)
    import torch.distributed as dist

    base = f"/dev/shm/blest_{name}_{shrink}_{os.environ.get('MASTER_PORT', '0')}"
    if rank == 0:
        n, rp, ci = gg.make_config(name, shrink)
        np.save(base + "_rp.npy", rp)
        np.save(base + "_ci.npy", ci)
    dist.barrier()
    if rank != 0:
        rp = np.load(base + "_rp.npy")
        ci = np.load(base + "_ci.npy")
        n = rp.size - 1
    dist.barrier()
    if rank == 0:
        for s in ("_rp.npy", "_ci.npy"):
            try:
                os.remove(base + s)
            except OSError:
                pass
    return n, rp, ci


def rank_sources(name: str, rowptr: np.ndarray, rank: int) -> np.ndarray:
    """Single-source BFS does not shard (replicas only): rank r traverses from its own seeded draw of the config's
    number of sources (rank 0: the config's sources), so the ranks do disjoint work of fixed size (weak scaling)."""
    return gg.config_sources(name, rowptr, replica=rank)


def source_range(n: int, rank: int, world: int):
    """Closeness partitions the sources over the ranks: contiguous, kappa-aligned ranges covering 0..n-1."""
    per = -(-n // world)
    per = -(-per // 256) * 256  # whole batches for every kappa
    first = min(rank * per, n)
    return first, min(per, n - first)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(",") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
                pw.append(float(r[2]))
                for k, nm in enumerate(names):
                    if r[3 + k].strip().lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                continue
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm),
                       power_w_max=float(max(pw)))
        return out


def component_edges(deg: np.ndarray, levels: np.ndarray) -> int:
    """TEPS numerator (BASELINE.json): edges of the source's component, each undirected edge once."""
    return int(deg[levels >= 0].sum() // 2)


def w_alg_bytes(trace: np.ndarray, n: int, reach: int, reordered: bool, sweep_words: int) -> int:
    """Algorithmic bytes of one blest_bfs launch, from the kernel's own per-level trace.
    per call:   4 bitmaps cleared (16 B per sweep word) + levels_out pre-filled with -1 (4n B);
    every level: `q_bytes` = the graph bytes its work items cover (top-down: 20 B per quad of a slice work item, 4 B per
                CSR edge + 8 B of row pointers per edge work item; bottom-up: 8 B inline head per unvisited vertex examined,
                8 B of row pointers + 4 B per neighbour for the vertices that need the CSR scan);
                top-down adds 12 B per frontier word consumed (list entry, frontier word, threshold) and the finalisation
                sweep (12 B per sweep word: V, F_next read, F_stale cleared); bottom-up adds its sweep (8 B per sweep word);
    per discovered vertex: 4 B level write + 4 B degree (+ 4 B iperm when the graph was reordered); the vertices of the
                level the pre-fill guessed (trace `reserved` bit 31) cost their degree only."""
    w = 16 * sweep_words + 4 * n + reach * (12 if reordered else 8)
    for r in trace:
        w += int(r["q_bytes"])
        if int(r["reserved"]) >> 31:  # the level the pre-fill guessed: no level write, no iperm read (degree only)
            w -= int(r["new_vertices"]) * (8 if reordered else 4)
        if r["mode"] == 1:
            w += 8 * sweep_words
        elif r["mode"] == 2:  # eager kernel (Alg. 2): no sweeps; at least one quad + the queue entry per work item
            w += 28 * int(r["q_entries"])
        else:
            w += 12 * int(r["q_entries"]) + 12 * sweep_words
    return int(w)


def ms_alg_bytes(stats: dict, kappa: int, n_slice_sets: int, n: int, accumulate: bool) -> int:
    """Algorithmic bytes of one multi-source launch (all batches), from the kernel's own totals (blest_get_ms_stats);
    everything is L2-resident on config 5.  KB = kappa / 8 bytes per kappa-bit word.
    Stage 1, per work-queue entry (VSS): 8 B entry + the 8 gathered frontier words (8 KB); per quad 20 B (row ids + masks);
      per slice whose selected frontier words are non-zero: one V_next probe (KB); per fresh row: one atomic OR (KB) +
      the dirtySets byte;
    Stage 2, per level: the dirtySets sweep (1 B per slice set); per dirty slice set: 8 rows x (V_next + V_curr read,
      F_curr + V_curr written: 4 KB) + 8 B setPtr + a queue entry per 32 quads (counted with Stage 1) + 12 B per row of
      far / reach accumulation;
    pull level (ms_pull_level: Stage 1 + 2 fused, no queue, no dirtySets): every row's visited word read and frontier
      word written (2 KB per row); per row some live source has not reached: 8 B of row pointers; per neighbour read:
      4 B column index + its frontier word (KB);
    per batch: V_curr and V_next cleared (2 x n KB; 3 x with pull levels enabled: F_curr too)."""
    kb = kappa // 8
    pull_levels = stats.get("pull_levels", 0)
    w = stats["entries"] * (8 + 8 * kb) + stats["quads"] * 20 + stats["probes"] * kb + stats["fresh"] * (kb + 1)
    w += (stats["levels"] - pull_levels + stats["batches"]) * n_slice_sets
    w += stats["dirty_sets"] * (8 * 4 * kb + 8 + (8 * 12 if accumulate else 0))
    w += pull_levels * 2 * n * kb + stats.get("pull_rows", 0) * 8 + stats.get("pull_neighbours", 0) * (4 + kb)
    w += stats["batches"] * (3 if pull_levels else 2) * n * kb
    return int(w)


# ----------------------------------------------------------------------------------------------------------------------
# CPU oracle legs (rank 0 only; outside every timed GPU region)
# ----------------------------------------------------------------------------------------------------------------------
def oracle_bfs_checks(n, rp, ci, srcs, deg, gpu_far, gpu_reach, gpu_levels, want_baseline: bool):
    """cpu_baseline + parity of the single-source workload.  The oracle (as it stands) runs one plain queue BFS per
    OpenMP thread: the first min(cores, #sources) sources are TIMED (the reported CPU baseline), the rest run untimed.
    Every source's (farness, reach) is compared with the sums of the GPU's level array; the sources in `gpu_levels`
    are compared element by element.  Returns (cpu_baseline dict | None, parity dict, per-source oracle edge counts)."""
    import oracle

    cores = os.cpu_count() or 1
    k = int(min(cores, len(srcs)))
    t0 = time.perf_counter()
    far0, reach0, _, used = oracle.closeness(n, rp, ci, srcs[:k], nthreads=k)
    dt = time.perf_counter() - t0
    far, reach = [int(x) for x in far0], [int(x) for x in reach0]
    if len(srcs) > k:
        f1, r1, _, _ = oracle.closeness(n, rp, ci, srcs[k:])
        far += [int(x) for x in f1]
        reach += [int(x) for x in r1]
    # element-wise: the oracle's level arrays of a few sources (threads: the C call releases the GIL)
    idx = sorted(gpu_levels)
    with concurrent.futures.ThreadPoolExecutor(max(1, len(idx))) as ex:
        ref = dict(zip(idx, ex.map(lambda i: oracle.bfs(n, rp, ci, int(srcs[i])), idx)))
    bad_far = [int(srcs[i]) for i in range(len(srcs)) if (far[i], reach[i]) != (int(gpu_far[i]), int(gpu_reach[i]))]
    bad_lv = [int(srcs[i]) for i in idx if not np.array_equal(ref[i], gpu_levels[i])]
    # TEPS numerators from the ORACLE's levels: a source inside the component of a reference array shares its edge count
    edges = np.zeros(len(srcs), dtype=np.int64)
    comps = [(lv, component_edges(deg, lv)) for lv in ref.values()]
    for i, s in enumerate(srcs):
        e = next((ce for lv, ce in comps if lv[int(s)] >= 0), None)
        if e is None:
            lv = oracle.bfs(n, rp, ci, int(s))
            e = component_edges(deg, lv)
            comps.append((lv, e))
        edges[i] = e
    parity = {"sources": int(len(srcs)), "elementwise": int(len(idx)), "ok": not bad_far and not bad_lv,
              "what": "levels of every timed source: farness + reach vs oracle; `elementwise` sources: full int32 level array"}
    if bad_far or bad_lv:
        parity["mismatch_sources"] = (bad_far + bad_lv)[:8]
    base = None
    if want_baseline:
        base = {"value": float(edges[:k].sum() / dt / 1e9), "unit": "GTEPS", "cores": int(used), "kind": "oracle", "seconds": dt,
                "sample": f"first {k} of the config's {len(srcs)} sources, one plain queue BFS per OpenMP thread"}
    return base, parity, edges


def oracle_closeness_checks(n, rp, ci, cc_gpu: np.ndarray, budget_s: float = 12.0):
    """cpu_baseline + parity of the closeness workload: the oracle (all host threads, one BFS per source) on a seeded
    sample sized to ~budget_s; its fp64 closeness must equal the GPU's bit for bit on that sample."""
    import oracle

    rng = np.random.Generator(np.random.PCG64(5))
    probe = np.sort(rng.choice(n, size=min(n, 256), replace=False)).astype(np.uint32)
    t0 = time.perf_counter()
    _, _, cc_p, used = oracle.closeness(n, rp, ci, probe)
    t_probe = time.perf_counter() - t0
    k = int(min(n, max(256, budget_s / max(t_probe, 1e-6) * probe.size)))
    sample = np.sort(rng.choice(n, size=k, replace=False)).astype(np.uint32)
    t0 = time.perf_counter()
    _, _, cc_w, used = oracle.closeness(n, rp, ci, sample)
    dt = time.perf_counter() - t0
    ok = bool(np.array_equal(cc_gpu[sample], cc_w) and np.array_equal(cc_gpu[probe], cc_p))
    base = {"value": float(k / dt), "unit": "sources/s", "cores": int(used), "kind": "oracle", "seconds": dt,
            "sample": f"{k} seeded sources of the config's {n}, one plain queue BFS + farness per source, sources over all OpenMP threads"}
    parity = {"sources": int(k + probe.size), "elementwise": int(k + probe.size), "ok": ok,
              "what": "fp64 closeness of the sampled sources, bit-equal to the oracle's"}
    return base, parity


def run_reference(args, rank: int, world: int):
    """--impl reference: the CPU oracle as it stands, on the host cores, bounded sample per step."""
    if rank != 0:
        return
    import oracle

    n, rp, ci = gg.make_config(args.config, args.shrink)
    cores = os.cpu_count() or 1
    if args.config == "c5_rmat18":
        rng = np.random.Generator(np.random.PCG64(5))
        probe = rng.choice(n, size=min(n, 64), replace=False).astype(np.uint32)
        t0 = time.perf_counter()
        oracle.closeness(n, rp, ci, probe)
        t_one = (time.perf_counter() - t0) / probe.size
        budget = 150.0 / max(1, args.steps + args.warmup)
        k = int(max(cores, min(n, budget / max(t_one, 1e-9))))
        sample = np.sort(rng.choice(n, size=k, replace=False)).astype(np.uint32)
        used = 1
        for _ in range(args.warmup):
            _, _, _, used = oracle.closeness(n, rp, ci, sample)
        t0 = time.perf_counter()
        for _ in range(args.steps):
            _, _, _, used = oracle.closeness(n, rp, ci, sample)
        dt = time.perf_counter() - t0
        val, unit, metric = k * args.steps / dt, "sources/s", "msbfs_sources_per_s"
        desc = f"{k} seeded sources per step, one plain queue BFS + farness per source over all OpenMP threads, {args.steps} steps"
        cfg = {"workload": args.config, "shrink": args.shrink, "n": int(n), "nnz": int(ci.size), "sources_per_step": int(k)}
    else:
        srcs_all = gg.config_sources(args.config, rp)
        deg = gg.degrees(rp)
        # calibrate the sample: one source on one thread, then size a step to ~budget seconds
        t0 = time.perf_counter()
        lv = oracle.bfs(n, rp, ci, int(srcs_all[0]))
        t_one = time.perf_counter() - t0
        budget = 150.0 / max(1, args.steps + args.warmup)
        k = int(max(1, min(len(srcs_all), cores, budget / max(t_one, 1e-6) * cores / 2.5)))
        sample = srcs_all[:k]
        edges = 0
        for s in sample:
            edges += component_edges(deg, lv if (s == srcs_all[0] or lv[int(s)] >= 0) else oracle.bfs(n, rp, ci, int(s)))
        used = 1
        for _ in range(args.warmup):
            _, _, _, used = oracle.closeness(n, rp, ci, sample, nthreads=k)
        t0 = time.perf_counter()
        for _ in range(args.steps):
            _, _, _, used = oracle.closeness(n, rp, ci, sample, nthreads=k)
        dt = time.perf_counter() - t0
        val, unit, metric = edges * args.steps / dt / 1e9, "GTEPS", "bfs_gteps"
        desc = (f"{k} of the config's {len(srcs_all)} sources per step, one plain queue BFS per thread "
                f"(oracle_closeness: BFS + farness), {args.steps} steps")
        cfg = {"workload": args.config, "shrink": args.shrink, "n": int(n), "nnz": int(ci.size), "sources_per_step": int(k)}
    line = {
        "impl": "reference", "metric": metric, "value": val, "unit": unit, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True,
        "scaling": "strong" if args.config == "c5_rmat18" else "weak",
        "vs_baseline": None, "dtype": "int32", "data": "synthetic", "config": cfg,
        "cpu_baseline": {"value": val, "unit": unit, "cores": int(used), "kind": "oracle", "sample": desc},
        "e2e": {"value": val, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------------------------------
# GPU workloads
# ----------------------------------------------------------------------------------------------------------------------
def forced_slice_extra(g, torch, srcs, edges, n, reordered, sweep_words, peak, stream, out):
    """Row A5's own number in the driver-run record: the BVSS slice path forced through every level (`switching = off`,
    the paper's Alg. 3 without Eq. 6) on a few of the headline sources: GTEPS and the HBM fraction of its algorithmic
    bytes.  Levels are compared with the default path's (policy independence) on the fly."""
    k = min(8, len(srcs))
    ref = []
    for s in srcs[:k]:
        g.bfs(int(s), out, stream=stream)
        with torch.cuda.stream(stream):  # (the copy must be ordered before the next traversal overwrites `out`)
            ref.append(out.clone())
        stream.synchronize()
    g.configure(switching="off")
    walg, same = 0, True
    for i, s in enumerate(srcs[:k]):
        g.bfs(int(s), out, stream=stream)
        stream.synchronize()
        same = same and bool(torch.equal(out, ref[i]))
        lv_reach = int((out >= 0).sum().item())
        walg += w_alg_bytes(g.trace(), n, lv_reach, reordered, sweep_words)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps = 2
    e0.record(stream)
    for _ in range(reps):
        for s in srcs[:k]:
            g.bfs(int(s), out, stream=stream)
    e1.record(stream)
    stream.synchronize()
    ms = e0.elapsed_time(e1) / reps
    g.configure(switching="auto")
    achieved = walg / (ms * 1e-3) / 1e9
    prof = committed_profile("c4_rmat24/0/switching_off") or {}
    return {"what": "BVSS slice path on every level (switching=off: PAPER.md Alg. 3 without Eq. 6), ALU contraction",
            "sources": int(k), "gteps": float(edges[:k].sum() / (ms * 1e-3) / 1e9), "ms_per_bfs": ms / k,
            "algorithmic_gb_per_bfs": walg / k / 1e9, "achieved_gbs": achieved, "hbm_frac": achieved / peak,
            "levels_equal_default_path": same, "dram_bytes_per_launch_ncu": prof.get("dram_bytes_per_launch_mean"),
            "tensor_pipe_active_pct_ncu": prof.get("tensor_pipe_active_pct")}


def microbench_extra(blest):
    """In-repo peaks (north_star: tensor-pipe utilisation is quoted against a peak measured by an in-repo microbenchmark)."""
    out = {}
    try:
        out["mma_sync_b1_tera_bitmacs"] = blest.mma_microbench("mma_b1", 2048)[0]
        out["mma_sync_u8_tera_bytemacs"] = blest.mma_microbench("mma_u8", 2048)[0]
        if hasattr(blest, "tcgen05_microbench"):
            out["tcgen05_i8_tera_bytemacs"] = blest.tcgen05_microbench(2048)[0]
        out["grid_barrier_ns"] = blest.barrier_microbench(2000)
        for ctas in (8, 16):  # thread-block clusters: barrier and distributed-shared-memory load latency
            try:
                b, d = blest.cluster_microbench(ctas, 2000)
                out[f"cluster{ctas}_barrier_ns"], out[f"cluster{ctas}_dsmem_load_ns"] = b, d
            except Exception as e:  # a cluster size the device refuses is reported, not fatal
                out[f"cluster{ctas}_error"] = str(e)
        out["l2_copy_gbs"] = blest.l2_microbench(48 << 20, 50)
    except Exception as e:  # a microbenchmark must not take the headline down
        out["error"] = repr(e)
    return out


def closeness_measure(args, torch, blest, rank, world, dist, steps, warmup, want_cpu):
    """Exact closeness of ALL vertices of config 5 (§6.2), kappa bit-packed sources per batch; one step = the
    whole source set once.  N = 1: one blest_closeness call.  N > 1: rank r runs blest_farness_partial over its source
    range, one all-reduce sums the partial target-side arrays, blest_closeness_from_sums divides."""
    n, rp, ci = load_graph("c5_rmat18", args.shrink, rank, world) if args.config == "c5_rmat18" else gg.make_config("c5_rmat18", args.shrink)
    g = blest.Graph(n, rp, ci, reorder="none", kappa=args.kappa, ms_pull=not args.no_ms_pull, ms_lanes=args.ms_lanes)
    info = g.info()
    stream = torch.cuda.current_stream() if world > 1 else torch.cuda.Stream()
    cc = torch.zeros(n, dtype=torch.float64, device="cuda")
    host_cc = torch.zeros(n, dtype=torch.float64).pin_memory()
    far = torch.zeros(n, dtype=torch.int64, device="cuda")
    reach = torch.zeros(n, dtype=torch.int32, device="cuda")
    first, count = source_range(n, rank, world)

    def step(dst):
        if world == 1:
            g.closeness(dst, stream=stream)
            return
        if count:
            g.farness_partial(first, count, far, reach, stream=stream)
        else:
            far.zero_()
            reach.zero_()
        dist.all_reduce(far)     # the path's one exchange step: partial sums -> totals, NCCL over NVLink
        dist.all_reduce(reach)
        blest.closeness_from_sums(far, reach, cc, stream=stream)
        if dst is not cc:
            dst.copy_(cc, non_blocking=True)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    with torch.cuda.stream(stream):
        for _ in range(max(warmup, 1)):
            step(cc)
        barrier()
        stats = g.ms_stats()
        stats.update({k: v for k, v in g.ms_phases().items() if k.startswith("pull_")})
        phases = {k: v for k, v in g.ms_phases().items() if k.endswith("_ns")}
        sampler = ClockSampler(int(os.environ.get("LOCAL_RANK", "0"))) if rank == 0 else None
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(steps):
            step(cc)
        e1.record(stream)
        barrier()
        dev_ms = e0.elapsed_time(e1)
        e0.record(stream)
        for _ in range(steps):
            step(host_cc)
            stream.synchronize()  # the step's result is read on the host
        e1.record(stream)
        barrier()
        e2e_ms = e0.elapsed_time(e1)
    clocks = sampler.stop() if sampler else None
    if dist is not None:
        t = torch.tensor([dev_ms, e2e_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dev_ms, e2e_ms = float(t[0]), float(t[1])
    res = None
    if rank == 0:
        l2_peak = blest.l2_microbench(48 << 20, 50)
        walg = ms_alg_bytes(stats, args.kappa, info.n_slice_sets, n, True)  # this rank's launch
        achieved = walg / (dev_ms / steps * 1e-3) / 1e9 if world == 1 else None
        res = {
            "value": n * steps / (dev_ms * 1e-3), "ms_per_step": dev_ms / steps, "clocks": clocks,
            "e2e": {"value": n * steps / (e2e_ms * 1e-3), "unit": "sources/s", "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": int(8 * n), "ms_per_step": e2e_ms / steps},
            "config": {"workload": "c5_rmat18", "shrink": args.shrink, "n": int(n), "nnz": int(ci.size), "kappa": args.kappa,
                       "batches": (n + args.kappa - 1) // args.kappa,
                       "l2": "L2-resident graph (the workload re-traverses a 40 MB graph; no flush)",
                       "bvss_bytes": int(info.bvss_bytes),
                       "parallelism": "sources partitioned over ranks + all-reduce of the target-side sums" if world > 1 else "1 GPU",
                       "levels_per_batch": stats["levels"] / max(stats["batches"], 1), "vss_entries_per_step": stats["entries"],
                       "concurrent_lanes": args.ms_lanes if args.ms_lanes else 8,
                       "pull_levels_per_batch": stats.get("pull_levels", 0) / max(stats["batches"], 1),
                       "pull_neighbours_per_step": stats.get("pull_neighbours", 0),
                       "phase_ms_cta0": {k[:-3]: round(v / 1e6, 2) for k, v in phases.items()}},
            "roofline": {"bound": "l2", "achieved": achieved, "peak": l2_peak, "unit": "GB/s",
                         "frac": (achieved / l2_peak) if achieved else None, "traffic": None,
                         "peak_source": "measured: blest_l2_microbench (48 MB footprint copy, persistent launch configuration)",
                         "kernel": "msbfs_kernel (persistent cooperative; the batches split over concurrent launches of grid / lanes CTAs)",
                         "algorithmic_bytes_per_launch_mean": float(walg), "ms_per_launch_mean": dev_ms / steps},
            "gpu_launches": int(steps * ((2 * (args.ms_lanes if args.ms_lanes else 8)) if world == 1 else 3 + 2 * ((args.ms_lanes if args.ms_lanes else 8) - 1))),
        }
        prof = committed_profile(f"c5_rmat18/{args.shrink}/kappa{args.kappa}")
        if prof:
            res["roofline"]["traffic"] = prof.get("l2_bytes_per_launch_mean")
            res["roofline"]["traffic_source"] = prof.get("source")
        if want_cpu:
            base, parity = oracle_closeness_checks(n, rp, ci, cc.cpu().numpy())
            res["cpu_baseline"], res["parity_checked"] = base, parity
    g.close()
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="blest", choices=["blest", "reference"])
    ap.add_argument("--config", default="c4_rmat24", choices=sorted(gg.CONFIGS))
    ap.add_argument("--shrink", type=int, default=0, help="halve the linear size this many times (debug only)")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle legs (cpu_baseline AND parity)")
    ap.add_argument("--no-parity", action="store_true", help="alias of --no-cpu-baseline")
    ap.add_argument("--no-extra", action="store_true", help="skip config.extra (closeness, forced slice path, microbenchmarks)")
    ap.add_argument("--kernel", default="auto")
    ap.add_argument("--switching", default="auto")
    ap.add_argument("--contraction", default="auto")
    ap.add_argument("--reorder", default=None)
    ap.add_argument("--kappa", type=int, default=64)
    ap.add_argument("--tma-tiles", action="store_true", help="options.tune[0]: TMA-staged slice tiles in the balanced phase")
    ap.add_argument("--no-ms-pull", action="store_true", help="options.tune[1]: the multi-source kernel never switches to pull levels")
    ap.add_argument("--ms-lanes", type=int, default=0, help="options.tune[3]: concurrent lanes of the closeness call (0 = default 8, 1 = one full-grid launch)")
    ap.add_argument("--no-persist", action="store_true", help="options.persist_l2 = off: internal-id levels + gather hand-off")
    ap.add_argument("--keep-trace", action="store_true", help="leave the per-level trace on inside the timed region")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    want_cpu = not (args.no_cpu_baseline or args.no_parity)

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the BLEST path has no CPU fallback")
    import paper_2606_05081_b200 as blest

    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist

        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("OMP_NUM_THREADS", str(max(1, (os.cpu_count() or 1) // world)))
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    if args.config == "c5_rmat18":  # multi-source BFS / closeness: the metric's third component as the main line
        res = closeness_measure(args, torch, blest, rank, world, dist, args.steps, args.warmup, want_cpu)
        if rank == 0:
            line = {"metric": "msbfs_sources_per_s", "value": res["value"], "unit": "sources/s", "n_gpus": world,
                    "steps": args.steps, "warmup": args.warmup, "ms_per_step": res["ms_per_step"], "higher_is_better": True,
                    "scaling": "strong" if world > 1 else "weak", "vs_baseline": None, "dtype": "u%d" % args.kappa,
                    "data": "synthetic", "config": res["config"], "e2e": res["e2e"], "gpu_launches": res["gpu_launches"],
                    "clocks": res["clocks"], "roofline": res["roofline"]}
            for k in ("cpu_baseline", "parity_checked"):
                if k in res:
                    line[k] = res[k]
            print(json.dumps(line), flush=True)
            if "parity_checked" in res and not res["parity_checked"]["ok"]:
                sys.exit(1)
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return

    t0 = time.perf_counter()
    n, rp, ci = load_graph(args.config, args.shrink, rank, world)
    gen_s = time.perf_counter() - t0
    deg = gg.degrees(rp)
    srcs = rank_sources(args.config, rp, rank)
    reorder = args.reorder or REORDER_FOR[args.config]
    log(f"[rank {rank}] {args.config} shrink {args.shrink}: n={n} nnz={ci.size} gen {gen_s:.1f}s; building (reorder={reorder})")
    t0 = time.perf_counter()
    g = blest.Graph(n, rp, ci, reorder=reorder, kernel=args.kernel, switching=args.switching, contraction=args.contraction,
                    tma_tiles=args.tma_tiles, persist_l2=not args.no_persist)
    build_wall = time.perf_counter() - t0
    info = g.info()
    stream = torch.cuda.Stream()
    out = torch.empty(n, dtype=torch.int32, device="cuda")
    out2 = torch.empty(n, dtype=torch.int32, device="cuda")
    host_out = torch.empty(n, dtype=torch.int32).pin_memory()
    host_out2 = torch.empty(n, dtype=torch.int32).pin_memory()

    # one untimed pass (also warm-up #0): per-source sums of the GPU's level array, algorithmic bytes from the trace
    sweep_words = int(info.n_sweep_words)
    gpu_edges = np.zeros(len(srcs), dtype=np.int64)
    gpu_far = np.zeros(len(srcs), dtype=np.int64)
    gpu_reach = np.zeros(len(srcs), dtype=np.int64)
    walg = np.zeros(len(srcs), dtype=np.int64)
    nlevels = np.zeros(len(srcs), dtype=np.int64)
    keep = {}  # GPU level arrays of the sources compared element by element
    elementwise = set(np.linspace(0, len(srcs) - 1, num=min(4, len(srcs)), dtype=int).tolist())
    with torch.cuda.stream(stream):
        for i, s in enumerate(srcs):
            g.bfs(int(s), out, stream=stream)
            stream.synchronize()
            lv = out.cpu().numpy()
            reached = lv >= 0
            gpu_edges[i] = int(deg[reached].sum() // 2)
            gpu_reach[i] = int(reached.sum())
            gpu_far[i] = int(lv[reached].astype(np.int64).sum())
            if i in elementwise:
                keep[i] = lv.copy()
            tr = g.trace()
            nlevels[i] = len(tr)
            walg[i] = w_alg_bytes(tr, n, int(gpu_reach[i]), reorder != "none", sweep_words)

    def one_step(dst, evs=None):
        for i, s in enumerate(srcs):
            g.bfs(int(s), dst, stream=stream)
            if evs is not None:
                evs[i].record(stream)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # the per-level trace is a diagnostic (its records fed the byte counts above): the timed calls run without it
    if not args.keep_trace:
        g.configure(trace=False)
    for _ in range(args.warmup):
        one_step(out)
    barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    ev0 = torch.cuda.Event(enable_timing=True)
    evs = [[torch.cuda.Event(enable_timing=True) for _ in srcs] for _ in range(args.steps)]
    ev0.record(stream)
    for k in range(args.steps):
        one_step(out, evs[k])
    barrier()
    dev_ms = ev0.elapsed_time(evs[-1][-1])
    # per-BFS device times (consecutive event pairs on the launching stream)
    per = np.zeros((args.steps, len(srcs)))
    prev = ev0
    for k in range(args.steps):
        for i in range(len(srcs)):
            per[k, i] = prev.elapsed_time(evs[k][i])
            prev = evs[k][i]

    # e2e: host output buffer through the C ABI (device->host copy inside the call, on the stream)
    for _ in range(min(args.warmup, 1)):
        one_step(host_out)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for k in range(args.steps):
        one_step(host_out)
    e1.record(stream)
    barrier()
    e2e_ms = e0.elapsed_time(e1)
    # e2e, overlapped by the caller: device output buffers alternate, the device->host copy of BFS i runs on a second
    # stream while BFS i+1 traverses (still 4n bytes to the host per BFS; the PCIe copy is the bound)
    copy_stream = torch.cuda.Stream()
    dbuf, hbuf = (out, out2), (host_out, host_out2)
    done = [torch.cuda.Event(), torch.cuda.Event()]
    freed = [torch.cuda.Event(), torch.cuda.Event()]
    e0.record(stream)
    j = 0
    for k in range(args.steps):
        for s in srcs:
            b = j & 1
            if j >= 2:
                stream.wait_event(freed[b])
            g.bfs(int(s), dbuf[b], stream=stream)
            done[b].record(stream)
            copy_stream.wait_event(done[b])
            with torch.cuda.stream(copy_stream):
                hbuf[b].copy_(dbuf[b], non_blocking=True)
                freed[b].record(copy_stream)
            j += 1
    stream.wait_stream(copy_stream)
    e1.record(stream)
    barrier()
    e2e_ov_ms = e0.elapsed_time(e1)
    clocks = sampler.stop() if sampler else None
    g.configure(trace=True)

    # oracle legs (rank 0): cpu_baseline + parity + TEPS numerators from the oracle's levels
    base, parity, edges = None, None, gpu_edges
    if rank == 0 and want_cpu:
        base, parity, edges = oracle_bfs_checks(n, rp, ci, srcs, deg, gpu_far, gpu_reach, keep, True)

    t_max, e2e_max, e2e_ov_max, edge_sum = dev_ms, e2e_ms, e2e_ov_ms, float(edges.sum())
    if dist is not None:
        t = torch.tensor([dev_ms, e2e_ms, e2e_ov_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        t_max, e2e_max, e2e_ov_max = float(t[0]), float(t[1]), float(t[2])
        es = torch.tensor([edge_sum], device="cuda", dtype=torch.float64)
        dist.all_reduce(es)  # units all ranks processed (every rank has its own sources)
        edge_sum = float(es[0])
    total_edges = edge_sum * args.steps
    gteps = total_edges / (t_max * 1e-3) / 1e9

    ok = True
    if rank == 0:
        peak, peak_src = measured_peaks()
        med = np.median(per, axis=0)  # per-source median over steps, ms
        giant = edges >= 0.5 * edges.max()
        achieved = float(walg.sum() * args.steps / (per.sum() * 1e-3) / 1e9)  # GB/s, all launches of the timed region
        prof = committed_profile(f"{args.config}/{args.shrink}") or {}
        line = {
            "metric": "bfs_gteps", "value": gteps, "unit": "GTEPS", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": t_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "int32", "data": "synthetic",
            "config": {
                "workload": args.config, "shrink": args.shrink, "n": int(n), "nnz": int(ci.size), "reorder": reorder,
                "sources_per_step": int(len(srcs)), "l2": "inputs larger than L2 (BVSS+CSR >> 126 MB)" if info.bvss_bytes > (1 << 28) else "L2-resident graph (no flush: the paper's workload re-traverses a resident graph)",
                "kernel": {1: "eager (Alg. 2)", 2: "lazy (Alg. 3) + switching"}[info.kernel_chosen],
                "parallelism": "replicas only (own sources per rank)" if world > 1 else "1 GPU",
                "hand_off": "gather pass (persist_l2 off)" if args.no_persist else "fused scatter under a persisting-L2 window when levels_out fits it",
                "teps_numerator": "oracle levels" if parity else "GPU levels (oracle legs skipped)",
                "bvss_bytes": int(info.bvss_bytes), "csr_bytes": int(info.csr_bytes), "mask_density": info.mask_density, "u_div": info.u_div,
                "gen_seconds": gen_s, "reorder_seconds": info.reorder_seconds, "bvss_build_seconds": info.build_seconds,
                "component_seconds": info.component_seconds, "upload_seconds": info.upload_seconds, "build_wall_seconds": build_wall,
                "gteps_harmonic_mean_giant": float(giant.sum() / np.sum((med[giant] * 1e-3) / (edges[giant] / 1e9))) if giant.any() else None,
                "ms_per_bfs_median": float(np.median(med)), "ms_per_bfs_min": float(med.min()), "ms_per_bfs_max": float(med.max()),
                "levels_median": float(np.median(nlevels)), "us_per_level": float(np.median(med * 1e3 / np.maximum(nlevels, 1))),
            },
            "e2e": {"value": total_edges / (e2e_max * 1e-3) / 1e9, "unit": "GTEPS", "h2d_bytes_per_step": int(4 * len(srcs)),
                    "d2h_bytes_per_step": int(4 * n * len(srcs)), "ms_per_step": e2e_max / args.steps,
                    "overlapped": {"value": total_edges / (e2e_ov_max * 1e-3) / 1e9, "ms_per_step": e2e_ov_max / args.steps,
                                   "what": "device levels_out double-buffered by the caller, device->host copy of BFS i on a second stream under BFS i+1"}},
            "gpu_launches": int(args.steps * len(srcs)),
            "clocks": clocks,
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": prof.get("dram_bytes_per_launch_mean"), "traffic_source": prof.get("source"),
                         "traffic_commit": prof.get("commit"), "peak_source": peak_src, "kernel": KERNEL_NAME,
                         "algorithmic_bytes_per_launch_mean": float(walg.mean()), "ms_per_launch_mean": float(per.mean())},
            "tensor_pipe": {"active_pct": prof.get("tensor_pipe_active_pct", 0.0),
                            "note": "the default contraction is the ALU form (no MMA instruction in the timed kernel); the MMA "
                                    "forms are measured on the forced slice path (profiles/, config.extra)"},
        }
        if parity is not None:
            line["parity_checked"] = parity
            ok = parity["ok"]
        if base is not None:
            line["cpu_baseline"] = base
        if world == 1 and not args.no_extra and args.shrink == 0 and args.config == "c4_rmat24":
            extra = {}
            try:
                extra["forced_slice_path"] = forced_slice_extra(g, torch, srcs, edges, n, reorder != "none", sweep_words, peak, stream, out)
            except Exception as e:
                extra["forced_slice_path"] = {"error": repr(e)}
            g.close()
            try:
                cres = closeness_measure(args, torch, blest, 0, 1, None, 1, 1, want_cpu)
                extra["msbfs_closeness_c5"] = {"metric": "msbfs_sources_per_s", "value": cres["value"], "unit": "sources/s",
                                               "ms_per_step": cres["ms_per_step"], "e2e": cres["e2e"], "config": cres["config"],
                                               "roofline": cres["roofline"], "cpu_baseline": cres.get("cpu_baseline"),
                                               "parity_checked": cres.get("parity_checked")}
                if cres.get("parity_checked") and not cres["parity_checked"]["ok"]:
                    ok = False
            except Exception as e:
                extra["msbfs_closeness_c5"] = {"error": repr(e)}
            extra["microbench"] = microbench_extra(blest)
            line["config"]["extra"] = extra
        print(json.dumps(line), flush=True)
    g.close()
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if not ok:
        sys.exit(1)


if __name__ == "__main__":
    main()
