#!/usr/bin/env python
"""bench.py -- the measurement contract of this repo.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config c4_rmat24] [--shrink S]

One "step" = one pass of the whole hot path (blest_bfs: init -> per-level contraction / switch -> lazy finalisation ->
hand-off, Alg. 2-4) over one batch of synthetic input = single-source BFS from each of the config's seeded
sources, on the resident graph.  The workload at N = 1 is BASELINE.json's headline config, configs[3] (RMAT scale 24,
edge factor 32, degree-sorted before the BVSS build, 64 sources): the config the GTEPS / HBM-roofline metric is quoted
on; it fits one GPU.  blest_build (reorder + BVSS build + upload) is timed separately, as the paper does (Table 7).

Prints ONE JSON line (rank 0).  `value` = GTEPS = (sum over timed BFS calls of the undirected edges of the source's
component) / device time, inputs resident in HBM.  `e2e` = the same through the C ABI with a pinned HOST levels_out
buffer (device->host copy of the 4n-byte level array inside the timed region; the only per-call input is the
4-byte source id).  `roofline` is for the persistent traversal kernel (the only kernel of the step).
`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores on a bounded sample.
N > 1: single-source BFS does not shard (replicas only) -- every rank holds the graph and runs
a disjoint slice of the sources' work; no data-path collective.
"""
from __future__ import annotations

import argparse
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


def rank_sources(srcs_all: np.ndarray, rank: int, world: int) -> np.ndarray:
    """Replicas only: every rank traverses from ALL the config's sources (fixed per-rank work => weak
    scaling), rotated by rank so that the ranks do not run the identical sequence at the same time."""
    return np.roll(srcs_all, -rank * max(1, len(srcs_all) // max(world, 1)))


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
    per discovered vertex: 4 B level write + 4 B degree (+ 4 B iperm when the graph was reordered)."""
    w = 16 * sweep_words + 4 * n + reach * (12 if reordered else 8)
    for r in trace:
        w += int(r["q_bytes"])
        if r["mode"] == 1:
            w += 8 * sweep_words
        elif r["mode"] == 2:  # eager kernel (Alg. 2): no sweeps; at least one quad + the queue entry per work item
            w += 28 * int(r["q_entries"])
        else:
            w += 12 * int(r["q_entries"]) + 12 * sweep_words
    return int(w)


def run_reference(args, rank: int, world: int):
    """--impl reference: the CPU oracle as it stands, on the host cores, bounded sample per step."""
    if rank != 0:
        return
    import oracle

    n, rp, ci = gg.make_config(args.config, args.shrink)
    srcs_all = gg.config_sources(args.config, rp)
    cores = os.cpu_count() or 1
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
        edges += component_edges(deg, lv if s == srcs_all[0] else oracle.bfs(n, rp, ci, int(s)))
    used = 1
    for _ in range(args.warmup):
        _, _, _, used = oracle.closeness(n, rp, ci, sample, nthreads=k)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _, _, _, used = oracle.closeness(n, rp, ci, sample, nthreads=k)
    dt = time.perf_counter() - t0
    gteps = edges * args.steps / dt / 1e9
    line = {
        "impl": "reference", "metric": "bfs_gteps", "value": gteps, "unit": "GTEPS", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": {"workload": args.config, "shrink": args.shrink, "n": int(n), "nnz": int(ci.size), "sources_per_step": int(k)},
        "cpu_baseline": {"value": gteps, "unit": "GTEPS", "cores": int(used), "kind": "oracle",
                         "sample": f"{k} of the config's {len(srcs_all)} sources per step, one plain queue BFS per thread "
                                   f"(oracle_closeness: BFS + farness), {args.steps} steps"},
        "e2e": {"value": gteps, "unit": "GTEPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="blest", choices=["blest", "reference"])
    ap.add_argument("--config", default="c4_rmat24", choices=sorted(gg.CONFIGS))
    ap.add_argument("--shrink", type=int, default=0, help="halve the linear size this many times (debug only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--kernel", default="auto")
    ap.add_argument("--switching", default="auto")
    ap.add_argument("--contraction", default="auto")
    ap.add_argument("--kappa", type=int, default=64)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)

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
    if args.config == "c5_rmat18":  # multi-source BFS / closeness: a different metric (sources per second)
        run_closeness(args, rank, world, torch, blest)
        return
    dist = None
    if world > 1:
        import torch.distributed as dist

        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("OMP_NUM_THREADS", str(max(1, (os.cpu_count() or 1) // world)))
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    t0 = time.perf_counter()
    n, rp, ci = load_graph(args.config, args.shrink, rank, world)
    gen_s = time.perf_counter() - t0
    deg = gg.degrees(rp)
    srcs_all = gg.config_sources(args.config, rp)
    # replicas only: every rank traverses the full graph; rank r takes the sources rotated by r so that the ranks do
    # not run the identical sequence.  Per-rank work is fixed as N grows => weak scaling.
    srcs = rank_sources(srcs_all, rank, world)
    reorder = REORDER_FOR[args.config]
    log(f"[rank {rank}] {args.config} shrink {args.shrink}: n={n} nnz={ci.size} gen {gen_s:.1f}s; building (reorder={reorder})")
    t0 = time.perf_counter()
    g = blest.Graph(n, rp, ci, reorder=reorder, kernel=args.kernel, switching=args.switching, contraction=args.contraction)
    build_wall = time.perf_counter() - t0
    info = g.info()
    stream = torch.cuda.Stream()
    out = torch.empty(n, dtype=torch.int32, device="cuda")
    host_out = torch.empty(n, dtype=torch.int32).pin_memory()

    # per-source numerators + algorithmic bytes from one untimed pass (also warm-up #0)
    sweep_words = int(info.n_sweep_words)
    edges = np.zeros(len(srcs), dtype=np.int64)
    walg = np.zeros(len(srcs), dtype=np.int64)
    nlevels = np.zeros(len(srcs), dtype=np.int64)
    with torch.cuda.stream(stream):
        for i, s in enumerate(srcs):
            g.bfs(int(s), out, stream=stream)
            stream.synchronize()
            lv = out.cpu().numpy()
            edges[i] = component_edges(deg, lv)
            tr = g.trace()
            nlevels[i] = len(tr)
            walg[i] = w_alg_bytes(tr, n, int((lv >= 0).sum()), reorder != "none", sweep_words)

    def one_step(dst, evs=None):
        for i, s in enumerate(srcs):
            g.bfs(int(s), dst, stream=stream)
            if evs is not None:
                evs[i].record(stream)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

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
    clocks = sampler.stop() if sampler else None

    t_max, e2e_max = dev_ms, e2e_ms
    if dist is not None:
        t = torch.tensor([dev_ms, e2e_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        t_max, e2e_max = float(t[0]), float(t[1])
    total_edges = int(edges.sum()) * args.steps * world
    gteps = total_edges / (t_max * 1e-3) / 1e9
    e2e_gteps = total_edges / (e2e_max * 1e-3) / 1e9

    if rank == 0:
        peak, peak_src = measured_peaks()
        med = np.median(per, axis=0)  # per-source median over steps, ms
        giant = edges >= 0.5 * edges.max()
        achieved = float(walg.sum() * args.steps / (per.sum() * 1e-3) / 1e9)  # GB/s, all launches of the timed region
        line = {
            "metric": "bfs_gteps", "value": gteps, "unit": "GTEPS", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": t_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "int32", "data": "synthetic",
            "config": {
                "workload": args.config, "shrink": args.shrink, "n": int(n), "nnz": int(ci.size), "reorder": reorder,
                "sources_per_step": int(len(srcs)), "l2": "inputs larger than L2 (BVSS+CSR >> 126 MB)" if info.bvss_bytes > (1 << 28) else "L2-resident graph (no flush: the paper's workload re-traverses a resident graph)",
                "kernel": {1: "eager (Alg. 2)", 2: "lazy (Alg. 3) + switching"}[info.kernel_chosen], "parallelism": "replicas only" if world > 1 else "1 GPU",
                "bvss_bytes": int(info.bvss_bytes), "csr_bytes": int(info.csr_bytes), "mask_density": info.mask_density, "u_div": info.u_div,
                "gen_seconds": gen_s, "reorder_seconds": info.reorder_seconds, "bvss_build_seconds": info.build_seconds,
                "upload_seconds": info.upload_seconds, "build_wall_seconds": build_wall,
                "gteps_harmonic_mean_giant": float(giant.sum() / np.sum((med[giant] * 1e-3) / (edges[giant] / 1e9))) if giant.any() else None,
                "ms_per_bfs_median": float(np.median(med)), "ms_per_bfs_min": float(med.min()), "ms_per_bfs_max": float(med.max()),
                "levels_median": float(np.median(nlevels)), "us_per_level": float(np.median(med * 1e3 / np.maximum(nlevels, 1))),
            },
            "e2e": {"value": e2e_gteps, "unit": "GTEPS", "h2d_bytes_per_step": int(4 * len(srcs)),
                    "d2h_bytes_per_step": int(4 * n * len(srcs)), "ms_per_step": e2e_max / args.steps},
            "gpu_launches": int(args.steps * len(srcs)),
            "clocks": clocks,
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": None, "peak_source": peak_src, "kernel": KERNEL_NAME,
                         "algorithmic_bytes_per_launch_mean": float(walg.mean()), "ms_per_launch_mean": float(per.mean())},
        }
        tp = os.path.join(ROOT, "profiles", "traffic.json")  # dram bytes per launch from the committed ncu capture
        if os.path.exists(tp):
            try:
                t = json.load(open(tp)).get(f"{args.config}/{args.shrink}")
                if t:  # bytes per launch, like `achieved`'s numerator
                    line["roofline"]["traffic"] = float(t["dram_bytes_per_launch_mean"])
                    line["roofline"]["traffic_source"] = t["source"]
            except Exception:
                pass
        if not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(n, rp, ci, srcs_all, deg)
        print(json.dumps(line), flush=True)
    g.close()
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def run_closeness(args, rank, world, torch, blest):
    """--config c5_rmat18: exact closeness of ALL vertices (§6.2), kappa bit-packed sources per batch; one step =
    one blest_closeness call over all n sources.  Reported as MS-BFS sources per second (BASELINE.json metric).  The
    graph (40 MB) is L2-resident by nature of the workload.  Replicas only for N > 1."""
    n, rp, ci = gg.make_config(args.config, args.shrink)
    g = blest.Graph(n, rp, ci, reorder="none", kappa=args.kappa)
    info = g.info()
    stream = torch.cuda.Stream()
    cc = torch.zeros(n, dtype=torch.float64, device="cuda")
    host_cc = torch.zeros(n, dtype=torch.float64).pin_memory()
    for _ in range(max(args.warmup, 1)):
        g.closeness(cc, stream=stream)
    torch.cuda.synchronize()
    sampler = ClockSampler(int(os.environ.get("LOCAL_RANK", "0"))) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        g.closeness(cc, stream=stream)
    e1.record(stream)
    torch.cuda.synchronize()
    dev_ms = e0.elapsed_time(e1)
    e0.record(stream)
    for _ in range(args.steps):
        g.closeness(host_cc, stream=stream)
    e1.record(stream)
    torch.cuda.synchronize()
    e2e_ms = e0.elapsed_time(e1)
    clocks = sampler.stop() if sampler else None
    if rank == 0:
        line = {
            "metric": "msbfs_sources_per_s", "value": n * args.steps * world / (dev_ms * 1e-3), "unit": "sources/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dev_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u%d" % args.kappa, "data": "synthetic",
            "config": {"workload": args.config, "shrink": args.shrink, "n": int(n), "nnz": int(ci.size), "kappa": args.kappa,
                       "batches": (n + args.kappa - 1) // args.kappa, "l2": "L2-resident graph (the workload re-traverses a 40 MB graph)",
                       "bvss_bytes": int(info.bvss_bytes), "parallelism": "replicas only" if world > 1 else "1 GPU"},
            "e2e": {"value": n * args.steps * world / (e2e_ms * 1e-3), "unit": "sources/s", "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": int(8 * n), "ms_per_step": e2e_ms / args.steps},
            "gpu_launches": int(2 * args.steps), "clocks": clocks,
        }
        print(json.dumps(line), flush=True)
    g.close()


def cpu_baseline(n, rp, ci, srcs_all, deg):
    """The oracle as it stands on the host cores, bounded sample (~10-30 s): min(cores, #sources) sources, one per thread."""
    import oracle

    cores = os.cpu_count() or 1
    k = int(min(cores, len(srcs_all)))
    sample = srcs_all[:k]
    t0 = time.perf_counter()
    far, reach, _, used = oracle.closeness(n, rp, ci, sample, nthreads=k)
    dt = time.perf_counter() - t0
    # component edges of the sampled sources: RMAT/G(n,m)/grid sources of one component share the numerator; recompute exactly
    e = 0
    lv0 = None
    for s, r in zip(sample, reach):
        if lv0 is None or lv0[int(s)] < 0:
            lv0 = oracle.bfs(n, rp, ci, int(s))
        e += component_edges(deg, lv0)
    return {"value": e / dt / 1e9, "unit": "GTEPS", "cores": int(used), "kind": "oracle", "seconds": dt,
            "sample": f"first {k} of the config's {len(srcs_all)} sources, one plain queue BFS per OpenMP thread"}


if __name__ == "__main__":
    main()
