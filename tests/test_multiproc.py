"""N > 1 paths of bench.py on CPU: two gloo ranks (world_size 2, 127.0.0.1).

Single-source BFS does not shard (replicas only), so what the ranks share is host plumbing: rank 0
generates the seeded graph and hands the CSR over through /dev/shm, every rank draws its OWN seeded sources (disjoint
work of fixed size), and the reported time is the maximum over ranks.

Closeness shards by source: contiguous, batch-aligned source ranges per rank, one all-reduce (sum) of the
partial target-side farness / reach arrays, then the division.  The ranks' GPU kernels cannot run here, so each rank's
partial sums come from the oracle's level arrays of its range -- what is under test is the partition, the reduction and
the final formula of the N > 1 path.  No GPU and no CUDA traversal here."""
import hashlib
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch
    import torch.distributed as dist

    import bench
    import graphgen as gg
    import oracle

    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n, rp, ci = bench.load_graph("c1_rmat16", 4, rank, world)  # RMAT scale 12
        h = hashlib.sha256(rp.tobytes() + ci.tobytes()).hexdigest()
        mine = bench.rank_sources("c1_rmat16", rp, rank)
        # the bench's reduction: device time of the job = MAX over ranks
        t = torch.tensor([10.0 + rank, 20.0 - rank], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        # closeness by source partition: partial target-side sums of this rank's range, summed over the ranks
        first, count = bench.source_range(n, rank, world)
        lv = oracle.msbfs(n, rp, ci, np.arange(first, first + count, dtype=np.uint32)).astype(np.int64)
        far = torch.from_numpy(np.where(lv > 0, lv, 0).sum(axis=0))
        reach = torch.from_numpy((lv >= 0).sum(axis=0).astype(np.int64))
        dist.all_reduce(far)
        dist.all_reduce(reach)
        far, reach = far.numpy(), reach.numpy()
        cc = np.divide(reach - 1, far, out=np.zeros(n), where=far > 0)
        q.put((rank, n, h, mine.tolist(), t.tolist(), (first, count), far.tolist(), reach.tolist(), cc.tolist()))
    finally:
        dist.barrier()
        dist.destroy_process_group()


def test_two_gloo_ranks():
    import torch.multiprocessing as mp

    import graphgen as gg
    import oracle

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=600) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, n0, h0, mine0, t0, rng0, far0, reach0, cc0), (r1, n1, h1, mine1, t1, rng1, far1, reach1, cc1) = res
    assert (r0, r1) == (0, 1) and n0 == n1 == 4096
    assert h0 == h1                                   # rank 1 received exactly rank 0's CSR
    n, rp, ci = gg.make_config("c1_rmat16", 4)
    assert mine0 == gg.config_sources("c1_rmat16", rp).tolist() and len(mine0) == len(mine1) == 64
    assert mine0 != mine1                             # replicas: each rank has its own seeded draw (disjoint work)
    deg = gg.degrees(rp)
    assert all(deg[s] > 0 for s in mine1)
    assert t0 == t1 == [11.0, 20.0]                   # max over ranks
    assert not [f for f in os.listdir("/dev/shm") if f.startswith("blest_c1_rmat16_4_")]  # hand-over files removed
    # source partition: disjoint ranges that cover 0..n-1, whole kappa = 256 batches
    assert rng0[0] == 0 and rng0[0] + rng0[1] == rng1[0] and rng1[0] + rng1[1] == n and rng0[1] % 256 == 0
    far_w, reach_w, cc_w, _ = oracle.closeness(n, rp, ci)
    assert far0 == far1 == far_w.tolist() and reach0 == reach1 == reach_w.tolist()   # all-reduced sums = per-source farness
    assert cc0 == cc1 == cc_w.tolist()                # (reach - 1) / far, 0.0 where far = 0: bit-equal


@pytest.mark.parametrize("n,world", [(262144, 1), (262144, 8), (1000, 3), (5, 4), (4096, 2)])
def test_source_range_partition(n, world):
    sys.path.insert(0, ROOT)
    import bench

    got = [bench.source_range(n, r, world) for r in range(world)]
    pos = 0
    for first, count in got:
        assert first == min(pos, n) and count >= 0
        pos = first + count
    assert pos == n
