"""N > 1 path of bench.py on CPU: two gloo ranks (world_size 2, 127.0.0.1).  Single-source BFS does not shard
(replicas only), so what the ranks share is host plumbing: rank 0 generates the seeded graph and hands
the CSR over through /dev/shm, every rank takes the full (rotated) source list, and the reported time is the maximum
over ranks.  No GPU and no traversal here."""
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

    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n, rp, ci = bench.load_graph("c1_rmat16", 4, rank, world)  # RMAT scale 12
        h = hashlib.sha256(rp.tobytes() + ci.tobytes()).hexdigest()
        srcs_all = gg.config_sources("c1_rmat16", rp)
        mine = bench.rank_sources(srcs_all, rank, world)
        # the bench's reduction: device time of the job = MAX over ranks
        t = torch.tensor([10.0 + rank, 20.0 - rank], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        q.put((rank, n, h, mine.tolist(), srcs_all.tolist(), t.tolist()))
    finally:
        dist.barrier()
        dist.destroy_process_group()


def test_two_gloo_ranks_share_graph_and_rotate_sources():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, n0, h0, mine0, all0, t0), (r1, n1, h1, mine1, all1, t1) = res
    assert (r0, r1) == (0, 1) and n0 == n1 == 4096
    assert h0 == h1                                   # rank 1 received exactly rank 0's CSR
    assert all0 == all1 and len(all0) == 64
    assert sorted(mine0) == sorted(mine1) == sorted(all0)      # replicas: every rank runs every source ...
    assert mine0 == all0 and mine1 == all0[32:] + all0[:32]    # ... rotated by rank * (64 / world)
    assert t0 == t1 == [11.0, 20.0]                   # max over ranks
    assert not [f for f in os.listdir("/dev/shm") if f.startswith("blest_c1_rmat16_4_")]  # hand-over files removed
