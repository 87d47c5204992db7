"""Seeded randomised parity on the GPU: a few hundred small graphs of mixed shape (RMAT, G(n,m), lattices with deleted
edges, stars, trees, disjoint unions with isolated vertices) x reorderings x kernels x forced paths, levels compared
element by element with the oracle; then multi-source BFS / farness / closeness for every kappa.  Time-boxed."""
import time

import numpy as np
import pytest

import graphgen as gg
import oracle

pytestmark = pytest.mark.gpu


def _graph(rng, small):
    kind = int(rng.integers(0, 6))
    seed = int(rng.integers(1, 1 << 30))
    if kind == 0:
        return gg.rmat(int(rng.integers(6, 11 if small else 15)), int(rng.integers(2, 20)), seed)
    if kind == 1:
        n = int(rng.integers(20, 3000 if small else 60000))
        return gg.gnm(n, int(n * rng.uniform(0.3, 6)), seed)
    if kind == 2:
        s = 50 if small else 200
        return gg.grid2d(int(rng.integers(2, s)), int(rng.integers(2, s)), float(rng.uniform(0, 0.3)), seed)
    if kind == 3:
        return gg.disjoint_union(gg.rmat(int(rng.integers(5, 10)), 8, seed), gg.path(int(rng.integers(1, 40))),
                                 gg.empty(int(rng.integers(0, 30))), gg.star(int(rng.integers(2, 500)), 0), gg.cycle(int(rng.integers(3, 30))))
    if kind == 4:
        return gg.star(int(rng.integers(2, 3000 if small else 50000)), int(rng.integers(0, 2)))
    return gg.binary_tree(int(rng.integers(1, 2000 if small else 30000)))


def test_fuzz_single_source():
    import torch

    import paper_2606_05081_b200 as blest

    rng = np.random.Generator(np.random.PCG64(20260605))
    t_end, cases = time.time() + 20.0, 0
    while time.time() < t_end or cases < 40:
        n, rp, ci = _graph(rng, small=False)
        reorder = ["none", "degree", "rcm", "jaccard"][int(rng.integers(0, 4))]
        kernel = ["auto", "lazy", "lazy", "eager"][int(rng.integers(0, 4))]
        switching = ["auto", "auto", "auto", "off", "bottom_up", "top_down", "slice"][int(rng.integers(0, 7))]
        directed = cases % 5 == 4
        if directed:  # every fifth case: a directed graph with the same vertex count and about as many edges
            n, rp, ci = gg.from_directed_edges(n, rng.integers(0, n, max(ci.size // 2, 1)), rng.integers(0, n, max(ci.size // 2, 1)))
            reorder = reorder if reorder in ("none", "degree") else "degree"
        with blest.Graph(n, rp, ci, reorder=reorder, kernel=kernel, switching=switching, directed=directed) as g:
            out = torch.full((n,), 7, dtype=torch.int32, device="cuda")
            for s in sorted(set([0, n - 1] + [int(x) for x in rng.integers(0, n, size=2)])):
                g.bfs(s, out)
                assert np.array_equal(out.cpu().numpy(), oracle.bfs(n, rp, ci, s)), (cases, n, reorder, kernel, switching, s)
            g.trace()
        cases += 1


def test_fuzz_multi_source_and_closeness():
    import torch

    import paper_2606_05081_b200 as blest

    rng = np.random.Generator(np.random.PCG64(5081))
    t_end, cases = time.time() + 15.0, 0
    while time.time() < t_end or cases < 24:
        n, rp, ci = _graph(rng, small=True)
        kappa = [32, 64, 128, 256][cases % 4]
        reorder = ["none", "degree", "rcm", "jaccard"][int(rng.integers(0, 4))]
        far_w, reach_w, cc_w, _ = oracle.closeness(n, rp, ci)
        with blest.Graph(n, rp, ci, kappa=kappa, reorder=reorder) as g:
            far = torch.zeros(n, dtype=torch.int64, device="cuda")
            reach = torch.zeros(n, dtype=torch.int32, device="cuda")
            g.farness(far, reach)
            assert np.array_equal(far.cpu().numpy().view(np.uint64), far_w), (cases, n, kappa, reorder)
            assert np.array_equal(reach.cpu().numpy().view(np.uint32), reach_w)
            cc = torch.zeros(n, dtype=torch.float64, device="cuda")
            g.closeness(cc)
            assert np.array_equal(cc.cpu().numpy(), cc_w)
            k = int(rng.integers(1, min(n, 300) + 1))
            srcs = rng.integers(0, n, size=k).astype(np.uint32)
            lv = torch.full((k, n), 9, dtype=torch.int32, device="cuda")
            g.msbfs(srcs, lv)
            assert np.array_equal(lv.cpu().numpy(), oracle.msbfs(n, rp, ci, srcs))
            fw, rw, _, _ = oracle.closeness(n, rp, ci, srcs)
            f2, r2 = np.zeros(k, dtype=np.uint64), np.zeros(k, dtype=np.uint32)
            g.farness(f2, r2, srcs=srcs)
            assert np.array_equal(f2, fw) and np.array_equal(r2, rw)
        cases += 1
