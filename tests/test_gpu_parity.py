"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, bit-exact for levels,
farness and reach; closeness within 1e-12 relative (expected bit-equal).  Sizes the oracle finishes in seconds, spanning
several tiles, ragged tails and the degenerate cases.  Every path is forced in turn (policy independence, T5)."""
import numpy as np
import pytest

import graphgen as gg
import oracle

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch

    assert torch.cuda.is_available()
    return torch


@pytest.fixture(scope="module")
def blest():
    import paper_2606_05081_b200 as b

    b.load()
    return b


SMALL = {
    "path1000": lambda: gg.path(1000),                                  # ~1000 levels: persistent loop
    "star_hub": lambda: gg.star(5000, 17),                              # one slice set with >> tau slices, hub row
    "complete": lambda: gg.complete(130),
    "union": lambda: gg.disjoint_union(gg.path(9), gg.empty(5), gg.complete(6), gg.cycle(11)),
    "ragged": lambda: gg.gnm(1003, 2500, 7),                            # n not a multiple of 8 / 32 / 128
    "grid": lambda: gg.grid2d(37, 41, 0.05, 8),
    "rmat12": lambda: gg.rmat(12, 16, 9),
    "tiny": lambda: gg.path(2),
    "single": lambda: gg.empty(1),
}


def sources_for(n, rp, k=4):
    deg = gg.degrees(rp)
    s = {0, n - 1, int(np.argmax(deg))}
    iso = np.flatnonzero(deg == 0)
    if iso.size:
        s.add(int(iso[0]))                                               # isolated source
    s |= {int(x) for x in gg.pick_sources(rp, min(k, n), 5, nonzero_degree=False)}
    return sorted(s)


def check_bfs(blest, torch, g, graph, srcs, host_out=False):
    n, rp, ci = graph
    for s in srcs:
        want = oracle.bfs(n, rp, ci, s)
        if host_out:
            out = np.full(n, 7, dtype=np.int32)
            g.bfs(s, out)
            torch.cuda.synchronize()
            got = out
        else:
            out = torch.full((n,), 7, dtype=torch.int32, device="cuda")
            g.bfs(s, out)
            got = out.cpu().numpy()
        assert np.array_equal(got, want), f"src {s}: {np.flatnonzero(got != want)[:8]}"
        tr = g.trace()                                                   # also surfaces a queue overflow
        assert len(tr) >= int(want.max())


def test_contraction_forms_exhaustive(blest, torch_cuda):
    """Every contraction form == (mask & alpha) != 0 over all 2^8 x 2^8 pairs in all four byte positions (T2)."""
    for form in ("alu", "mma_b1", "mma_u8"):
        assert blest.contraction_selftest(form) == 0, form


@pytest.mark.parametrize("name", sorted(SMALL))
@pytest.mark.parametrize("kernel", ["lazy", "eager"])
def test_small_graphs_default_policy(blest, torch_cuda, name, kernel):
    graph = SMALL[name]()
    with blest.Graph(*graph, kernel=kernel) as g:
        check_bfs(blest, torch_cuda, g, graph, sources_for(graph[0], graph[1]))


@pytest.mark.parametrize("name", sorted(SMALL))
def test_small_graphs_eager_grid_wide_only(blest, torch_cuda, name):
    """Alg. 2 proper: switching="off" keeps the eager kernel on the grid-wide slice path (no small-frontier mode)."""
    graph = SMALL[name]()
    with blest.Graph(*graph, kernel="eager", switching="off") as g:
        check_bfs(blest, torch_cuda, g, graph, sources_for(graph[0], graph[1]))


@pytest.mark.parametrize("maker", [lambda: gg.gnm(200_000, 800_000, 3), lambda: gg.rmat(15, 16, 4), lambda: gg.grid2d(300, 700, 0.05, 6)])
def test_eager_larger_graphs(blest, torch_cuda, maker):
    """Alg. 2 on graphs whose frontiers grow to tens of thousands of vertices and shrink again (queue parity flips,
    cooperative segment expansion).  The eager kernel has one mode: every trace record says 2."""
    graph = maker()
    with blest.Graph(*graph, kernel="eager") as g:
        check_bfs(blest, torch_cuda, g, graph, sources_for(graph[0], graph[1], 3))
        assert set(int(m) for m in g.trace()["mode"]) == {2}


@pytest.mark.parametrize("name", ["star_hub", "union", "ragged", "rmat12", "grid"])
@pytest.mark.parametrize("switching", ["auto", "off", "bottom_up", "top_down", "slice"])
def test_policy_independence_lazy(blest, torch_cuda, name, switching):
    """Forcing each path on every level yields identical levels."""
    graph = SMALL[name]()
    with blest.Graph(*graph, kernel="lazy", switching=switching) as g:
        check_bfs(blest, torch_cuda, g, graph, sources_for(graph[0], graph[1], 3))


@pytest.mark.parametrize("mask", [0b10, 0b1100, 0b10101010, 0xFFFFFFF0])
def test_scripted_direction_per_level(blest, torch_cuda, mask):
    graph = SMALL["rmat12"]()
    with blest.Graph(*graph, kernel="lazy", switching="scripted", bu_mask=mask) as g:
        check_bfs(blest, torch_cuda, g, graph, sources_for(graph[0], graph[1], 2))
        modes = g.trace()["mode"]
        for lvl, m in enumerate(modes, start=1):
            assert m == ((mask >> min(lvl, 31)) & 1)


@pytest.mark.parametrize("contraction", ["alu", "mma_b1", "mma_u8"])
@pytest.mark.parametrize("kernel", ["lazy", "eager"])
def test_contraction_forms_in_traversal(blest, torch_cuda, contraction, kernel):
    graph = SMALL["rmat12"]()
    with blest.Graph(*graph, kernel=kernel, contraction=contraction, switching="off") as g:
        check_bfs(blest, torch_cuda, g, graph, sources_for(graph[0], graph[1], 2))


@pytest.mark.parametrize("reorder", ["none", "degree", "rcm", "jaccard"])
@pytest.mark.parametrize("kernel", ["lazy", "eager"])
def test_reordering_is_invisible(blest, torch_cuda, reorder, kernel):
    for name in ("rmat12", "grid", "union"):
        graph = SMALL[name]()
        with blest.Graph(*graph, kernel=kernel, reorder=reorder, validate=True) as g:
            check_bfs(blest, torch_cuda, g, graph, sources_for(graph[0], graph[1], 2))
            check_bfs(blest, torch_cuda, g, graph, sources_for(graph[0], graph[1], 1)[:2], host_out=True)


def test_device_csr_input_and_stream(blest, torch_cuda):
    torch = torch_cuda
    n, rp, ci = SMALL["rmat12"]()
    drp = torch.from_numpy(rp.view(np.int32)).cuda()
    dci = torch.from_numpy(ci.view(np.int32)).cuda()
    st = torch.cuda.Stream()
    with blest.Graph(n, drp, dci) as g:
        out = torch.empty(n, dtype=torch.int32, device="cuda")
        with torch.cuda.stream(st):
            g.bfs(3, out, stream=st)
        st.synchronize()
        assert np.array_equal(out.cpu().numpy(), oracle.bfs(n, rp, ci, 3))


def test_config1_rmat16_all_64_sources(blest, torch_cuda):
    """BASELINE.json configs[0] at full size: RMAT scale 16, 64 seeded sources."""
    torch = torch_cuda
    n, rp, ci = gg.make_config("c1_rmat16")
    srcs = gg.config_sources("c1_rmat16", rp)
    assert srcs.size == 64
    for opts in (dict(), dict(reorder="degree"), dict(kernel="eager"), dict(kernel="lazy", switching="off")):
        with blest.Graph(n, rp, ci, **opts) as g:
            out = torch.empty(n, dtype=torch.int32, device="cuda")
            for s in srcs:
                g.bfs(int(s), out)
                assert np.array_equal(out.cpu().numpy(), oracle.bfs(n, rp, ci, int(s))), (opts, int(s))


@pytest.mark.parametrize("name,shrink", [("c2_grid4096", 4), ("c3_gnm25", 7), ("c4_rmat24", 6), ("c5_rmat18", 2)])
def test_configs_reduced(blest, torch_cuda, name, shrink):
    torch = torch_cuda
    n, rp, ci = gg.make_config(name, shrink)
    srcs = gg.config_sources(name, rp)[:4] if name != "c5_rmat18" else gg.pick_sources(rp, 4, 3)
    reorder = {"c4_rmat24": "degree", "c3_gnm25": "rcm"}.get(name, "none")
    with blest.Graph(n, rp, ci, reorder=reorder) as g:
        out = torch.empty(n, dtype=torch.int32, device="cuda")
        for s in srcs:
            g.bfs(int(s), out)
            assert np.array_equal(out.cpu().numpy(), oracle.bfs(n, rp, ci, int(s)))


# ---- multi-source BFS (A11) and closeness (A12) ------------------------------------------------------------------
@pytest.mark.parametrize("kappa", [32, 64, 128, 256])
def test_msbfs_rows_equal_single_source(blest, torch_cuda, kappa):
    torch = torch_cuda
    graph = gg.disjoint_union(gg.rmat(9, 8, 11), gg.path(13), gg.empty(3))
    n, rp, ci = graph
    rng = np.random.Generator(np.random.PCG64(kappa))
    with blest.Graph(n, rp, ci, kappa=kappa) as g:
        for k in (1, kappa - 1, kappa, kappa + 1, 2 * kappa + 3):
            srcs = rng.integers(0, n, size=k).astype(np.uint32)
            if k >= 4:
                srcs[1] = srcs[0]                                        # duplicate sources
                srcs[2] = (srcs[0] & ~np.uint32(7)) | ((srcs[0] + 1) & 7)  # two sources sharing a slice set
                srcs[3] = n - 1                                          # isolated vertex
            want = oracle.msbfs(n, rp, ci, srcs)
            out = torch.full((k, n), 9, dtype=torch.int32, device="cuda")
            g.msbfs(srcs, out)
            assert np.array_equal(out.cpu().numpy(), want), k
            host = np.full((k, n), 9, dtype=np.int32)
            g.msbfs(srcs, host)
            assert np.array_equal(host, want)


@pytest.mark.parametrize("reorder", ["none", "degree"])
@pytest.mark.parametrize("kappa", [32, 64, 128, 256])
def test_closeness_all_vertices(blest, torch_cuda, reorder, kappa):
    torch = torch_cuda
    graph = gg.disjoint_union(gg.rmat(10, 8, 21), gg.star(30, 2), gg.empty(5), gg.path(2))
    n, rp, ci = graph
    far_w, reach_w, cc_w, _ = oracle.closeness(n, rp, ci)
    with blest.Graph(n, rp, ci, kappa=kappa, reorder=reorder) as g:
        far = torch.zeros(n, dtype=torch.int64, device="cuda")
        reach = torch.zeros(n, dtype=torch.int32, device="cuda")
        g.farness(far, reach)
        assert np.array_equal(far.cpu().numpy().view(np.uint64), far_w)           # bit-exact integers
        assert np.array_equal(reach.cpu().numpy().view(np.uint32), reach_w)
        cc = torch.zeros(n, dtype=torch.float64, device="cuda")
        g.closeness(cc)
        got = cc.cpu().numpy()
        assert np.allclose(got, cc_w, rtol=1e-12, atol=0.0) and np.array_equal(got == 0.0, cc_w == 0.0)
        assert np.array_equal(got, cc_w)                                          # one IEEE division on both sides
        host = np.zeros(n, dtype=np.float64)
        g.closeness(host)
        assert np.array_equal(host, cc_w)


@pytest.mark.parametrize("kappa", [32, 64])
def test_closeness_source_subset(blest, torch_cuda, kappa):
    """Arbitrary source subsets use per-source counts (reading R13), incl. duplicates and k not a multiple of kappa."""
    torch = torch_cuda
    n, rp, ci = gg.disjoint_union(gg.rmat(9, 8, 31), gg.cycle(7), gg.empty(2))
    srcs = np.array([5, 5, 0, n - 1, n - 4, 100, 17] + list(range(40, 40 + kappa)), dtype=np.uint32)
    far_w, reach_w, cc_w, _ = oracle.closeness(n, rp, ci, srcs)
    with blest.Graph(n, rp, ci, kappa=kappa) as g:
        far = np.zeros(srcs.size, dtype=np.uint64)
        reach = np.zeros(srcs.size, dtype=np.uint32)
        g.farness(far, reach, srcs=srcs)
        assert np.array_equal(far, far_w) and np.array_equal(reach, reach_w)
        cc = torch.zeros(srcs.size, dtype=torch.float64, device="cuda")
        g.closeness(cc, srcs=srcs)
        assert np.array_equal(cc.cpu().numpy(), cc_w)


def test_trace_and_info(blest, torch_cuda):
    torch = torch_cuda
    n, rp, ci = SMALL["rmat12"]()
    with blest.Graph(n, rp, ci, kernel="lazy", reorder="degree") as g:
        i = g.info()
        assert i.n == n and i.nnz == ci.size and i.num_sms > 0 and i.grid_blocks == i.num_sms and i.kernel_chosen == 2
        out = torch.empty(n, dtype=torch.int32, device="cuda")
        s = int(gg.pick_sources(rp, 1, 1)[0])
        g.bfs(s, out)
        want = oracle.bfs(n, rp, ci, s)
        tr = g.trace()
        depth = int(want.max())
        # either a last level that discovers nothing, or the traversal stopped because the component was exhausted
        assert len(tr) in (depth, depth + 1)
        for lvl in range(1, depth + 1):
            assert tr["new_vertices"][lvl - 1] == np.count_nonzero(want == lvl)
        assert (len(tr) == depth or tr["new_vertices"][-1] == 0) and np.all(np.diff(tr["t_ns"].astype(np.int64)) > 0)
        assert tr["unvisited"][-1] == np.count_nonzero(want < 0)


def test_bad_arguments(blest, torch_cuda):
    from paper_2606_05081_b200 import binding

    torch = torch_cuda
    n, rp, ci = SMALL["union"]()
    with blest.Graph(n, rp, ci) as g:
        out = torch.empty(n, dtype=torch.int32, device="cuda")
        with pytest.raises(blest.BlestError) as e:
            g.bfs(n, out)
        assert e.value.status == binding.EINVAL
        with pytest.raises(blest.BlestError):
            g.msbfs(np.array([n], np.uint32), torch.empty((1, n), dtype=torch.int32, device="cuda"))
        with pytest.raises(blest.BlestError):
            g.closeness(torch.empty(3, dtype=torch.float64, device="cuda"), srcs=np.array([0, 1, n + 5], np.uint32))


def test_gather_handoff_path(blest, torch_cuda):
    """Reordered graphs whose levels_out does not fit the persisting-L2 window use internal-id levels + a final gather pass
    (C3-sized arrays).  persist_l2=False forces that path on small graphs."""
    torch = torch_cuda
    for maker in (lambda: gg.rmat(12, 16, 9), lambda: gg.disjoint_union(gg.path(9), gg.empty(5), gg.complete(6)),
                  lambda: gg.gnm(1003, 2500, 7)):
        n, rp, ci = maker()
        for reorder in ("degree", "rcm"):
            with blest.Graph(n, rp, ci, kernel="lazy", reorder=reorder, persist_l2=False) as g:
                out = torch.full((n,), 7, dtype=torch.int32, device="cuda")
                for s in (0, n // 2, n - 1):
                    g.bfs(s, out)
                    assert np.array_equal(out.cpu().numpy(), oracle.bfs(n, rp, ci, s)), (reorder, s)
                g.configure(persist_l2=True)   # and back to the fused scatter on the same handle
                g.bfs(1, out)
                assert np.array_equal(out.cpu().numpy(), oracle.bfs(n, rp, ci, 1))


def with_loops_and_duplicates(graph, seed):
    """The same graph with self-loops on a third of the vertices (also isolated ones) and every fifth entry duplicated:
    still sorted and symmetric (both are legal and change nothing)."""
    n, rp, ci = graph
    rng = np.random.Generator(np.random.PCG64(seed))
    loops = rng.random(n) < 0.34
    loops[0] = True
    rows = []
    for u in range(n):
        row = ci[rp[u]:rp[u + 1]].astype(np.int64)
        dup = row[rng.random(row.size) < 0.2]
        extra = [np.array([u, u] if u % 2 else [u], dtype=np.int64)] if loops[u] else []
        rows.append(np.sort(np.concatenate([row, dup] + extra)))
    rp2 = np.zeros(n + 1, dtype=np.uint32)
    rp2[1:] = np.cumsum([r.size for r in rows])
    ci2 = (np.concatenate(rows) if rows else np.empty(0)).astype(np.uint32)
    return n, rp2, ci2


@pytest.mark.parametrize("name", ["union", "ragged", "rmat12", "star_hub"])
def test_self_loops_and_duplicate_entries(blest, torch_cuda, name):
    """Diagonal and repeated CSR entries (SuiteSparse matrices carry them) through every kernel, forced path and
    reordering, and through the multi-source kernel.  The level-1 fast path of the lazy kernel must not re-discover
    the source through (src, src)."""
    torch = torch_cuda
    base = SMALL[name]()
    graph = with_loops_and_duplicates(base, 77)
    n, rp, ci = graph
    want0 = oracle.bfs(*base, 0)
    assert np.array_equal(oracle.bfs(n, rp, ci, 0), want0)            # the oracle itself: loops / duplicates are inert
    srcs = sources_for(n, rp, 3)
    for opts in (dict(kernel="lazy"), dict(kernel="lazy", reorder="degree"), dict(kernel="lazy", reorder="rcm", persist_l2=False),
                 dict(kernel="lazy", switching="off"), dict(kernel="lazy", switching="bottom_up"),
                 dict(kernel="lazy", switching="top_down"), dict(kernel="lazy", switching="slice", contraction="mma_u8"),
                 dict(kernel="eager"), dict(kernel="eager", reorder="degree")):
        with blest.Graph(n, rp, ci, validate=True, **opts) as g:
            check_bfs(blest, torch, g, graph, srcs)
    ms = np.array(srcs + srcs[:2], dtype=np.uint32)
    with blest.Graph(n, rp, ci, kappa=32, reorder="degree") as g:
        lv = torch.full((ms.size, n), 9, dtype=torch.int32, device="cuda")
        g.msbfs(ms, lv)
        assert np.array_equal(lv.cpu().numpy(), oracle.msbfs(n, rp, ci, ms))
        far_w, reach_w, cc_w, _ = oracle.closeness(n, rp, ci)
        cc = torch.zeros(n, dtype=torch.float64, device="cuda")
        g.closeness(cc)
        assert np.array_equal(cc.cpu().numpy(), cc_w)


def test_multi_source_calls_do_not_block_the_host(blest, torch_cuda):
    """include/blest.h "Asynchrony": blest_msbfs / blest_closeness enqueue and return.  The stream is first kept busy by a
    long spin kernel; both calls (and an event recorded between them) must return while it is still running."""
    torch = torch_cuda
    n, rp, ci = gg.rmat(12, 16, 9)
    srcs = gg.pick_sources(rp, 70, 3)
    st = torch.cuda.Stream()
    with blest.Graph(n, rp, ci, kappa=64) as g:
        lv1 = torch.full((srcs.size, n), 9, dtype=torch.int32, device="cuda")
        lv2 = torch.full((srcs.size, n), 9, dtype=torch.int32, device="cuda")
        cc = torch.zeros(srcs.size, dtype=torch.float64, device="cuda")
        g.msbfs(srcs, lv1, stream=st)                                     # warm-up: workspace + staging slot exist
        st.synchronize()
        lv1.fill_(9)
        torch.cuda.synchronize()
        done = torch.cuda.Event()
        mid = torch.cuda.Event()
        with torch.cuda.stream(st):
            torch.cuda._sleep(int(2e9))                                   # ~1 s of device time ahead of the calls
            g.msbfs(srcs, lv1, stream=st)
            mid.record(st)
            g.msbfs(srcs[::-1].copy(), lv2, stream=st)
            g.closeness(cc, srcs=srcs, stream=st)
            done.record(st)
        assert not mid.query() and not done.query(), "a multi-source call waited for the device"
        st.synchronize()
        assert g.last_status() == 0
        want = oracle.msbfs(n, rp, ci, srcs)
        assert np.array_equal(lv1.cpu().numpy(), want) and np.array_equal(lv2.cpu().numpy(), want[::-1])
        assert np.array_equal(cc.cpu().numpy(), oracle.closeness(n, rp, ci, srcs)[2])


@pytest.mark.parametrize("kernel", ["eager", "lazy", "msbfs"])
def test_queue_overflow_is_reported(blest, torch_cuda, kernel):
    """A deliberately tiny work-queue capacity: the kernels drop what does not fit, finish, and latch BLEST_EOVERFLOW;
    blest_last_status returns and clears it, later calls are refused until then (never silent)."""
    from paper_2606_05081_b200 import binding

    torch = torch_cuda
    n, rp, ci = gg.star(5000, 17) if kernel == "lazy" else gg.rmat(12, 16, 9)
    opts = dict(kernel="eager") if kernel == "eager" else dict(kernel="lazy", switching="top_down")
    with blest.Graph(n, rp, ci, queue_capacity=2, kappa=32, **opts) as g:
        out = torch.empty(n, dtype=torch.int32, device="cuda")
        if kernel == "msbfs":
            g.msbfs(np.arange(40, dtype=np.uint32), torch.empty((40, n), dtype=torch.int32, device="cuda"))
        else:
            g.bfs(17, out)
        torch.cuda.synchronize()
        with pytest.raises(blest.BlestError) as e:                       # the latch refuses the next call
            g.bfs(17, out)
        assert e.value.status == binding.EOVERFLOW
        assert g.last_status() == binding.EOVERFLOW
        assert g.last_status() == binding.OK                              # cleared
    with blest.Graph(n, rp, ci, kappa=32, **opts) as g:                  # automatic capacities never overflow
        out = torch.empty(n, dtype=torch.int32, device="cuda")
        g.bfs(17, out)
        assert g.last_status() == binding.OK and np.array_equal(out.cpu().numpy(), oracle.bfs(n, rp, ci, 17))


@pytest.mark.parametrize("reorder", ["none", "degree"])
def test_closeness_by_source_partition(blest, torch_cuda, reorder):
    """The multi-GPU form of PAPER.md:678 on one device: partial target-side sums of three source ranges (one of them
    not batch-aligned) added up = farness / reach of every vertex; blest_closeness_from_sums = the oracle's division."""
    torch = torch_cuda
    n, rp, ci = gg.disjoint_union(gg.rmat(10, 8, 21), gg.star(30, 2), gg.empty(5), gg.path(2))
    far_w, reach_w, cc_w, _ = oracle.closeness(n, rp, ci)
    with blest.Graph(n, rp, ci, kappa=64, reorder=reorder) as g:
        far = torch.zeros(n, dtype=torch.int64, device="cuda")
        reach = torch.zeros(n, dtype=torch.int32, device="cuda")
        pf = torch.zeros(n, dtype=torch.int64, device="cuda")
        pr = torch.zeros(n, dtype=torch.int32, device="cuda")
        for first, count in ((0, 512), (512, 301), (813, n - 813)):
            g.farness_partial(first, count, pf, pr)
            far += pf
            reach += pr
        assert np.array_equal(far.cpu().numpy().view(np.uint64), far_w)
        assert np.array_equal(reach.cpu().numpy().view(np.uint32), reach_w)
        cc = torch.zeros(n, dtype=torch.float64, device="cuda")
        blest.closeness_from_sums(far, reach, cc)
        assert np.array_equal(cc.cpu().numpy(), cc_w)
        st = g.ms_stats()
        assert st["batches"] == -(-(n - 813) // 64) and st["levels"] >= st["batches"] and st["quads"] >= st["entries"] > 0
        assert st["probes"] >= st["fresh"] > 0 and st["dirty_sets"] > 0


@pytest.mark.parametrize("reorder", ["none", "degree", "rcm"])
def test_level_guess(blest, torch_cuda, reorder):
    """The lazy kernel pre-fills levels_out with the level that discovered the most vertices in an earlier call from a
    source of the same class (and -1 where the traversal cannot reach): right or wrong, the result is the oracle's.
    Sources alternate between hubs, leaves, a far corner of an attached path and other components, so that right
    guesses, wrong guesses and "no guess" (source outside the labelled component) all occur on one handle."""
    torch = torch_cuda
    n, rp, ci = gg.disjoint_union(gg.rmat(12, 12, 77), gg.path(40), gg.star(9, 3), gg.empty(4))
    deg = np.diff(rp.astype(np.int64))
    big = int(np.argmax(deg))
    srcs = [big, int(np.flatnonzero(deg == 1)[0]), 4096 + 39, big, int(np.flatnonzero(deg == 2)[0]), 4096 + 40 + 3, n - 1, big,
            int(np.flatnonzero(deg == 1)[1]), int(np.flatnonzero(deg == 1)[0])]
    for guess in (True, False):
        used = 0
        with blest.Graph(n, rp, ci, kernel="lazy", reorder=reorder, level_guess=guess) as g:
            out = torch.full((n,), 5, dtype=torch.int32, device="cuda")
            for rep in range(2):
                for s in srcs:
                    g.bfs(s, out)
                    assert np.array_equal(out.cpu().numpy(), oracle.bfs(n, rp, ci, s)), (guess, reorder, s)
                    tr = g.trace()
                    used += int(np.any(tr["reserved"] >> 31)) if tr.size else 0
            assert g.last_status() == 0
        assert (used > 0) == guess


@pytest.mark.parametrize("lanes", [1, 2, 3, 8, 16])
def test_ms_concurrent_lanes(blest, torch_cuda, lanes):
    """Closeness / farness calls split their source batches over concurrent cooperative launches (options.tune[3]):
    every lane count gives the oracle's farness / reach / closeness, for all vertices (target-side sums added over the
    lanes), for a source subset (per-source sums, disjoint per lane) and for a source range; the launch totals are sums
    over the lanes."""
    torch = torch_cuda
    n, rp, ci = gg.disjoint_union(gg.rmat(10, 10, 31), gg.grid2d(9, 11), gg.star(40, 1), gg.empty(6))
    far_w, reach_w, cc_w, _ = oracle.closeness(n, rp, ci)
    for kappa, reorder in ((32, "none"), (64, "degree"), (128, "none")):
        with blest.Graph(n, rp, ci, kappa=kappa, reorder=reorder, ms_lanes=lanes) as g:
            far = torch.zeros(n, dtype=torch.int64, device="cuda")
            reach = torch.zeros(n, dtype=torch.int32, device="cuda")
            cc = torch.zeros(n, dtype=torch.float64, device="cuda")
            for _ in range(2):  # twice: the lanes' workspaces are reused
                g.farness(far, reach)
                g.closeness(cc)
                assert np.array_equal(far.cpu().numpy().view(np.uint64), far_w)
                assert np.array_equal(reach.cpu().numpy().view(np.uint32), reach_w)
                assert np.array_equal(cc.cpu().numpy(), cc_w)
            st = g.ms_stats()
            assert st["batches"] == -(-n // kappa) and st["levels"] >= st["batches"]
            sub = np.concatenate([np.arange(5, n, 7), [0, n - 1, 5]]).astype(np.uint32)
            f2, r2 = np.zeros(sub.size, dtype=np.uint64), np.zeros(sub.size, dtype=np.uint32)
            g.farness(f2, r2, srcs=sub)
            assert np.array_equal(f2, far_w[sub]) and np.array_equal(r2, reach_w[sub])
            assert g.ms_stats()["batches"] == -(-sub.size // kappa)
            pf = torch.zeros(n, dtype=torch.int64, device="cuda")
            pr = torch.zeros(n, dtype=torch.int32, device="cuda")
            tot_f, tot_r = torch.zeros_like(pf), torch.zeros_like(pr)
            for first, count in ((0, 333), (333, n - 333)):
                g.farness_partial(first, count, pf, pr)
                tot_f += pf
                tot_r += pr
            assert np.array_equal(tot_f.cpu().numpy().view(np.uint64), far_w)
            assert np.array_equal(tot_r.cpu().numpy().view(np.uint32), reach_w)
            assert g.last_status() == 0


@pytest.mark.parametrize("kappa", [32, 64, 128, 256])
def test_msbfs_pull_levels(blest, torch_cuda, kappa):
    """The pull levels of the multi-source kernel (a batch switches once a level's queue holds half of all VSSs): farness /
    reach / closeness of every vertex bit-equal to the oracle and to the run that never switches (ms_pull=False); the
    level trace shows that the switch happened, and only on the all-vertices path."""
    torch = torch_cuda
    for maker in (lambda: gg.rmat(11, 12, 5), lambda: gg.disjoint_union(gg.rmat(10, 16, 3), gg.star(70, 0), gg.path(9), gg.empty(3)),
                  lambda: gg.grid2d(24, 17), lambda: gg.complete(77)):
        n, rp, ci = maker()
        far_w, reach_w, cc_w, _ = oracle.closeness(n, rp, ci)
        got = {}
        for pull in (True, False):
            for reorder in ("none", "degree"):
                with blest.Graph(n, rp, ci, kappa=kappa, ms_pull=pull, reorder=reorder) as g:
                    far = torch.zeros(n, dtype=torch.int64, device="cuda")
                    reach = torch.zeros(n, dtype=torch.int32, device="cuda")
                    cc = torch.zeros(n, dtype=torch.float64, device="cuda")
                    g.farness(far, reach)
                    ph, tr = g.ms_phases(), g.ms_level_trace()
                    g.closeness(cc)
                    assert g.last_status() == 0
                    assert np.array_equal(far.cpu().numpy().view(np.uint64), far_w), (pull, reorder)
                    assert np.array_equal(reach.cpu().numpy().view(np.uint32), reach_w), (pull, reorder)
                    assert np.array_equal(cc.cpu().numpy(), cc_w), (pull, reorder)
                    got[(pull, reorder)] = ph["pull_levels"]
                    assert (ph["pull_levels"] > 0) == any(r["pull"] for r in tr) or len(tr) == 60
                    if not pull:
                        assert ph["pull_levels"] == 0 and ph["pull_rows"] == 0
                    # a source subset counts per source: that path never pulls
                    sub = np.arange(0, n, 3, dtype=np.uint32)
                    f2, r2 = np.zeros(sub.size, dtype=np.uint64), np.zeros(sub.size, dtype=np.uint32)
                    g.farness(f2, r2, srcs=sub)
                    assert np.array_equal(f2, far_w[sub]) and np.array_equal(r2, reach_w[sub])
                    assert g.ms_phases()["pull_levels"] == 0
        if n >= 1000 and kappa < 256:  # the scale-free graphs reach most slice sets within two levels (kappa = 256 never pulls)
            assert got[(True, "none")] > 0 and got[(True, "degree")] > 0


def test_microbenchmarks_run(blest, torch_cuda):
    assert blest.l2_microbench(32 << 20, 10) > 500.0          # GB/s, L2-resident copy
    assert 200.0 < blest.barrier_microbench(500) < 20000.0     # ns per grid barrier
    for ctas in (1, 2, 8):                                       # thread-block clusters (portable sizes)
        b, d = blest.cluster_microbench(ctas, 500)
        assert 10.0 < b < 20000.0 and 5.0 < d < 20000.0, (ctas, b, d)
    assert blest.mma_microbench("mma_u8", 256)[0] > 10.0


def test_small_graph_suite_under_bounds_asserts():
    """compute-sanitizer is closed on this GPU pool, so the kernels carry their own bounds checks: libblest_debug.so is
    the same source with -DBLEST_DEBUG (a device assert on every queue / list / chunk / bitmap / graph-array index).
    The small and degenerate graphs go through every kernel, forced path, reordering and kappa against it, in a
    subprocess (the library is chosen when it is first loaded); a tripped assert kills the context and fails the run."""
    import os
    import subprocess
    import sys

    code = (
        "import numpy as np, torch, graphgen as gg, oracle, paper_2606_05081_b200 as blest\n"
        "from paper_2606_05081_b200 import binding\n"
        "assert binding.load()._name.endswith('libblest_debug.so')\n"
        "makers = [lambda: gg.path(1000), lambda: gg.star(5000, 17), lambda: gg.complete(130), lambda: gg.gnm(1003, 2500, 7),\n"
        "          lambda: gg.disjoint_union(gg.path(9), gg.empty(5), gg.complete(6), gg.cycle(11)), lambda: gg.grid2d(37, 41, 0.05, 8),\n"
        "          lambda: gg.rmat(12, 16, 9), lambda: gg.path(2), lambda: gg.empty(1), lambda: gg.rmat(15, 16, 4)]\n"
        "opts = [dict(kernel='lazy'), dict(kernel='lazy', reorder='degree'), dict(kernel='lazy', reorder='rcm', persist_l2=False),\n"
        "        dict(kernel='lazy', switching='off'), dict(kernel='lazy', switching='bottom_up'), dict(kernel='lazy', switching='top_down'),\n"
        "        dict(kernel='lazy', switching='slice', contraction='mma_b1'), dict(kernel='eager'), dict(kernel='eager', reorder='jaccard'),\n"
        "        dict(kernel='lazy', switching='off', tma_tiles=True, reorder='degree')]\n"
        "cases = 0\n"
        "for mk in makers:\n"
        "    n, rp, ci = mk()\n"
        "    srcs = sorted({0, n - 1, int(np.argmax(gg.degrees(rp)))})\n"
        "    for o in opts:\n"
        "        with blest.Graph(n, rp, ci, **o) as g:\n"
        "            out = torch.empty(n, dtype=torch.int32, device='cuda')\n"
        "            for s in srcs:\n"
        "                g.bfs(s, out)\n"
        "                assert np.array_equal(out.cpu().numpy(), oracle.bfs(n, rp, ci, s)), (o, s)\n"
        "            assert g.last_status() == 0\n"
        "            cases += 1\n"
        "    if n <= 5000:\n"
        "        for kappa in (32, 64, 128, 256):\n"
        "            with blest.Graph(n, rp, ci, kappa=kappa, reorder='degree') as g:\n"
        "                cc = torch.zeros(n, dtype=torch.float64, device='cuda')\n"
        "                g.closeness(cc)\n"
        "                assert np.array_equal(cc.cpu().numpy(), oracle.closeness(n, rp, ci)[2])\n"
        "                k = min(n, kappa + 3)\n"
        "                ms = np.arange(k, dtype=np.uint32)\n"
        "                lv = torch.empty((k, n), dtype=torch.int32, device='cuda')\n"
        "                g.msbfs(ms, lv)\n"
        "                assert np.array_equal(lv.cpu().numpy(), oracle.msbfs(n, rp, ci, ms))\n"
        "                assert g.last_status() == 0\n"
        "                cases += 1\n"
        "print('debug build ok', cases)\n"
    )
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, BLEST_DEBUG_LIB="1", PYTHONPATH=root)
    r = subprocess.run([sys.executable, "-c", code], env=env, cwd=root, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0 and "debug build ok" in r.stdout, (r.stdout[-500:], r.stderr[-2000:])


@pytest.mark.parametrize("name", ["star_hub", "rmat12", "ragged"])
def test_tma_staged_slice_tiles(blest, torch_cuda, name):
    """options.tune[0]: the balanced phase of the slice path stages its tiles with cp.async.bulk + mbarrier (two stages
    per warp, masks copied from the 16-byte-aligned word below their start).  Same levels; hub slice sets of thousands
    of slices (star, RMAT hubs) cross many tiles and both stage parities."""
    torch = torch_cuda
    graph = SMALL[name]() if name != "rmat12" else gg.rmat(15, 16, 4)
    for opts in (dict(switching="off"), dict(switching="slice", reorder="degree"), dict(switching="auto", reorder="degree")):
        with blest.Graph(*graph, kernel="lazy", tma_tiles=True, **opts) as g:
            check_bfs(blest, torch, g, graph, sources_for(graph[0], graph[1], 3))
            check_bfs(blest, torch, g, graph, sources_for(graph[0], graph[1], 2))   # again: parities carried over calls


# ---- directed graphs (NEXT 4) -------------------------------------------------------------------
def directed_graphs():
    rng = np.random.Generator(np.random.PCG64(38))
    n = 3001
    yield "gnm", gg.from_directed_edges(n, rng.integers(0, n, 9000), rng.integers(0, n, 9000))
    yield "rmat13", gg.rmat_directed(13, 8, 7)
    i = np.arange(999)
    yield "path", gg.from_directed_edges(1000, i, i + 1)                              # 999 levels one way, nothing back
    yield "instar", gg.from_directed_edges(4000, np.arange(1, 4000), np.zeros(3999, int))   # hub of in-degree 3999
    yield "outstar", gg.from_directed_edges(4000, np.zeros(3999, int), np.arange(1, 4000))  # hub slice set, leaves are dead ends
    yield "dag", gg.from_directed_edges(600, rng.integers(0, 300, 2000), rng.integers(300, 600, 2000))  # sources with in-degree 0


@pytest.mark.parametrize("name", ["gnm", "rmat13", "path", "instar", "outstar", "dag"])
def test_directed_graphs_every_path(blest, torch_cuda, name):
    """Levels along the edge direction, bit-exact against the oracle, through every kernel and forced path: top-down reads
    the out-neighbour CSR / the BVSS of A, bottom-up (Alg. 4) the transposed CSR the library builds."""
    torch = torch_cuda
    graph = dict(directed_graphs())[name]
    n, rp, ci = graph
    indeg = np.bincount(ci, minlength=n)
    srcs = sorted({0, n - 1, int(np.argmax(np.diff(rp.astype(np.int64)))), int(np.argmax(indeg)), int(np.argmin(indeg))})
    for opts in (dict(kernel="lazy"), dict(kernel="lazy", reorder="degree"), dict(kernel="lazy", reorder="degree", persist_l2=False),
                 dict(kernel="lazy", switching="off"), dict(kernel="lazy", switching="bottom_up"),
                 dict(kernel="lazy", switching="top_down"), dict(kernel="lazy", switching="scripted", bu_mask=0b10101010),
                 dict(kernel="eager"), dict(kernel="eager", reorder="degree")):
        with blest.Graph(n, rp, ci, directed=True, **opts) as g:
            check_bfs(blest, torch, g, graph, srcs)
            assert g.last_status() == 0


@pytest.mark.parametrize("kappa", [32, 64, 256])
def test_directed_msbfs_and_closeness(blest, torch_cuda, kappa):
    """Multi-source rows = single-source levels; closeness of all vertices on a directed graph counts per source (the
    target-side sums of Eq. 7 would be the IN-farness): bit-equal to the oracle; the partial-sum call is refused."""
    from paper_2606_05081_b200 import binding

    torch = torch_cuda
    n, rp, ci = gg.rmat_directed(10, 8, 3)
    far_w, reach_w, cc_w, _ = oracle.closeness(n, rp, ci)
    for reorder in ("none", "degree"):
        with blest.Graph(n, rp, ci, directed=True, kappa=kappa, reorder=reorder) as g:
            srcs = np.array([0, 5, 5, n - 1, 77] + list(range(100, 100 + kappa)), dtype=np.uint32)
            lv = torch.empty((srcs.size, n), dtype=torch.int32, device="cuda")
            g.msbfs(srcs, lv)
            assert np.array_equal(lv.cpu().numpy(), oracle.msbfs(n, rp, ci, srcs))
            far = torch.zeros(n, dtype=torch.int64, device="cuda")
            reach = torch.zeros(n, dtype=torch.int32, device="cuda")
            g.farness(far, reach)
            assert np.array_equal(far.cpu().numpy().view(np.uint64), far_w)
            assert np.array_equal(reach.cpu().numpy().view(np.uint32), reach_w)
            cc = torch.zeros(n, dtype=torch.float64, device="cuda")
            g.closeness(cc)
            assert np.array_equal(cc.cpu().numpy(), cc_w)
            with pytest.raises(blest.BlestError) as e:
                g.farness_partial(0, 64, far, reach)
            assert e.value.status == binding.EUNSUPPORTED
