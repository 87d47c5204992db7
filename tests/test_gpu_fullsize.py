"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (same Graph options, same
sources): levels compared element by element with the oracle for a few sources per config (the oracle finishes one
BFS in seconds), plus integer farness / reach of further sources (bit-exact).  Config 5: closeness of ALL vertices on
the GPU, compared on a seeded sample of sources the oracle computes one by one."""
import numpy as np
import pytest

import graphgen as gg
import oracle

pytestmark = pytest.mark.gpu


_CACHE = {}


def config_graph(name):
    """One generated CSR per config for the whole module (config 4 takes 20 s to generate; all four are < 6 GB)."""
    if name not in _CACHE:
        _CACHE[name] = gg.make_config(name)
    return _CACHE[name]

# reorder as in bench.py (REORDER_FOR); number of sources compared element-wise / by (far, reach)
FULL = {
    "c2_grid4096": dict(reorder="none", n_levels=2, n_far=2),
    "c3_gnm25": dict(reorder="none", n_levels=2, n_far=4),
    "c4_rmat24": dict(reorder="degree", n_levels=3, n_far=0),   # all 64 by (far, reach) in the test below
}


@pytest.fixture(scope="module")
def env():
    import torch

    import paper_2606_05081_b200 as blest

    assert torch.cuda.is_available()
    blest.load()
    return torch, blest


@pytest.mark.parametrize("name", sorted(FULL))
def test_full_size_levels_and_farness(env, name):
    torch, blest = env
    cfg = FULL[name]
    n, rp, ci = config_graph(name)
    srcs = gg.config_sources(name, rp)
    out = torch.empty(n, dtype=torch.int32, device="cuda")
    with blest.Graph(n, rp, ci, reorder=cfg["reorder"]) as g:
        for s in srcs[: cfg["n_levels"]]:
            g.bfs(int(s), out)
            got = out.cpu().numpy()
            want = oracle.bfs(n, rp, ci, int(s))
            bad = np.flatnonzero(got != want)
            assert bad.size == 0, f"{name} src {int(s)}: {bad.size} mismatches, first {bad[:5]}"
            g.trace()  # surfaces a work-queue overflow
        more = srcs[cfg["n_levels"]: cfg["n_levels"] + cfg["n_far"]]
        if more.size:
            far_w, reach_w, _, _ = oracle.closeness(n, rp, ci, more)
            for s, fw, rw in zip(more, far_w, reach_w):
                g.bfs(int(s), out)
                lv = out.cpu().numpy()
                far, reach = oracle.farness(lv)  # plain sum / count of the GPU's level array
                assert (far, reach) == (int(fw), int(rw)), f"{name} src {int(s)}"
                assert lv[int(s)] == 0 and lv.min() >= -1
        assert g.last_status() == 0


def test_full_size_c4_all_sources_and_odd_components(env):
    """Config 4 in bench.py's launch configuration: farness / reach of ALL 64 timed sources against the oracle, plus
    sources the seeded draw does not contain: one outside the hub's component (RMAT leaves a few two- and three-vertex
    components) and, with the component pruning switched off, the same sources again."""
    torch, blest = env
    n, rp, ci = config_graph("c4_rmat24")
    srcs = gg.config_sources("c4_rmat24", rp)
    deg = gg.degrees(rp)
    giant = oracle.bfs(n, rp, ci, int(np.argmax(deg))) >= 0
    small = np.flatnonzero(~giant & (deg > 0))                       # vertices of the small components
    assert small.size > 0
    odd = np.array([small[0], small[-1], np.flatnonzero(deg == 0)[0]], dtype=np.uint32)
    all_srcs = np.concatenate([srcs, odd]).astype(np.uint32)
    far_w, reach_w, _, _ = oracle.closeness(n, rp, ci, all_srcs)
    out = torch.empty(n, dtype=torch.int32, device="cuda")
    for prune in (True, False):
        with blest.Graph(n, rp, ci, reorder="degree", prune_components=prune) as g:
            assert (g.info().component_seconds > 0) == prune
            todo = all_srcs if prune else np.concatenate([srcs[:4], odd])
            for s in todo:
                g.bfs(int(s), out)
                lv = out.cpu().numpy()
                i = int(np.flatnonzero(all_srcs == s)[0])
                assert oracle.farness(lv) == (int(far_w[i]), int(reach_w[i])), f"src {int(s)} prune {prune}"
                assert lv[int(s)] == 0 and lv.min() >= -1
            for s in odd[:2]:                                          # element-wise on the small components
                g.bfs(int(s), out)
                assert np.array_equal(out.cpu().numpy(), oracle.bfs(n, rp, ci, int(s)))
            assert g.last_status() == 0


@pytest.mark.parametrize("contraction", ["mma_b1", "mma_u8"])
def test_mma_contraction_forms_on_c4_shrunk(env, contraction):
    """The tensor-core contraction forms inside a traversal of a graph with hub slice sets (config 4 at scale 20),
    slice path forced on every level."""
    torch, blest = env
    n, rp, ci = gg.make_config("c4_rmat24", 4)
    srcs = gg.config_sources("c4_rmat24", rp)[:3]
    out = torch.empty(n, dtype=torch.int32, device="cuda")
    with blest.Graph(n, rp, ci, reorder="degree", switching="off", contraction=contraction) as g:
        for s in srcs:
            g.bfs(int(s), out)
            assert np.array_equal(out.cpu().numpy(), oracle.bfs(n, rp, ci, int(s))), (contraction, int(s))
        assert g.last_status() == 0


def test_full_size_c3_rcm(env):
    """Config 3 'with and without RCM reordering before BVSS build': the reordered run gives the same levels."""
    torch, blest = env
    n, rp, ci = config_graph("c3_gnm25")
    s = int(gg.config_sources("c3_gnm25", rp)[0])
    out = torch.empty(n, dtype=torch.int32, device="cuda")
    with blest.Graph(n, rp, ci, reorder="rcm") as g:
        g.bfs(s, out)
        assert np.array_equal(out.cpu().numpy(), oracle.bfs(n, rp, ci, s))


@pytest.mark.parametrize("kappa", [64, 128, 256])
def test_full_size_c5_closeness_sampled(env, kappa):
    """Config 5: all 262 144 vertices are sources (kappa-wide batches); farness / reach bit-exact and closeness equal to
    the oracle's IEEE division on a seeded sample of 512 sources (incl. isolated vertices), for every width the
    sources-per-second figures are quoted at."""
    torch, blest = env
    n, rp, ci = config_graph("c5_rmat18")
    rng = np.random.Generator(np.random.PCG64(5))
    sample = np.sort(rng.choice(n, size=512, replace=False)).astype(np.uint32)
    far_w, reach_w, cc_w, _ = oracle.closeness(n, rp, ci, sample)
    with blest.Graph(n, rp, ci, kappa=kappa) as g:
        far = torch.zeros(n, dtype=torch.int64, device="cuda")
        reach = torch.zeros(n, dtype=torch.int32, device="cuda")
        g.farness(far, reach)
        cc = torch.zeros(n, dtype=torch.float64, device="cuda")
        g.closeness(cc)
        far_g = far.cpu().numpy().view(np.uint64)
        reach_g = reach.cpu().numpy().view(np.uint32)
        cc_g = cc.cpu().numpy()
        assert g.last_status() == 0
        if kappa == 64:  # a source subset at full size: per-source counts (reading R13)
            sub = sample[:96]
            f2, r2 = np.zeros(sub.size, dtype=np.uint64), np.zeros(sub.size, dtype=np.uint32)
            g.farness(f2, r2, srcs=sub)
            assert np.array_equal(f2, far_w[:96]) and np.array_equal(r2, reach_w[:96])
    assert np.array_equal(far_g[sample], far_w)
    assert np.array_equal(reach_g[sample], reach_w)
    assert np.allclose(cc_g[sample], cc_w, rtol=1e-12, atol=0.0)
    assert np.array_equal(cc_g[sample], cc_w)
    # properties that hold for every source: reach >= 1; far = 0 iff reach = 1; closeness in [0, 1]
    assert reach_g.min() >= 1 and np.array_equal(far_g == 0, reach_g == 1)
    assert cc_g.min() >= 0.0 and cc_g.max() <= 1.0
    # the component sizes agree: every vertex of a component reports the same reach
    lv = oracle.bfs(n, rp, ci, int(sample[np.argmax(reach_w)]))
    comp = lv >= 0
    assert np.all(reach_g[comp] == reach_g[comp][0])


def test_large_directed_rmat(env):
    """A directed graph at a size where every phase of the lazy kernel runs (RMAT scale 21, 16 M directed edges, hub
    slice sets, bottom-up levels over the transposed CSR, degree order): levels of four sources element by element,
    default switch and forced bottom-up."""
    torch, blest = env
    n, rp, ci = gg.rmat_directed(21, 8, 4711)
    outdeg = np.diff(rp.astype(np.int64))
    indeg = np.bincount(ci, minlength=n)
    srcs = [int(np.argmax(outdeg)), int(np.flatnonzero((outdeg > 0) & (indeg == 0))[0]), int(np.flatnonzero(outdeg > 3)[1000]),
            int(np.flatnonzero(outdeg == 0)[0])]
    want = [oracle.bfs(n, rp, ci, s) for s in srcs]
    assert max(int(w.max()) for w in want) >= 4 and min(int((w >= 0).sum()) for w in want) == 1   # deep traversals and a dead end
    out = torch.empty(n, dtype=torch.int32, device="cuda")
    for opts in (dict(reorder="degree"), dict(reorder="none", switching="bottom_up"), dict(reorder="degree", kernel="eager")):
        with blest.Graph(n, rp, ci, directed=True, **opts) as g:
            for s, w in zip(srcs, want):
                g.bfs(s, out)
                got = out.cpu().numpy()
                assert np.array_equal(got, w), (opts, s, int(np.count_nonzero(got != w)))
            assert g.last_status() == 0
