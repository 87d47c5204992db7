"""CPU tests of the library's host logic (no GPU, no compute calls): the C-ABI library loads and exports every symbol
of include/blest.h; the BVSS builder round-trips the CSR edge set and satisfies the paper's structure invariants
(PAPER.md:88-96); reorderings are bijections that preserve the edge set; getVI and the fragB lane set match the
values the paper prints (tests/golden/)."""
import os
import re

import numpy as np
import pytest

import graphgen as gg
import paper_2606_05081_b200 as blest
from paper_2606_05081_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
GOLDEN = os.path.join(ROOT, "tests", "golden")


def golden_ints(name):
    rows = [l for l in open(os.path.join(GOLDEN, name)) if l.strip() and not l.startswith("#")]
    return rows


def test_library_exports_every_declared_symbol():
    L = blest.load()
    header = open(os.path.join(ROOT, "include", "blest.h")).read()
    declared = set(re.findall(r"\b(blest_[a-z_0-9]+)\s*\(", header))
    assert declared, "no declarations parsed"
    assert declared == set(binding.EXPORTS)
    for sym in declared:
        assert hasattr(L, sym), sym


def test_strerror_and_getvi_golden():
    assert blest.strerror(0) == "ok" and "sorted" in blest.strerror(binding.EUNSORTED)
    order = [int(x) for x in golden_ints("getvi_n24.txt")[0].split()]
    rho = 3                                                    # n = 24, sigma = 8
    pos = [blest.get_vi(u, rho) for u in range(24)]
    assert sorted(pos) == list(range(24))                      # bijection on [0, rho * sigma)
    storage = [0] * 24
    for u, p in enumerate(pos):
        storage[p] = u
    assert storage == order                                    # PAPER.md:506 printed layout


def test_fragb_lane_set_golden():
    lanes = [int(x) for x in golden_ints("fragb_lanes.txt")[0].split()]
    assert [t for t in range(32) if t % 9 in (0, 4)] == lanes  # the predicate device_common.cuh uses
    src = open(os.path.join(ROOT, "paper_2606_05081_b200", "csrc", "device_common.cuh")).read()
    assert "lane % 9u" in src and "r9 == 0u" in src and "r9 == 4u" in src


def test_fig1_slice_example_golden():
    cols, front, hit = [f.strip() for f in golden_ints("fig1_slice.txt")[0].split("|")]
    mask = sum(1 << (int(c) - 1) for c in cols.split())        # code order: bit j = j-th column (reading R7)
    alpha = sum(1 << (int(c) - 1) for c in front.split())
    assert ((mask & alpha) != 0) == bool(int(hit))
    assert bin(mask).count("1") == 3 and mask == 0b01001010 and alpha == 0b00000011


def decode_bvss(g):
    """BVSS -> set of (row, column) pairs, plus per-slice-set slice counts."""
    i = g.info()
    setPtr, rowIds, masks = g.array("setPtr"), g.array("rowIds"), g.array("masks")
    mb = masks.view(np.uint8)                                   # little endian: slice c of quad q = byte 4q + c
    assert mb.size == rowIds.size
    set_of_slice = np.repeat(np.arange(i.n_slice_sets, dtype=np.int64), 4 * np.diff(setPtr.astype(np.int64)))
    rows, cols = [], []
    for j in range(8):
        sel = ((mb >> j) & 1).astype(bool)
        rows.append(rowIds[sel].astype(np.int64))
        cols.append(set_of_slice[sel] * 8 + j)
    return np.concatenate(rows), np.concatenate(cols), mb, rowIds, setPtr, set_of_slice


GRAPHS = {
    "rmat10": lambda: gg.rmat(10, 16, 3),
    "grid": lambda: gg.grid2d(19, 23, 0.05, 4),
    "gnm": lambda: gg.gnm(1000, 3000, 5),
    "star_many_vss": lambda: gg.star(1000, 5),                   # one slice set with >> tau slices
    "path_ragged": lambda: gg.path(77),                          # n not a multiple of 8 / 32
    "empty": lambda: gg.empty(13),
    "complete": lambda: gg.complete(70),
    "union": lambda: gg.disjoint_union(gg.path(9), gg.empty(5), gg.complete(6)),
}


@pytest.mark.parametrize("name", sorted(GRAPHS))
@pytest.mark.parametrize("reorder", ["none", "degree", "rcm", "jaccard"])
def test_bvss_roundtrip_and_invariants(name, reorder):
    n, rp, ci = GRAPHS[name]()
    g = blest.Graph(n, rp, ci, host_only=True, reorder=reorder, validate=True)
    i = g.info()
    assert i.n == n and i.nnz == ci.size and i.n_slice_sets == (n + 7) // 8
    # the graph the BVSS encodes is the (relabelled) input graph
    irp, ici = g.array("rowptr"), g.array("colidx")
    if reorder == "none":
        assert np.array_equal(irp, rp) and np.array_equal(ici, ci)
        perm = np.arange(n)
    else:
        perm, iperm = g.array("perm").astype(np.int64), g.array("iperm").astype(np.int64)
        assert np.array_equal(np.sort(perm), np.arange(n)) and np.array_equal(iperm[perm], np.arange(n))  # bijection
        rows_o = np.repeat(np.arange(n), np.diff(rp.astype(np.int64)))
        want = np.sort(perm[rows_o] * n + perm[ci.astype(np.int64)])
        rows_i = np.repeat(np.arange(n), np.diff(irp.astype(np.int64)))
        assert np.array_equal(rows_i * n + ici.astype(np.int64), want)        # same edge set, rows sorted
        if reorder == "degree":
            deg_new = np.diff(irp.astype(np.int64))
            assert np.all(np.diff(deg_new) <= 0)                               # degree-descending
    r, c, mb, rowIds, setPtr, set_of_slice = decode_bvss(g)
    rows_i = np.repeat(np.arange(n), np.diff(irp.astype(np.int64)))
    # round trip: mask bit j of slice (row u) in set s  <=>  A[u][8s + j] = 1
    assert np.array_equal(np.sort(r * n + c), np.sort(rows_i * n + ici.astype(np.int64)))
    assert int(np.unpackbits(mb).sum()) == ci.size                             # sum popc(mask) = nnz
    # structure invariants
    real = mb != 0
    assert int(real.sum()) == i.n_slices
    quads = np.diff(setPtr.astype(np.int64))
    slices_per_set = np.bincount(set_of_slice[real], minlength=i.n_slice_sets)
    assert np.array_equal(quads, (slices_per_set + 3) // 4)                    # padded to a multiple of 4 only
    realPtrs, v2r = g.array("realPtrs").astype(np.int64), g.array("virtualToReal")
    assert realPtrs[0] == 0 and realPtrs[-1] == i.n_vss
    assert np.array_equal(np.diff(realPtrs), (slices_per_set + 127) // 128)    # #VSS of set s; none for empty sets
    assert np.array_equal(v2r, np.repeat(np.arange(i.n_slice_sets), np.diff(realPtrs)))
    key = set_of_slice[real] * n + rowIds[real].astype(np.int64)
    assert np.all(np.diff(key) > 0)                    # rows ascending inside a set, no row twice (reading R8)
    assert np.all(rowIds < n)                          # padding row ids are valid
    pad = ~real
    first_of_set = np.zeros(mb.size, bool)
    first_of_set[setPtr[:-1][quads > 0].astype(np.int64) * 4] = True
    assert not np.any(pad & first_of_set)              # padding only at the tail of a set
    assert abs(i.mask_density - (ci.size / max(i.n_slices, 1))) < 1e-12


def test_udiv_matches_numpy_restatement():
    """U_div (reading R20) recomputed here from the exported arrays with numpy."""
    for maker, reorder in [(lambda: gg.grid2d(40, 40), "none"), (lambda: gg.rmat(11, 8, 9), "none"),
                           (lambda: gg.grid2d(40, 40), "rcm")]:
        g = blest.Graph(*maker(), host_only=True, reorder=reorder)
        i = g.info()
        setPtr, rowIds, mb = g.array("setPtr").astype(np.int64), g.array("rowIds").astype(np.float64), g.array("masks").view(np.uint8)
        realPtrs, v2r = g.array("realPtrs").astype(np.int64), g.array("virtualToReal").astype(np.int64)
        tot = 0.0
        for v in range(i.n_vss):
            s = v2r[v]
            a = (setPtr[s] + 32 * (v - realPtrs[s])) * 4
            b = min(a + 128, setPtr[s + 1] * 4)
            acc, cols = 0.0, 0
            for c in range(4):
                ids = rowIds[a + c:b:4][mb[a + c:b:4] != 0]
                if ids.size:
                    acc += ids.std()
                    cols += 1
            tot += acc / cols if cols else 0.0
        assert i.u_div == pytest.approx(tot / max(i.n_vss, 1), rel=1e-9, abs=1e-9)


def test_rcm_reduces_udiv_on_a_shuffled_grid():
    n, rp, ci = gg.grid2d(64, 64)
    rng = np.random.Generator(np.random.PCG64(1))
    p = rng.permutation(n)
    rows = np.repeat(np.arange(n), np.diff(rp.astype(np.int64)))
    n2, rp2, ci2 = gg.from_edges(n, p[rows].astype(np.uint32), p[ci].astype(np.uint32))
    u0 = blest.Graph(n2, rp2, ci2, host_only=True).info().u_div
    u1 = blest.Graph(n2, rp2, ci2, host_only=True, reorder="rcm").info().u_div
    assert u1 < 0.25 * u0                               # PAPER.md Table 1: RCM tightens row-id clustering


def test_build_rejects_bad_input():
    n, rp, ci = gg.gnm(200, 600, 2)
    bad = ci.copy()
    r = int(np.flatnonzero(np.diff(rp.astype(np.int64)) >= 2)[0])
    bad[rp[r]], bad[rp[r] + 1] = bad[rp[r] + 1], bad[rp[r]]
    with pytest.raises(blest.BlestError) as e:
        blest.Graph(n, rp, bad, host_only=True)
    assert e.value.status == binding.EUNSORTED
    asym = gg.from_edges(4, [0], [1])
    rp2 = np.array([0, 1, 1, 1, 1], np.uint32)                  # edge 0->1 without 1->0
    with pytest.raises(blest.BlestError) as e:
        blest.Graph(4, rp2, np.array([1], np.uint32), host_only=True, validate=True)
    assert e.value.status == binding.ENOTSYM
    with pytest.raises(blest.BlestError) as e:
        blest.Graph(4, rp2, np.array([7], np.uint32), host_only=True)
    assert e.value.status == binding.ENOTSYM                    # column id out of range
    with pytest.raises(blest.BlestError) as e:
        blest.Graph(0, np.zeros(1, np.uint32), np.zeros(0, np.uint32), host_only=True)
    assert e.value.status == binding.ERANGE
    with pytest.raises(blest.BlestError) as e:
        blest.Graph(*asym, host_only=True, kappa=48)
    assert e.value.status == binding.EINVAL
    g = blest.Graph(*asym, host_only=True)
    with pytest.raises(blest.BlestError) as e:                   # host-only handles refuse traversal: no CPU fallback
        g.bfs(0, np.zeros(4, np.int32))
    assert e.value.status == binding.EUNSUPPORTED


def test_jaccard_with_windows_groups_overlapping_columns():
    """PAPER.md §4.1 / Alg. 1: columns whose neighbourhoods overlap end up in the same slice set, so masks get denser.
    Planted case: 64 groups of 8 columns with IDENTICAL neighbourhoods (a complete bipartite block each), ids shuffled.
    Every group must become exactly one slice set (mask density 8 on those sets); plain degree order cannot do that
    (all degrees are equal).  On an RMAT graph the density must not drop below the degree order's."""
    rng = np.random.Generator(np.random.PCG64(11))
    groups, rows_per = 64, 24
    n = groups * 8 + groups * rows_per
    ids = rng.permutation(n)
    src, dst = [], []
    for gidx in range(groups):
        cols = ids[gidx * 8:(gidx + 1) * 8]
        rows = ids[groups * 8 + gidx * rows_per: groups * 8 + (gidx + 1) * rows_per]
        for c in cols:
            src += [c] * rows_per
            dst += list(rows)
    n, rp, ci = gg.from_edges(n, np.array(src, np.uint32), np.array(dst, np.uint32))
    gj = blest.Graph(n, rp, ci, host_only=True, reorder="jaccard")
    perm = gj.array("perm").astype(np.int64)
    for gidx in range(groups):
        cols = ids[gidx * 8:(gidx + 1) * 8]
        assert len(set(perm[cols] // 8)) == 1, "a group of identical columns was split over slice sets"
    dj = gj.info().mask_density
    dd = blest.Graph(n, rp, ci, host_only=True, reorder="degree").info().mask_density
    assert dj > dd and dj > 3.0
    n2, rp2, ci2 = gg.rmat(13, 16, 5)
    d_deg = blest.Graph(n2, rp2, ci2, host_only=True, reorder="degree").info().mask_density
    d_jac = blest.Graph(n2, rp2, ci2, host_only=True, reorder="jaccard").info().mask_density
    assert d_jac >= d_deg


@pytest.mark.parametrize("reorder", ["none", "degree"])
def test_bvss_of_a_directed_graph(reorder):
    """A is the TRANSPOSED adjacency matrix, so an edge u -> v is the non-zero A[v][u]: the slice of row v in
    the slice set of column u.  Decoding the BVSS of a directed CSR must give exactly the edges, as (row = head,
    column = tail) pairs; RCM / Jaccard need a symmetric input and are refused."""
    n, rp, ci = gg.rmat_directed(10, 8, 5)
    g = blest.Graph(n, rp, ci, host_only=True, directed=True, reorder=reorder)
    irp, ici = g.array("rowptr").astype(np.int64), g.array("colidx").astype(np.int64)
    perm = g.array("perm").astype(np.int64) if reorder != "none" else np.arange(n)
    tails_o = np.repeat(np.arange(n), np.diff(rp.astype(np.int64)))
    tails_i = np.repeat(np.arange(n), np.diff(irp))
    assert np.array_equal(np.sort(perm[tails_o] * n + perm[ci.astype(np.int64)]), tails_i * n + ici)   # same directed edges
    r, c, mb, rowIds, setPtr, set_of_slice = decode_bvss(g)
    assert np.array_equal(np.sort(c * n + r), tails_i * n + ici)          # column = tail u, row = head v
    assert not np.array_equal(np.sort(r * n + c), tails_i * n + ici)      # (and not the other way round: the graph is asymmetric)
    assert int(np.unpackbits(mb).sum()) == ci.size
    for bad in ("rcm", "jaccard"):
        with pytest.raises(blest.BlestError):
            blest.Graph(n, rp, ci, host_only=True, directed=True, reorder=bad)
