"""Pins for the CPU oracle (oracle/bfs_oracle.c) against what the paper and the mathematics fix.

None of these re-types the oracle's own formula or re-calls its routine: the expected values are closed
forms, invariants of shortest-path distances, the literal Boolean-semiring recurrence of PAPER.md Eq. 1
executed on bit rows (n <= 64), and a library routine (scipy.sparse.csgraph).  A dropped term, wrong sign,
off-by-one level, transposed operand or wrong sentinel in the oracle fails at least one of them.
"""
import numpy as np
import pytest
import scipy.sparse as sp
import scipy.sparse.csgraph as csg

import graphgen as gg
import oracle


# ---- closed forms (SURVEY.md §8(c) "bfs_oracle levels") ------------------------------------------
@pytest.mark.parametrize("n,s", [(1, 0), (2, 1), (17, 0), (17, 16), (40, 13)])
def test_path(n, s):
    lv = oracle.bfs(*gg.path(n), s)
    assert np.array_equal(lv, np.abs(np.arange(n) - s))


@pytest.mark.parametrize("n,s", [(3, 0), (8, 5), (9, 2), (33, 32)])
def test_cycle(n, s):
    d = np.abs(np.arange(n) - s)
    assert np.array_equal(oracle.bfs(*gg.cycle(n), s), np.minimum(d, n - d))


@pytest.mark.parametrize("a,b,s", [(1, 9, 4), (5, 7, 0), (5, 7, 34), (6, 6, 14), (33, 9, 100)])
def test_grid_is_manhattan(a, b, s):
    r, c = np.divmod(np.arange(a * b), b)
    r0, c0 = divmod(s, b)
    assert np.array_equal(oracle.bfs(*gg.grid2d(a, b), s), np.abs(r - r0) + np.abs(c - c0))


def test_complete_star_tree():
    lv = oracle.bfs(*gg.complete(11), 4)
    exp = np.ones(11, np.int32); exp[4] = 0
    assert np.array_equal(lv, exp)
    lv = oracle.bfs(*gg.star(9, 0), 0)                       # from the centre
    assert lv[0] == 0 and np.all(lv[1:] == 1)
    lv = oracle.bfs(*gg.star(9, 0), 5)                       # from a leaf
    assert lv[5] == 0 and lv[0] == 1 and np.all(np.delete(lv, [0, 5]) == 2)
    n = 100
    lv = oracle.bfs(*gg.binary_tree(n), 0)                   # heap order: depth = floor(log2(i+1))
    assert np.array_equal(lv, np.floor(np.log2(np.arange(n) + 1)).astype(np.int32))


def test_unreachable_is_minus_one():
    g = gg.disjoint_union(gg.path(5), gg.empty(3), gg.cycle(6))
    lv = oracle.bfs(*g, 2)
    assert np.array_equal(lv, [2, 1, 0, 1, 2] + [-1] * 9)
    lv = oracle.bfs(*g, 6)                                   # isolated source
    exp = -np.ones(14, np.int32); exp[6] = 0
    assert np.array_equal(lv, exp)
    lv = oracle.bfs(*g, 8)
    assert np.array_equal(lv[:8], [-1] * 8) and np.array_equal(lv[8:], [0, 1, 2, 3, 2, 1])
    assert lv.dtype == np.int32


# ---- the literal recurrence of PAPER.md Eq. 1 on bit rows, n <= 64 --------------------------------
def eq1_levels(n, rowptr, colidx, src):
    """x(k+1) = (A x(k)) AND NOT v(k) over the Boolean semiring with one Python int per matrix row."""
    rows = [0] * n
    for i in range(n):
        for e in range(int(rowptr[i]), int(rowptr[i + 1])):
            rows[i] |= 1 << int(colidx[e])                   # A[i][j] = 1 iff (j, i) in E; graph is symmetric
    x = 1 << src
    v = x
    level = [-1] * n
    level[src] = 0
    k = 0
    while x:
        nxt = 0
        for i in range(n):
            if (rows[i] & x) != 0 and not (v >> i) & 1:      # popc(a_i AND x) > 0  (Eq. 2), filtered by NOT v
                nxt |= 1 << i
        k += 1
        for i in range(n):
            if (nxt >> i) & 1:
                level[i] = k
        v |= nxt
        x = nxt
    return np.array(level, dtype=np.int32)


@pytest.mark.parametrize("n,m,seed", [(1, 0, 0), (2, 1, 1), (8, 0, 2), (13, 10, 3), (31, 40, 4), (64, 64, 5),
                                      (64, 200, 6), (64, 2016, 7), (50, 25, 8), (64, 40, 9), (33, 500, 10)])
def test_bruteforce_eq1(n, m, seed):
    g = gg.random_graph(n, m, seed)
    for s in sorted({0, n // 2, n - 1}):
        assert np.array_equal(oracle.bfs(*g, s), eq1_levels(*g, s))


def test_bruteforce_eq1_complete_and_empty():
    for g in (gg.complete(64), gg.empty(64), gg.disjoint_union(gg.complete(5), gg.path(7))):
        for s in (0, g[0] - 1):
            assert np.array_equal(oracle.bfs(*g, s), eq1_levels(*g, s))


# ---- invariants of hop distances on any graph ----------------------------------------------------
def check_invariants(n, rowptr, colidx, src, lv):
    assert lv[src] == 0 and np.count_nonzero(lv == 0) == 1
    rows = np.repeat(np.arange(n), np.diff(rowptr.astype(np.int64)))
    lu, lw = lv[rows].astype(np.int64), lv[colidx].astype(np.int64)
    assert np.array_equal(lu < 0, lw < 0)                    # an edge never crosses the reachable set
    ok = lu >= 0
    assert np.all(np.abs(lu[ok] - lw[ok]) <= 1)              # |level(u) - level(v)| <= 1 on every edge
    has_parent = np.zeros(n, bool)
    np.logical_or.at(has_parent, rows[ok & (lw == lu - 1)], True)
    assert np.all(has_parent[lv > 0])                        # every vertex at L > 0 has a neighbour at L-1
    A = sp.csr_matrix((np.ones(colidx.size, np.int8), colidx, rowptr), shape=(n, n))
    _, lab = csg.connected_components(A, directed=False)
    assert np.array_equal(lv >= 0, lab == lab[src])          # reachable set == connected component


@pytest.mark.parametrize("maker", [lambda: gg.rmat(12, 8, 21), lambda: gg.gnm(5000, 6000, 22),
                                   lambda: gg.grid2d(40, 50, 0.2, 23), lambda: gg.rmat(10, 2, 24)])
def test_invariants(maker):
    g = maker()
    for s in gg.pick_sources(g[1], 4, 99, nonzero_degree=False):
        check_invariants(*g, int(s), oracle.bfs(*g, int(s)))


# ---- a library routine on larger inputs ----------------------------------------------------------
@pytest.mark.parametrize("maker", [lambda: gg.rmat(14, 16, 31), lambda: gg.grid2d(128, 96, 0.05, 32),
                                   lambda: gg.gnm(1 << 15, 1 << 17, 33)])
def test_against_scipy(maker):
    n, rp, ci = maker()
    A = sp.csr_matrix((np.ones(ci.size, np.int8), ci, rp), shape=(n, n))
    srcs = gg.pick_sources(rp, 3, 5)
    D = csg.shortest_path(A, method="D", unweighted=True, indices=srcs.astype(np.int64))
    for row, s in zip(D, srcs):
        exp = np.where(np.isinf(row), -1, row).astype(np.int32)
        assert np.array_equal(oracle.bfs(n, rp, ci, int(s)), exp)


# ---- farness / reach / closeness (Eq. 7-8) ----------------------------------------------
def test_farness_closed_forms():
    n = 23
    far, reach, cc, _ = oracle.closeness(*gg.path(n))
    i = np.arange(n)
    assert np.array_equal(far, i * (i + 1) // 2 + (n - 1 - i) * (n - i) // 2)      # P_n from vertex i
    assert np.all(reach == n)
    for m in (8, 9):
        far, reach, cc, _ = oracle.closeness(*gg.cycle(m))
        assert np.all(far == m * m // 4) and np.all(reach == m)                   # C_n: floor(n^2/4)
    far, reach, cc, _ = oracle.closeness(*gg.complete(n))
    assert np.all(far == n - 1) and np.all(cc == 1.0)                             # K_n: closeness exactly 1
    far, reach, cc, _ = oracle.closeness(*gg.star(n, 0))
    assert far[0] == n - 1 and cc[0] == 1.0
    assert np.all(far[1:] == 2 * n - 3) and np.all(cc[1:] == (n - 1) / (2 * n - 3))
    a, b = 6, 9
    far, reach, cc, _ = oracle.closeness(*gg.grid2d(a, b), srcs=[0])
    assert far[0] == a * b * (a + b - 2) // 2                                    # grid from a corner


def test_farness_disconnected_and_isolated():
    g = gg.disjoint_union(gg.path(4), gg.empty(2), gg.complete(5))
    far, reach, cc, used = oracle.closeness(*g)
    assert used >= 1
    assert list(reach) == [4, 4, 4, 4, 1, 1, 5, 5, 5, 5, 5]
    assert list(far) == [6, 4, 4, 6, 0, 0, 4, 4, 4, 4, 4]
    assert cc[4] == 0.0 and cc[5] == 0.0 and cc[0] == 3 / 6 and cc[6] == 1.0
    assert cc.dtype == np.float64 and far.dtype == np.uint64


def test_farness_source_target_symmetry_and_msbfs_rows():
    n, rp, ci = gg.rmat(9, 8, 41)
    srcs = np.arange(n, dtype=np.uint32)
    L = oracle.msbfs(n, rp, ci, srcs)
    for b in (0, 17, n - 1):
        assert np.array_equal(L[b], oracle.bfs(n, rp, ci, b))
    far, reach, cc, _ = oracle.closeness(n, rp, ci)
    Lz = np.where(L < 0, 0, L).astype(np.int64)
    assert np.array_equal(far, Lz.sum(axis=1))
    assert np.array_equal(far, Lz.sum(axis=0))                # undirected: target-side sums equal source-side (R13)
    assert np.array_equal(reach, (L >= 0).sum(axis=1))
    f0, r0 = oracle.farness(L[3])
    assert (f0, r0) == (int(far[3]), int(reach[3]))
    assert oracle.closeness_value(r0, f0) == cc[3]
    sub = np.array([5, 5, 300, 2], dtype=np.uint32)           # duplicates allowed, order preserved
    fs, rs, cs, _ = oracle.closeness(n, rp, ci, sub)
    assert np.array_equal(fs, far[sub]) and np.array_equal(rs, reach[sub]) and np.array_equal(cs, cc[sub])


def test_component_edges():
    g = gg.disjoint_union(gg.path(4), gg.complete(5))
    assert oracle.component_edges(g[1], oracle.bfs(*g, 0)) == 3
    assert oracle.component_edges(g[1], oracle.bfs(*g, 6)) == 10


# ---- directed graphs (A is the TRANSPOSED adjacency matrix; BFS follows the edge direction) ----------
def eq1_levels_directed(n, rowptr, colidx, src):
    """Eq. 1 literally, on a DIRECTED CSR whose row u lists the out-neighbours of u: edge u -> v is A[v][u] = 1."""
    rows = [0] * n
    for u in range(n):
        for e in range(int(rowptr[u]), int(rowptr[u + 1])):
            rows[int(colidx[e])] |= 1 << u
    x = v = 1 << src
    level = [-1] * n
    level[src] = 0
    k = 0
    while x:
        nxt = 0
        for i in range(n):
            if (rows[i] & x) != 0 and not (v >> i) & 1:
                nxt |= 1 << i
        k += 1
        for i in range(n):
            if (nxt >> i) & 1:
                level[i] = k
        v |= nxt
        x = nxt
    return np.array(level, dtype=np.int32)


def test_directed_closed_forms():
    n = 17
    i = np.arange(n - 1)
    dpath = gg.from_directed_edges(n, i, i + 1)                      # 0 -> 1 -> ... -> n-1
    for s in (0, 5, n - 1):
        want = np.where(np.arange(n) >= s, np.arange(n) - s, -1)     # only forward vertices are reachable
        assert np.array_equal(oracle.bfs(*dpath, s), want)
    dcycle = gg.from_directed_edges(n, np.arange(n), (np.arange(n) + 1) % n)
    for s in (0, 9):
        assert np.array_equal(oracle.bfs(*dcycle, s), (np.arange(n) - s) % n)   # one way round, not min of both
    out_star = gg.from_directed_edges(n, np.zeros(n - 1, int), np.arange(1, n))
    assert np.array_equal(oracle.bfs(*out_star, 0), [0] + [1] * (n - 1))
    assert np.array_equal(oracle.bfs(*out_star, 3), [-1] * 3 + [0] + [-1] * (n - 4))     # a leaf reaches nothing
    in_star = gg.from_directed_edges(n, np.arange(1, n), np.zeros(n - 1, int))
    assert np.array_equal(oracle.bfs(*in_star, 3), [1] + [-1] * 2 + [0] + [-1] * (n - 4))
    far, reach, cc, _ = oracle.closeness(*dpath, np.array([0, n - 1], np.uint32))
    assert list(far) == [n * (n - 1) // 2, 0] and list(reach) == [n, 1] and cc[1] == 0.0


@pytest.mark.parametrize("n,m,seed", [(2, 1, 1), (13, 20, 3), (31, 60, 4), (64, 100, 5), (64, 600, 6), (64, 4000, 7), (40, 30, 8)])
def test_directed_bruteforce_eq1(n, m, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    g = gg.from_directed_edges(n, rng.integers(0, n, m), rng.integers(0, n, m))
    for s in sorted({0, n // 2, n - 1}):
        assert np.array_equal(oracle.bfs(*g, s), eq1_levels_directed(*g, s))


def test_directed_against_scipy_and_invariants():
    import scipy.sparse as sp
    from scipy.sparse.csgraph import shortest_path

    n, rp, ci = gg.rmat_directed(12, 8, 21)
    A = sp.csr_matrix((np.ones(ci.size), ci.astype(np.int64), rp.astype(np.int64)), shape=(n, n))
    srcs = [0, 17, n - 1, int(np.argmax(np.diff(rp.astype(np.int64))))]
    d = shortest_path(A, method="D", directed=True, unweighted=True, indices=srcs)
    rows = np.repeat(np.arange(n), np.diff(rp.astype(np.int64)))
    for k, s in enumerate(srcs):
        lv = oracle.bfs(n, rp, ci, s)
        assert np.array_equal(lv, np.where(np.isinf(d[k]), -1, d[k]).astype(np.int32))
        lu, lw = lv[rows].astype(np.int64), lv[ci].astype(np.int64)
        ok = lu >= 0
        assert np.all(lw[ok] >= 0) and np.all(lw[ok] <= lu[ok] + 1)      # u -> w: w is reached, at most one level later
        has_parent = np.zeros(n, bool)
        has_parent[ci[ok & (lw == lu + 1)]] = True
        assert np.all(has_parent[lv > 0])                                # every vertex at L > 0 has an in-neighbour at L-1
