"""The generators emit what every consumer assumes: symmetric, sorted, loop-free, duplicate-free uint32 CSR,
deterministic in the seed and independent of the thread count."""
import numpy as np
import pytest

import graphgen as gg


def check_csr(n, rowptr, colidx):
    assert rowptr.dtype == np.uint32 and colidx.dtype == np.uint32
    assert rowptr.size == n + 1 and rowptr[0] == 0 and rowptr[-1] == colidx.size
    rp = rowptr.astype(np.int64)
    assert np.all(np.diff(rp) >= 0)
    rows = np.repeat(np.arange(n, dtype=np.int64), np.diff(rp))
    cols = colidx.astype(np.int64)
    assert np.all(cols < n) and np.all(cols != rows)            # in range, no self loops
    key = rows * n + cols
    assert np.all(np.diff(key) > 0)                             # rows sorted, no duplicates
    assert np.array_equal(np.sort(cols * n + rows), key)        # structurally symmetric


@pytest.mark.parametrize("maker", [
    lambda: gg.rmat(10, 16, 7), lambda: gg.rmat(8, 4, 3, relabel=False), lambda: gg.grid2d(17, 33, 0.05, 5),
    lambda: gg.grid2d(8, 8), lambda: gg.gnm(1000, 4000, 9), lambda: gg.path(50), lambda: gg.cycle(9),
    lambda: gg.star(12, 3), lambda: gg.complete(13), lambda: gg.binary_tree(31), lambda: gg.empty(5),
    lambda: gg.disjoint_union(gg.path(5), gg.empty(3), gg.cycle(4)),
])
def test_csr_wellformed(maker):
    check_csr(*maker())


def test_deterministic_and_seeded():
    a = gg.rmat(9, 8, 11)
    b = gg.rmat(9, 8, 11)
    c = gg.rmat(9, 8, 12)
    assert np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])
    assert not (np.array_equal(a[1], c[1]) and np.array_equal(a[2], c[2]))


def test_shapes():
    n, rp, ci = gg.grid2d(6, 7)
    assert n == 42 and ci.size == 2 * (6 * 6 + 5 * 7)
    n, rp, ci = gg.grid2d(64, 64, 0.05, 1)
    full = 2 * (64 * 63 * 2)
    assert 0.90 * full < ci.size < 0.99 * full                 # ~5 % of lattice edges deleted
    n, rp, ci = gg.complete(7)
    assert ci.size == 42
    n, rp, ci = gg.rmat(12, 16, 1)
    deg = gg.degrees(rp)
    assert deg.max() > 20 * max(deg.mean(), 1)                  # heavy tail (RMAT a=0.57)
    n, rp, ci = gg.gnm(1 << 12, 1 << 14, 2)
    assert abs(ci.size / n - 8.0) < 0.2                         # average degree 8


def test_sources():
    n, rp, ci = gg.rmat(10, 4, 5)
    s = gg.pick_sources(rp, 64, 6)
    assert s.size == 64 and np.unique(s).size == 64 and np.all(gg.degrees(rp)[s] > 0)
    assert np.array_equal(s, gg.pick_sources(rp, 64, 6))


def test_rmat_quadrant_probabilities_at_every_bit_level():
    """BASELINE.json configs: Graph500 parameters (a, b, c, d) = (0.57, 0.19, 0.19, 0.05) at EVERY one of the `scale`
    recursion levels.  The raw edge list (no relabelling, before clean-up) is drawn directly from the generator and
    the quadrant of each endpoint-bit pair is counted per level; each frequency must sit within 5 standard errors."""
    import ctypes

    scale, m = 14, 1 << 18
    L = gg._load()
    src = np.empty(m, dtype=np.uint32)
    dst = np.empty(m, dtype=np.uint32)
    L.gg_rmat_edges(scale, m, 4242, 0.57, 0.19, 0.19, None, gg._p(src), gg._p(dst))
    want = np.array([0.57, 0.19, 0.19, 0.05])
    for lvl in range(scale):
        ub = (src >> lvl) & 1
        vb = (dst >> lvl) & 1
        freq = np.bincount((ub * 2 + vb).astype(np.int64), minlength=4) / m      # quadrant = (row bit, column bit)
        se = np.sqrt(want * (1 - want) / m)
        assert np.all(np.abs(freq - want) < 5 * se), (lvl, freq)
    # the levels are independent draws: the joint frequency of (a at level 0, a at level 1) is a * a
    both = np.mean((((src | dst) & 3) == 0))
    assert abs(both - 0.57 * 0.57) < 5 * np.sqrt(0.3249 * 0.6751 / m)
