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
