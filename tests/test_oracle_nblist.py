"""Pins P12: the neighbour-list side of the oracle --
Hilbert sort key, wrapping, block boxes and the brute-force block-pair set --
against brute force written here in numpy."""
import numpy as np
import pytest

import oracle
from synth_inputs import make_config, tiny_cluster


@pytest.mark.parametrize("b", [1, 2, 3, 4])
def test_hilbert_key_is_a_continuous_bijection(b):
    n = 1 << b
    g = np.stack(np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij"),
                 axis=-1).reshape(-1, 3)
    key = oracle.hilbert_key(g, b)
    assert np.array_equal(np.sort(key), np.arange(n**3))          # bijection
    order = np.argsort(key)
    step = np.abs(np.diff(g[order], axis=0)).sum(axis=1)
    assert np.all(step == 1)                                       # unit steps: a Hilbert curve
    assert np.array_equal(g[order[0]], [0, 0, 0])


def test_hilbert_key_is_hierarchical():
    """Each aligned octant of the grid occupies one contiguous eighth of the curve."""
    b = 4
    n = 1 << b
    g = np.stack(np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij"),
                 axis=-1).reshape(-1, 3)
    key = oracle.hilbert_key(g, b)
    octant = (g[:, 0] >> (b - 1)) * 4 + (g[:, 1] >> (b - 1)) * 2 + (g[:, 2] >> (b - 1))
    top = key >> (3 * (b - 1))
    for o in range(8):
        assert np.unique(top[octant == o]).size == 1


def test_wrap_and_cells():
    L = 18.64
    x = np.array([[-0.1, 0.0, L], [L + 3.0, -L - 1.0, 2 * L - 1e-13], [5.0, 1e-300, -1e-300]])
    w = oracle.wrap(x, L)
    assert np.all((w >= 0) & (w < L))
    np.testing.assert_allclose(w[0], [L - 0.1, 0.0, 0.0], atol=1e-12)
    assert oracle.grid_bits(18.64) == 3 and oracle.grid_bits(61.7) == 5
    assert oracle.grid_bits(99.4) == 6 and oracle.grid_bits(220.1) == 7
    assert oracle.grid_bits(1e6) == 8 and oracle.grid_bits(0.5) == 1
    cells, b = oracle.cell_coords(x, L)
    assert b == 3 and cells.min() >= 0 and cells.max() <= 7
    # the C helper agrees with the numpy wrap
    for v in x.reshape(-1):
        assert oracle.lib().oracle_wrap(float(v), L) == oracle.wrap(np.array([v]), L)[0]


def test_open_boundary_cells_wide_system():
    """Open-boundary branch of cell_coords (Q14) on a system wider than
    2^6 x 2.5 A, where the OPEN_MAX_BITS cap decides the grid: origin = per-axis minimum, one
    extent for all axes = 1.000001 * (largest axis span) + 1e-9, 64 cells per axis.  The expected
    cells are written out by hand for atoms placed at known fractions of the extent."""
    span = 400.0                                     # > 64 * 2.5 = 160 A: uncapped, grid_bits would give 8
    extent = span * 1.000001 + 1e-9
    assert oracle.grid_bits(extent) == 8 and oracle.OPEN_MAX_BITS == 6
    h = extent / 64.0                                # cell edge of the capped grid, 6.25 A
    origin = np.array([-123.0, 7.5, 1000.0])         # an open system sits anywhere
    frac_cells = np.array([[0, 0, 0],                # the three per-axis minima
                           [63, 0, 0],               # x = origin + span: last cell, not 64 (the 1.000001 margin)
                           [0, 31, 0], [0, 32, 0],   # either side of the middle of y
                           [10, 20, 30], [5, 63, 1]])
    pos = origin[None, :] + (frac_cells + 0.5) * h
    pos[0] = origin                                  # exactly on the minimum corner
    pos[1, 0] = origin[0] + span                     # the maximum of the widest axis defines the extent
    pos[5, 1] = origin[1] + 63.25 * h                # y and z spans are shorter than x's: same h on every axis
    cells, b = oracle.cell_coords(pos, 0.0)
    assert b == 6
    np.testing.assert_array_equal(cells, frac_cells)
    # coarser cells, same rule: a translation of the whole system changes no cell
    cells2, b2 = oracle.cell_coords(pos + np.array([1e3, -2e3, 5.0]), 0.0)
    assert b2 == 6
    np.testing.assert_array_equal(cells2, frac_cells)
    # narrower than 160 A the cap is idle: 100 A -> 2^6 cells of 1.5625 A by grid_bits itself, 30 A -> 2^4
    small = np.array([[0.0, 0.0, 0.0], [100.0, 50.0, 25.0]])
    c3, b3 = oracle.cell_coords(small, -1.0)
    assert b3 == 6 and c3[1].tolist() == [63, 31, 15]
    c4, b4 = oracle.cell_coords(small * 0.3, 0.0)
    assert b4 == 4 and c4[1].tolist() == [15, 7, 3]


def _sorted_perm(s):
    key = oracle.sort_keys(s.pos, s.box)
    order = np.lexsort((np.arange(s.n_atoms), key))
    n_b = (s.n_atoms + 31) // 32
    perm = np.full(32 * n_b, -1, dtype=np.int32)
    perm[:s.n_atoms] = order
    return perm


def _boxes_numpy(perm, pos, box):
    n_b = perm.size // 32
    w = oracle.wrap(pos, box)
    c = np.zeros((n_b, 3)); h = np.zeros((n_b, 3))
    for b in range(n_b):
        idx = perm[32 * b:32 * b + 32]
        idx = idx[idx >= 0]
        lo, hi = w[idx].min(axis=0), w[idx].max(axis=0)
        c[b], h[b] = 0.5 * (lo + hi), 0.5 * (hi - lo)
    return c, h


@pytest.mark.parametrize("which", ["cfg0", "tiny_open", "tiny_periodic"])
def test_block_boxes_and_pairs_vs_numpy_bruteforce(which):
    if which == "cfg0":
        s = make_config(0)
    elif which == "tiny_open":
        s = tiny_cluster(97, 5, box=0.0, spread=16.0, cutoff=4.0, skin=1.0)
    else:
        s = tiny_cluster(130, 6, box=15.0, spread=15.0, cutoff=4.0, skin=1.0)
    perm = _sorted_perm(s)
    oracle.check_perm(perm, s.pos, s.box)
    c, h = oracle.block_boxes(perm, s.pos, s.box)
    c2, h2 = _boxes_numpy(perm, s.pos, s.box)
    np.testing.assert_array_equal(c, c2)
    np.testing.assert_array_equal(h, h2)
    reach = s.cutoff + s.skin
    pairs = oracle.block_pairs(perm, s.pos, s.box, reach)
    n_b = c.shape[0]
    want = []
    for I in range(n_b):
        for J in range(I, n_b):
            D = np.abs(c[I] - c[J])
            if s.box > 0:
                D = np.minimum(D, s.box - D)
            gap = np.maximum(0.0, D - (h[I] + h[J]))
            if (gap[0] ** 2 + gap[1] ** 2) + gap[2] ** 2 <= reach * reach:
                want.append((I, J))
    assert np.array_equal(pairs, np.array(want, dtype=np.int32).reshape(-1, 2))
    # every block is its own neighbour; list is strictly lexicographic
    assert np.all(np.any((pairs[:, 0] == pairs[:, 1])[:, None] &
                         (pairs[:, 0][:, None] == np.arange(n_b)[None, :]), axis=0))
    lin = pairs[:, 0].astype(np.int64) * n_b + pairs[:, 1]
    assert np.all(np.diff(lin) > 0)
    # (N iv) atom-level superset property
    assert oracle.atom_pairs_covered(perm, pairs, s.pos, s.box, reach)


def test_superset_check_detects_a_missing_pair():
    s = tiny_cluster(130, 6, box=15.0, spread=15.0, cutoff=4.0, skin=1.0)
    perm = _sorted_perm(s)
    pairs = oracle.block_pairs(perm, s.pos, s.box, s.cutoff + s.skin)
    offdiag = np.nonzero(pairs[:, 0] != pairs[:, 1])[0]
    broken = np.delete(pairs, offdiag[0], axis=0)
    assert not oracle.atom_pairs_covered(perm, broken, s.pos, s.box, s.cutoff + s.skin)


def test_check_perm_rejects_bad_orders():
    s = make_config(0)
    perm = _sorted_perm(s)
    bad = perm.copy()
    bad[[0, 400]] = bad[[400, 0]]
    with pytest.raises(AssertionError):
        oracle.check_perm(bad, s.pos, s.box)
    dup = perm.copy()
    dup[1] = dup[0]
    with pytest.raises(AssertionError):
        oracle.check_perm(dup, s.pos, s.box)
