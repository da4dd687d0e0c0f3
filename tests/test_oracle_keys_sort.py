"""Pins for oracle O1 (box), O2 (Morton keys) and O3 (stable sort).  CPU only."""
import os

import numpy as np
import pytest

import oracle
from helpers import L, decode_key, grid_coords
from paper_2307_06345_b200 import workloads as W


def _read_table(path):
    rows = []
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        x, y, z, k = line.split()
        rows.append((float(x), float(y), float(z), int(k, 8)))
    return rows


def test_box_is_minmax():
    x, y, z = W.plummer(5000, 7)
    b = oracle.box(x, y, z)
    assert b.tolist() == [x.min(), x.max(), y.min(), y.max(), z.min(), z.max()]


def test_box_negative_zero_is_canonical():
    x = np.array([-0.0, -0.0]); y = np.array([0.0, -0.0]); z = np.array([-1.0, -0.0])
    b = oracle.box(x, y, z)
    assert not np.signbit(b[0]) and not np.signbit(b[1]) and not np.signbit(b[5])


def test_box_empty_raises():
    e = np.empty(0)
    with pytest.raises(ValueError):
        oracle.box(e, e, e)


def test_hand_table(golden_dir):
    rows = _read_table(os.path.join(golden_dir, "morton_hand_table.txt"))
    x = np.array([r[0] for r in rows]); y = np.array([r[1] for r in rows]); z = np.array([r[2] for r in rows])
    box6 = np.array([0.0, 1.0, 0.0, 1.0, 0.0, 1.0])
    k = oracle.keys(x, y, z, box6)
    assert [int(v) for v in k] == [r[3] for r in rows]


def test_digit_convention_unit_cells():
    """A3: (1,0,0) -> 4, (0,1,0) -> 2, (0,0,1) -> 1 in the last octal digit."""
    h = 2.0 ** -21
    box6 = np.array([0.0, 1.0] * 3)
    pts = [(1, 0, 0), (0, 1, 0), (0, 0, 1), (1, 1, 1), (1, 0, 1)]
    x = np.array([p[0] * h for p in pts]); y = np.array([p[1] * h for p in pts]); z = np.array([p[2] * h for p in pts])
    assert oracle.keys(x, y, z, box6).tolist() == [4, 2, 1, 7, 5]


def test_decode_encode_identity_exact_box():
    """Box [-4, 4]: extent 8 is a power of two, so (c-lo)/e*2^21 is exact for grid-aligned
    points and exact rational arithmetic gives the grid coordinate for the others."""
    rng = np.random.default_rng(11)
    g = rng.integers(0, 1 << L, size=(2000, 3))
    lo, hi = -4.0, 4.0
    frac = rng.random((2000, 3)) * 0.999
    c = lo + (g + frac) * (8.0 / (1 << L))          # exact: 8/2^21 = 2^-18, sums fit 53 bits
    box6 = np.array([lo, hi] * 3)
    k = oracle.keys(c[:, 0].copy(), c[:, 1].copy(), c[:, 2].copy(), box6)
    for i in range(0, 2000, 7):
        assert decode_key(k[i]) == tuple(grid_coords(c[i], lo, hi))
    dec = np.array([decode_key(v) for v in k])
    assert np.array_equal(dec, g)


def test_upper_edge_clamps_and_keys_below_2_63():
    x, y, z = W.uniform(4096, -1.0, 1.0, 3)
    b = oracle.box(x, y, z)
    k = oracle.keys(x, y, z, b)
    assert int(k.max()) < (1 << 63)
    ix = int(np.argmax(x))
    assert decode_key(k[ix])[0] == (1 << L) - 1      # x == xmax -> 2^21 exactly -> clamped
    iy = int(np.argmin(y))
    assert decode_key(k[iy])[1] == 0


def test_outside_user_box_clamps():
    box6 = np.array([0.0, 1.0] * 3)
    x = np.array([-0.5, 1.5, 0.5]); y = np.array([0.5, 0.5, -3.0]); z = np.array([0.5, 0.5, 9.0])
    dec = [decode_key(v) for v in oracle.keys(x, y, z, box6)]
    assert dec[0][0] == 0 and dec[1][0] == (1 << L) - 1
    assert dec[2][1] == 0 and dec[2][2] == (1 << L) - 1


def test_flat_box_gives_coordinate_zero():
    """A1: hi == lo -> 0/0 -> grid coordinate 0 for that dimension."""
    x = np.array([0.1, 0.9, 0.5]); y = np.full(3, 2.5); z = np.array([0.2, 0.3, 0.4])
    b = oracle.box(x, y, z)
    dec = [decode_key(v) for v in oracle.keys(x, y, z, b)]
    assert all(d[1] == 0 for d in dec)
    assert dec[1][0] == (1 << L) - 1


def test_octal_prefix_is_octree_cell():
    """the first i octal digits of two keys match iff both points lie in the
    same octree node at division level i (brute force over cube membership)."""
    x, y, z = W.blobs(3000, 5, nblobs=20)
    b = np.array([0.0, 1.0] * 3)
    k = oracle.keys(x, y, z, b)
    g = np.stack([np.floor(x * (1 << L)), np.floor(y * (1 << L)), np.floor(z * (1 << L))], 1).astype(np.int64)
    rng = np.random.default_rng(1)
    pairs = rng.integers(0, 3000, size=(4000, 2))
    for lvl in (1, 2, 5, 9, 14, 21):
        sh = L - lvl
        same_cell = np.all((g[pairs[:, 0]] >> sh) == (g[pairs[:, 1]] >> sh), axis=1)
        same_prefix = (k[pairs[:, 0]] >> np.uint64(3 * sh)) == (k[pairs[:, 1]] >> np.uint64(3 * sh))
        assert np.array_equal(same_cell, same_prefix)


def test_rounding_order_division_then_scale():
    """A2: t = fl(fl(c-lo)/e) then *2^21 then floor; checked against exact rationals with the
    two roundings applied explicitly (python floats are IEEE binary64)."""
    rng = np.random.default_rng(5)
    lo, hi = -0.3, 1.7
    e = hi - lo
    c = rng.uniform(lo, hi, 3000)
    box6 = np.array([lo, hi, lo, hi, lo, hi])
    k = oracle.keys(c, c, c, box6)
    for i in range(3000):
        t = (float(c[i]) - lo) / e           # python: one rounding per operation
        g = int(np.floor(t * 2097152.0))
        g = min(max(g, 0), (1 << L) - 1)
        assert decode_key(k[i]) == (g, g, g)


# ---------------------------------------------------------------- O3 sort

def test_sort_matches_library_stable_argsort():
    rng = np.random.default_rng(2)
    k = rng.integers(0, 1 << 63, 20000, dtype=np.uint64)
    k[rng.integers(0, 20000, 5000)] = k[rng.integers(0, 20000, 5000)]     # duplicates
    P, perm = oracle.sort(k)
    ref = np.argsort(k, kind="stable")
    assert np.array_equal(perm, ref.astype(np.uint32))
    assert np.array_equal(P, k[ref])


def test_sort_stability_heavy_duplicates():
    rng = np.random.default_rng(3)
    k = rng.integers(0, 7, 5000, dtype=np.uint64) << np.uint64(40)
    P, perm = oracle.sort(k)
    assert np.all(P[1:] >= P[:-1])
    assert sorted(perm.tolist()) == list(range(5000))
    same = P[1:] == P[:-1]
    assert np.all(perm[1:][same] > perm[:-1][same])
    assert np.array_equal(k[perm], P)


def test_sort_empty_and_single():
    P, perm = oracle.sort(np.empty(0, dtype=np.uint64))
    assert P.size == 0 and perm.size == 0
    P, perm = oracle.sort(np.array([42], dtype=np.uint64))
    assert P.tolist() == [42] and perm.tolist() == [0]
