"""Pins for the oracle functions behind SURVEY 8(f)'s NEXT rows: Hilbert keys (O2h, reading A28), keys of L = 10
octal digits, one round of the distributed build (O11, Eq. 11) and the SFC domain
decomposition (O12, reading A29).  CPU only.  Nothing here comes from the CUDA path."""
import itertools
import os

import numpy as np
import pytest

import oracle
from helpers import check_cornerstone, decode_key
from paper_2307_06345_b200 import workloads as W


# ---- O2h: Hilbert keys -------------------------------------------------------------------------------------------

def _grid(k):
    g = np.arange(1 << k, dtype=np.uint32)
    x, y, z = np.meshgrid(g, g, g, indexing="ij")
    return x.ravel(), y.ravel(), z.ravel()


def test_hilbert_level1_hand_table(golden_dir):
    rows = [tuple(int(v) for v in ln.split()) for ln in open(os.path.join(golden_dir, "hilbert_level1.txt"))
            if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 8
    x, y, z, want = (np.array(c, dtype=np.uint32) for c in zip(*rows))
    assert np.array_equal(oracle.hilbert_from_grid(x, y, z, 1), want.astype(np.uint64))


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5])
def test_hilbert_is_a_bijection_and_consecutive_keys_are_face_neighbours(k):
    """Exhaustive on the 2^k grid: every key of [0, 8^k) occurs once (the curve visits every cell), and the cells of
    keys h, h + 1 differ by one step along one axis (the curve is continuous: what distinguishes a Hilbert curve from
    the Morton Z-curve)."""
    x, y, z = _grid(k)
    h = oracle.hilbert_from_grid(x, y, z, k)
    assert np.array_equal(np.sort(h), np.arange(8 ** k, dtype=np.uint64))
    order = np.argsort(h)
    step = (np.abs(np.diff(x[order].astype(np.int64))) + np.abs(np.diff(y[order].astype(np.int64)))
            + np.abs(np.diff(z[order].astype(np.int64))))
    assert np.all(step == 1)
    assert h[0] == 0 and (x[order][0], y[order][0], z[order][0]) == (0, 0, 0)


def test_hilbert_first_i_digits_name_the_level_i_cell():
    """"Octant by octant": the first i octal digits of a key are the key of the level-i cell that contains
    the point, so Eq. 1's correspondence between digits and octree nodes holds and Secs. 4-5 run unchanged."""
    rng = np.random.default_rng(5)
    g = rng.integers(0, 1 << 21, (3, 20000), dtype=np.uint32)
    full = oracle.hilbert_from_grid(g[0], g[1], g[2], 21)
    assert np.all(full < np.uint64(1 << 63))
    for i in (1, 2, 3, 7, 10, 15, 20):
        sh = 21 - i
        coarse = oracle.hilbert_from_grid(g[0] >> sh, g[1] >> sh, g[2] >> sh, i)
        assert np.array_equal(coarse, full >> np.uint64(3 * sh)), i


def _connected(cells):
    cells = set(cells)
    start = next(iter(cells))
    seen, todo = {start}, [start]
    while todo:
        c = todo.pop()
        for d in range(3):
            for s in (-1, 1):
                nb = list(c); nb[d] += s; nb = tuple(nb)
                if nb in cells and nb not in seen:
                    seen.add(nb); todo.append(nb)
    return len(seen) == len(cells)


def test_hilbert_segments_are_connected_volumes_morton_segments_are_not():
    """"any continuous segment of the curve is mapped to a compact 3D volume, while an interval of Morton
    keys may correspond to disconnected 3D volumes"."""
    k = 4
    x, y, z = _grid(k)
    h = oracle.hilbert_from_grid(x, y, z, k)
    cell_of = {int(key): (int(a), int(b), int(c)) for key, a, b, c in zip(h, x, y, z)}
    rng = np.random.default_rng(9)
    for _ in range(60):
        a, b = sorted(rng.integers(0, 8 ** k, 2))
        if a == b:
            continue
        assert _connected([cell_of[i] for i in range(a, b)])
    # the Morton interval [3, 5) = cells (0,1,1) and (1,0,0) is not connected (keys decoded by the independent helper)
    assert not _connected([tuple(c >> 20 for c in decode_key(m << 60)) for m in (3, 4)])


def test_hilbert_keys_use_the_grid_coordinates_of_the_morton_keys():
    """orc_hilbert_keys = the Hilbert encoding applied to O2's grid coordinates (the pinned clamp(floor(...)) formula):
    decode the Morton key of every particle with the independent helper and encode those grid points."""
    x, y, z = W.plummer(3000, 77)
    box = oracle.box(x, y, z)
    morton = oracle.keys(x, y, z, box)
    g = np.array([decode_key(m) for m in morton], dtype=np.uint32)
    assert np.array_equal(oracle.hilbert_keys(x, y, z, box), oracle.hilbert_from_grid(g[:, 0], g[:, 1], g[:, 2], 21))


def test_hilbert_tree_counts_match_brute_force_cube_membership():
    x, y, z = W.blobs(4000, 3, nblobs=5)
    t = oracle.full_build(x, y, z, 16, curve="hilbert")
    K, counts = t["leaves"], t["counts"]
    levels = check_cornerstone(K)
    assert int(counts.sum()) == x.size
    morton = oracle.keys(x, y, z, t["box"])
    g = np.array([decode_key(m) for m in morton], dtype=np.uint32)
    for i in np.random.default_rng(0).choice(len(levels), 80, replace=False):
        lv = levels[i]
        if lv == 0:
            continue
        cell = oracle.hilbert_from_grid(g[:, 0] >> (21 - lv), g[:, 1] >> (21 - lv), g[:, 2] >> (21 - lv), lv)
        assert int((cell == (K[i] >> np.uint64(3 * (21 - lv)))).sum()) == int(counts[i])


# ---- L = 10: 30-bit keys ------------------------------------------------------------------------------

def test_hilbert_node_cells_invert_the_key_encoding():
    """O8h walks the curve backwards.  Pin: for random cells of the 2^m grid, the cell decoded from the placeholder-bit
    key (1 followed by the m Hilbert digits of the cell, O2h) is that cell again; with the box [0, 2^m]^3 its centre is
    (g + 0.5) and its half size 0.5 exactly."""
    rng = np.random.default_rng(11)
    for m in (1, 2, 3, 5, 8, 13, 21):
        g = rng.integers(0, 1 << m, (3, 4000), dtype=np.uint32)
        h = oracle.hilbert_from_grid(g[0], g[1], g[2], m)
        prefixes = h | (np.uint64(1) << np.uint64(3 * m))
        box = np.array([0.0, float(1 << m)] * 3)
        c, half = oracle.node_geometry(prefixes, box, curve="hilbert")
        for d in range(3):
            assert np.array_equal(c[d], g[d].astype(np.float64) + 0.5), (m, d)
        assert np.all(half == 0.5)
    c, half = oracle.node_geometry(np.array([1], dtype=np.uint64), np.array([-1.0, 3.0, 0.0, 2.0, 5.0, 6.0]), curve="hilbert")
    assert c[:, 0].tolist() == [1.0, 1.0, 5.5] and half[:, 0].tolist() == [2.0, 1.0, 0.5]          # the root is the box


def test_hilbert_node_cells_contain_their_particles_and_children_tile_parents():
    """Every particle lies in the cell of the leaf that holds it, and the 8 children of an internal node are the 8
    octants of its cell (in the curve's order, not in Morton order): the geometry belongs to the tree of Hilbert keys."""
    x, y, z = W.plummer(20_000, W.BASE_SEED + 77)
    r = oracle.full_build(x, y, z, 16, curve="hilbert")
    c, h = oracle.node_geometry(r["prefixes"], r["box"], curve="hilbert")
    xs = [a[r["perm"]] for a in (x, y, z)]
    leaf_nodes = r["leafToNode"]
    node_of_particle = np.repeat(leaf_nodes, r["counts"])
    for d in range(3):
        lo, hi = c[d] - h[d], c[d] + h[d]
        eps = 1e-9 * (r["box"][2 * d + 1] - r["box"][2 * d])
        assert np.all(xs[d] >= lo[node_of_particle] - eps) and np.all(xs[d] <= hi[node_of_particle] + eps), d
    internal = np.nonzero(r["childOffsets"])[0]
    for i in internal[:: max(1, internal.size // 300)]:
        kids = r["childOffsets"][i] + np.arange(8)
        octants = set()
        for k in kids:
            assert np.allclose(h[:, k], 0.5 * h[:, i], rtol=1e-12)
            octants.add(tuple(bool(c[d, k] > c[d, i]) for d in range(3)))
            assert np.all(np.abs(c[:, k] - c[:, i]) <= 0.5000001 * h[:, i])
        assert len(octants) == 8


def test_keys_with_10_levels_are_the_top_10_digits_of_the_21_level_keys():
    """floor(t 2^10) = floor(floor(t 2^21) / 2^11) for every t >= 0 (scaling by a power of two is exact), and the clamps
    agree, so the 30-bit key is the 63-bit key shifted right by 33 bits -- for Morton and for Hilbert keys."""
    x, y, z = W.plummer(20000, 11)
    x[0], y[0], z[0] = x.max(), y.min(), z.max()                  # c == hi: clamped to 2^L - 1 on both sides
    box = oracle.box(x, y, z)
    k21, h21 = oracle.keys(x, y, z, box), oracle.hilbert_keys(x, y, z, box)
    with oracle.key_levels(10):
        k10, h10 = oracle.keys(x, y, z, box), oracle.hilbert_keys(x, y, z, box)
    assert np.array_equal(k10, k21 >> np.uint64(33))
    assert np.array_equal(h10, h21 >> np.uint64(33))
    assert int(k10.max()) < 1 << 30
    assert oracle.L == 21 and oracle.KEY_END == 1 << 63           # the setting does not leak


def test_tree_with_10_levels_is_the_21_level_tree_of_the_embedded_keys_cut_at_depth_10():
    x, y, z = W.blobs(30000, 21, nblobs=8)
    box = oracle.box(x, y, z)
    with oracle.key_levels(10):
        P10, _ = oracle.sort(oracle.keys(x, y, z, box))
        K10, c10 = oracle.leaves_topdown(P10, 8)
        Kit, cit, rounds, conv = oracle.leaves_iterative(P10, 8)
        t10 = oracle.link(K10)
        f10, n10 = oracle.node_counts(c10, t10)
    assert int(K10[0]) == 0 and int(K10[-1]) == 1 << 30 and int(c10.sum()) == x.size
    assert np.array_equal(K10, Kit) and np.array_equal(c10, cit) and conv and rounds <= 11   # at most L + 1 rounds
    delta10 = np.diff(K10)
    assert np.all((c10 <= 8) | (delta10 == 1))
    assert np.any((c10 > 8) & (delta10 == 1))                     # the clustered input does pile up at depth 10
    # the same particles with 21 levels: the leaves above depth 10 coincide, the deeper ones refine depth-10 cells
    K21, c21 = oracle.leaves_topdown(P10 << np.uint64(33), 8)
    shallow = np.diff(K21) >= np.uint64(1 << 33)
    assert np.all(np.isin(K21[:-1][shallow] >> np.uint64(33), K10[:-1]))
    assert set((K21[:-1] >> np.uint64(33)).tolist()) == set(K10[:-1].tolist())
    # links: same prefixes as linking the embedded leaves with 21 levels (a prefix holds only the leading digits)
    t21 = oracle.link(K10 << np.uint64(33))
    for k in ("prefixes", "levels", "childOffsets", "parents", "leafToNode", "nodeToLeaf"):
        assert np.array_equal(t10[k], t21[k]), k
    assert np.array_equal(t10["levelRange"][:12], t21["levelRange"][:12])
    assert f10[0] == 0 and n10[0] == x.size


# ---- O11: one round of the distributed build ------------------------------------------------------------------------

def _sharded_keys(n, R, seed):
    x, y, z = W.blobs(n, seed, nblobs=6)
    box = oracle.box(x, y, z)
    keys = oracle.keys(x, y, z, box)
    owner = np.random.default_rng(seed).integers(0, R, n)         # "distributed arbitrarily" over the ranks
    shards = [np.sort(keys[owner == r]) for r in range(R)]
    return shards, np.sort(keys)


@pytest.mark.parametrize("R", [1, 2, 5])
def test_global_round_equals_the_round_on_the_union(R):
    """f_glob = f_r o f (Eq. 11): summing the per-rank histograms gives the histogram of the union, so every round, and
    hence the converged array, equals the single-rank one: "identically replicate ... the octree that arises from the
    globally unified set of particles"."""
    shards, union = _sharded_keys(20000, R, 40 + R)
    K = np.array([0, 1 << 63], dtype=np.uint64)
    for r in range(30):
        g = oracle.global_round(shards, K, 32)
        s = oracle.round_(union, K, 32)
        for k in ("N", "O", "Oprime", "K"):
            assert np.array_equal(g[k], s[k]), (r, k)
        if np.all(g["O"] == 1):
            break
        K = g["K"]
    Ktd, ctd = oracle.leaves_topdown(union, 32)
    assert np.array_equal(K, Ktd) and np.array_equal(g["N"], ctd)


def test_global_round_with_an_empty_rank_and_unequal_shards():
    shards, union = _sharded_keys(5000, 3, 8)
    shards = [shards[0], np.empty(0, dtype=np.uint64), np.concatenate(shards[1:])]
    shards[2].sort()
    K, _ = oracle.leaves_topdown(union[::3], 16)                   # some valid array that is not the fixpoint
    g, s = oracle.global_round(shards, K, 16), oracle.round_(union, K, 16)
    for k in ("N", "O", "Oprime", "K"):
        assert np.array_equal(g[k], s[k]), k


# ---- O12: SFC domain decomposition ------------------------------------------------------------------------------------

def test_partition_special_cases():
    assert oracle.partition(np.full(12, 5), 4).tolist() == [0, 3, 6, 9, 12]       # equal counts: equal bins
    assert oracle.partition(np.array([3, 1, 4, 1, 5]), 1).tolist() == [0, 5]
    assert oracle.partition(np.array([10, 0, 0, 0]), 2).tolist() == [0, 1, 4]      # first boundary AT OR PAST the split
    assert oracle.partition(np.array([1, 1, 1, 1]), 2).tolist() == [0, 2, 4]       # ... "at" counts
    assert oracle.partition(np.array([0, 0, 0]), 3).tolist() == [0, 0, 0, 3]       # no particles: the ideal split is 0


@pytest.mark.parametrize("R", [2, 3, 8, 64])
def test_partition_is_the_first_boundary_past_each_ideal_split(R):
    rng = np.random.default_rng(R)
    N = rng.integers(0, 200, 5000).astype(np.uint32)
    N[rng.integers(0, N.size, 300)] = 0
    b = oracle.partition(N, R).astype(np.int64)
    C = np.concatenate([[0], np.cumsum(N.astype(np.int64))])
    total = int(C[-1])
    assert b[0] == 0 and b[-1] == N.size and np.all(np.diff(b) >= 0)
    for r in range(1, R):
        assert C[b[r]] * R >= r * total                           # at or past the ideal split r N_tot / R ...
        assert b[r] == 0 or C[b[r] - 1] * R < r * total           # ... and the first such boundary
    # hence every bin holds N_tot / R up to one leaf: "approximately N_tot / n_ranks"
    per_bin = np.diff(C[b])
    assert np.all(np.abs(per_bin - total / R) < N.max() + 1)
