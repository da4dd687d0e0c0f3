"""Pins for oracle O4/O5 (cornerstone leaves), O6 (linked octree), O7 (node counts).  CPU only.

Each test ties the oracle to something other than itself: values the paper prints
(Fig. 1/2, Table 1's tree size), invariants it states (Eq. 2, balance, n_i = (n_l-1)/7),
closed forms, library routines (numpy searchsorted), or brute force on tiny inputs.
"""
import os

import numpy as np
import pytest

import oracle
from helpers import KEY_END, L, check_cornerstone, decode_key, random_octree
from paper_2307_06345_b200 import workloads as W


def _sorted_keys(x, y, z):
    b = oracle.box(x, y, z)
    P, _ = oracle.sort(oracle.keys(x, y, z, b))
    return P


def _read_golden(path):
    sec, cur = {}, None
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        if line.startswith("["):
            cur = line[1:-1]
            sec[cur] = []
        else:
            sec[cur].extend(line.split())
    return sec


SETS = {
    "uniform": lambda n, s: W.uniform(n, 0.0, 1.0, s),
    "plummer": lambda n, s: W.plummer(n, s),
    "blobs": lambda n, s: W.blobs(n, s, nblobs=30),
}


# ------------------------------------------------------------------ O4: invariants

@pytest.mark.parametrize("kind", list(SETS))
@pytest.mark.parametrize("bucket", [1, 16, 64])
def test_leaves_invariants(kind, bucket):
    x, y, z = SETS[kind](20000, 17)
    P = _sorted_keys(x, y, z)
    K, cnt = oracle.leaves_topdown(P, bucket)
    levels = check_cornerstone(K)                               # Eq. 2 + alignment
    nl = K.size - 1
    assert int(cnt.sum()) == P.size                             # leaf counts sum to N
    delta = (K[1:] - K[:-1])
    assert np.all((cnt <= bucket) | (delta == 1))               # PAPER.md:68, A7
    assert (nl - 1) % 7 == 0
    # counts equal the library lower_bound differences (Eq. 3, reading A6)
    off = np.searchsorted(P, K, side="left")
    assert np.array_equal(np.diff(off).astype(np.uint32), cnt)
    # balanced: every internal node holds more than bucket particles
    tree = oracle.link(K)
    first, count = oracle.node_counts(cnt, tree)
    internal = tree["childOffsets"] != 0
    assert np.all(count[internal] > bucket)
    assert len(levels) == nl


def test_config1_closed_form():
    """N=65536 uniform, bucket 64: level-3 cells hold ~128 (all split), level-4 cells ~16
    (none above 64) -> exactly 8^4 = 4096 leaves, all at level 4; 5 rounds from the root."""
    cfg = W.CONFIGS[0]
    x, y, z = cfg.generate()
    P = _sorted_keys(x, y, z)
    K, cnt = oracle.leaves_topdown(P, 64)
    assert K.size - 1 == 4096
    assert set(check_cornerstone(K)) == {4}
    K2, cnt2, rounds, conv = oracle.leaves_iterative(P, 64)
    assert conv and rounds == 5
    assert np.array_equal(K, K2) and np.array_equal(cnt, cnt2)


def test_brute_force_cube_membership():
    """Tiny input: decode each leaf's (level, ix, iy, iz) from K_i and count the particles
    whose integer grid coordinates fall in that cube."""
    x, y, z = W.blobs(800, 23, nblobs=5)
    box6 = np.array([0.0, 1.0] * 3)
    k = oracle.keys(x, y, z, box6)
    P, _ = oracle.sort(k)
    g = np.stack([np.floor(x * (1 << L)), np.floor(y * (1 << L)), np.floor(z * (1 << L))], 1).astype(np.int64)
    g = np.clip(g, 0, (1 << L) - 1)
    for bucket in (1, 4, 16):
        K, cnt = oracle.leaves_topdown(P, bucket)
        levels = check_cornerstone(K)
        total = 0
        for i, lv in enumerate(levels):
            cx, cy, cz = decode_key(K[i])
            sh = L - lv
            inside = np.all((g >> sh) == np.array([cx >> sh, cy >> sh, cz >> sh]), axis=1)
            assert int(inside.sum()) == int(cnt[i])
            total += int(cnt[i])
        assert total == 800


# ------------------------------------------------------------------ O5: the paper's iteration

@pytest.mark.parametrize("kind", list(SETS))
@pytest.mark.parametrize("bucket", [1, 16, 64])
def test_iteration_reaches_topdown(kind, bucket):
    x, y, z = SETS[kind](6000, 29)
    P = _sorted_keys(x, y, z)
    K, cnt = oracle.leaves_topdown(P, bucket)
    K2, cnt2, rounds, conv = oracle.leaves_iterative(P, bucket)
    assert conv and rounds <= L + 1                              # PAPER.md:126, A12
    assert np.array_equal(K, K2) and np.array_equal(cnt, cnt2)
    # a converged array is a fixpoint of one more round with O all ones
    r = oracle.round_(P, K, bucket)
    assert np.all(r["O"] == 1) and np.array_equal(r["K"], K)
    assert np.array_equal(r["N"], cnt)
    assert np.array_equal(r["Oprime"], np.arange(K.size, dtype=np.uint32))


def test_fig1_single_split(golden_dir):
    """PAPER.md:124 (Fig. 1): only the third octant holds more than Ncrit particles, so one
    f+g round replaces it by its 8 children and yields the lower panel's array."""
    gold = _read_golden(os.path.join(golden_dir, "fig2_linked_octree.txt"))
    top = np.array([int(v, 8) for v in gold["cornerstone_top"]], dtype=np.uint64)
    want = np.array([int(v, 8) for v in gold["cornerstone"]], dtype=np.uint64)
    d = 8 ** 20
    # 2 particles per octant, 5 in the third octant spread over its children; bucket 4
    P = []
    for o in range(8):
        P += [o * d + 1, o * d + 2]
    P += [2 * d + c * (d // 8) + 5 for c in (0, 3, 7)]
    P = np.sort(np.array(P, dtype=np.uint64))
    r = oracle.round_(P, top, 4)
    assert r["O"].tolist() == [1, 1, 8, 1, 1, 1, 1, 1]
    assert r["Oprime"].tolist() == [0, 1, 2, 10, 11, 12, 13, 14, 15]   # Eq. 6
    assert np.array_equal(r["K"], want)
    assert want.size - 1 == int(gold["num_leaves"][0])


def test_merge_threshold_is_le():
    """A8: 8 particles, one per octant, Ncrit = 8: from the 8-children array the siblings
    must merge back into the root (combined count == Ncrit), as the balance definition
    (leaves <= Ncrit) demands; from the root it stays the root."""
    d = 8 ** 20
    P = np.array([o * d + 3 for o in range(8)], dtype=np.uint64)
    K8 = np.array([o * d for o in range(8)] + [KEY_END], dtype=np.uint64)
    r = oracle.round_(P, K8, 8)
    assert r["O"].tolist() == [1, 0, 0, 0, 0, 0, 0, 0]
    assert r["K"].tolist() == [0, KEY_END]
    K, cnt, rounds, conv = oracle.leaves_iterative(P, 8, K_start=K8)
    assert K.tolist() == [0, KEY_END] and cnt.tolist() == [8] and conv
    K, cnt = oracle.leaves_topdown(P, 8)
    assert K.tolist() == [0, KEY_END]
    # one more particle -> 9 > 8 -> stays split
    P9 = np.sort(np.append(P, np.uint64(5)))
    r = oracle.round_(P9, K8, 8)
    assert np.all(r["O"] == 1)


def test_max_depth_duplicates():
    """A7: 500 copies of each of 3 points, Ncrit 64 -> leaves at level 21 holding 500."""
    pts = np.array([0o123456712345671234567, 0o123456712345671234570, 0o700000000000000000001], dtype=np.uint64)
    P = np.sort(np.repeat(pts, 500))
    K, cnt = oracle.leaves_topdown(P, 64)
    lv = check_cornerstone(K)
    assert sorted(cnt[cnt > 0].tolist()) == [500, 500, 500]
    assert max(lv) == L
    assert np.all((cnt <= 64) | ((K[1:] - K[:-1]) == 1))
    K2, cnt2, rounds, conv = oracle.leaves_iterative(P, 64)
    assert conv and rounds == L + 1 and np.array_equal(K, K2)


def test_incremental_from_previous_leaves():
    """keep K balanced by updating the previous step's array; A13: iterating
    from any valid previous K gives the from-scratch tree."""
    x, y, z = W.plummer(30000, 31)
    P0 = _sorted_keys(x, y, z)
    K0, _ = oracle.leaves_topdown(P0, 32)
    x1, y1, z1 = W.displace(x, y, z, 1e-3, 99)
    P1 = _sorted_keys(x1, y1, z1)
    K1, cnt1 = oracle.leaves_topdown(P1, 32)
    K1i, cnt1i, rounds, conv = oracle.leaves_iterative(P1, 32, K_start=K0)
    assert conv and rounds <= 4
    assert np.array_equal(K1, K1i) and np.array_equal(cnt1, cnt1i)
    # paper's single-update mode (maxRounds = 1) returns a valid cornerstone array
    K1s, cnt1s, r1, conv1 = oracle.leaves_iterative(P1, 32, K_start=K0, max_rounds=1)
    assert r1 == 1
    check_cornerstone(K1s)
    assert int(cnt1s.sum()) == P1.size
    # from a badly wrong previous tree (different distribution) it still converges to the same
    xu, yu, zu = W.uniform(30000, 0.0, 1.0, 5)
    Ku, _ = oracle.leaves_topdown(_sorted_keys(xu, yu, zu), 8)
    K1u, cnt1u, rounds_u, conv_u = oracle.leaves_iterative(P1, 32, K_start=Ku)
    assert conv_u and rounds_u <= L + 1 and np.array_equal(K1, K1u)


def test_gaussian_tree_size_matches_table1():
    """PAPER.md:168 (Table 1): 1 million particles, 3D Gaussian density, Ncrit = 64 ->
    55.8K leaves.  Statistical pin (different random numbers, box = particle min/max)."""
    x, y, z = W.gaussian(1_000_000, 41)
    P = _sorted_keys(x, y, z)
    K, cnt = oracle.leaves_topdown(P, 64)
    nl = K.size - 1
    assert abs(nl - 55800) / 55800 < 0.05, nl


def test_empty_particle_set():
    K, cnt = oracle.leaves_topdown(np.empty(0, dtype=np.uint64), 64)
    assert K.tolist() == [0, KEY_END] and cnt.tolist() == [0]
    K, cnt, rounds, conv = oracle.leaves_iterative(np.empty(0, dtype=np.uint64), 64)
    assert K.tolist() == [0, KEY_END] and cnt.tolist() == [0] and rounds == 1 and conv


# ------------------------------------------------------------------ O6: linked octree

def test_fig2_golden(golden_dir):
    gold = _read_golden(os.path.join(golden_dir, "fig2_linked_octree.txt"))
    K = np.array([int(v, 8) for v in gold["cornerstone"]], dtype=np.uint64)
    t = oracle.link(K)
    assert t["numNodes"] == int(gold["num_nodes"][0]) == 17
    assert t["levelRange"].tolist() == [int(v) for v in gold["level_offsets"]]
    assert [int(v) for v in t["prefixes"]] == [int(v, 8) for v in gold["node_keys"]]
    assert t["childOffsets"].tolist() == [int(v) for v in gold["child_offsets"]]
    assert t["parents"].tolist() == [0] + [0] * 8 + [3] * 8
    assert t["levels"].tolist() == [0] + [1] * 8 + [2] * 8
    # red line of Fig. 2: leaves in cornerstone order
    assert t["leafToNode"].tolist() == [1, 2, 9, 10, 11, 12, 13, 14, 15, 16, 4, 5, 6, 7, 8]


def _internal_nodes_by_paper_step2(K):
    """PAPER.md:157 (step 2), reading A17: d = number of common leading bits of K_i and
    K_{i+1} in the 63-bit key; if d mod 3 == 0, the first d bits of K_i are an internal
    node at level d/3.  Returns the set of placeholder-bit keys."""
    out = set()
    Kp = [int(v) for v in K]
    for a, b in zip(Kp[:-2], Kp[1:-1]):
        xr = a ^ b
        d = 63 - xr.bit_length()
        if d % 3 == 0:
            lvl = d // 3
            out.add((1 << (3 * lvl)) | (a >> (3 * (L - lvl))))
    return out


@pytest.mark.parametrize("seed", range(8))
def test_link_invariants_random_octrees(seed):
    import random
    rng = random.Random(seed)
    K = random_octree(rng, max_leaves=50 + 200 * seed, max_level=3 + seed)
    nl = K.size - 1
    t = oracle.link(K)
    n = t["numNodes"]
    ni = (nl - 1) // 7
    assert n == nl + ni
    pre = [int(v) for v in t["prefixes"]]
    assert all(a < b for a, b in zip(pre[:-1], pre[1:]))          # "radix sort NK"
    co = t["childOffsets"]; par = t["parents"]; lev = t["levels"]
    assert int((co != 0).sum()) == ni
    for i in range(n):
        assert pre[i].bit_length() == 3 * int(lev[i]) + 1         # placeholder bit
        if co[i]:
            for c in range(8):
                assert pre[co[i] + c] == (pre[i] << 3) | c
                assert par[co[i] + c] == i
    # LO: first node of each level, n beyond the deepest level (A19)
    lr = t["levelRange"]
    for l in range(L + 2):
        idx = np.flatnonzero(lev == l)
        deeper = np.flatnonzero(lev >= l)
        assert lr[l] == (idx[0] if idx.size else (deeper[0] if deeper.size else n))
    # leaves visited in leafToNode order reproduce K
    for j in range(nl):
        i = int(t["leafToNode"][j])
        assert co[i] == 0 and t["nodeToLeaf"][i] == j
        l = int(lev[i])
        start = (pre[i] ^ (1 << (3 * l))) << (3 * (L - l))
        assert start == int(K[j]) and start + 8 ** (L - l) == int(K[j + 1])
    assert np.all(t["nodeToLeaf"][co != 0] == 0xFFFFFFFF)
    # the internal nodes are exactly those of the paper's step 2
    assert _internal_nodes_by_paper_step2(K) == {pre[i] for i in range(n) if co[i]}


def test_link_root_only():
    t = oracle.link(np.array([0, KEY_END], dtype=np.uint64))
    assert t["numNodes"] == 1 and t["prefixes"].tolist() == [1] and t["childOffsets"].tolist() == [0]
    assert t["levelRange"].tolist() == [0] + [1] * 22
    assert t["leafToNode"].tolist() == [0] and t["nodeToLeaf"].tolist() == [0] and t["parents"].tolist() == [0]


def test_link_rejects_non_octree():
    with pytest.raises(ValueError):
        oracle.link(np.array([0, 8 ** 20, KEY_END], dtype=np.uint64))


# ------------------------------------------------------------------ O7: node counts

@pytest.mark.parametrize("kind", list(SETS))
def test_node_counts(kind):
    x, y, z = SETS[kind](15000, 3)
    P = _sorted_keys(x, y, z)
    K, cnt = oracle.leaves_topdown(P, 16)
    t = oracle.link(K)
    first, count = oracle.node_counts(cnt, t)
    assert first[0] == 0 and count[0] == P.size                  # root
    co = t["childOffsets"]
    for i in np.flatnonzero(co):
        ch = slice(int(co[i]), int(co[i]) + 8)
        assert int(count[ch].sum()) == int(count[i])             # parent = sum of children
        assert first[i] == first[co[i]]
    # equals the lower_bound definition via the library routine
    lev = t["levels"].astype(np.uint64)
    pre = t["prefixes"]
    shift = np.uint64(3) * (np.uint64(L) - lev)
    start = (pre ^ (np.uint64(1) << (np.uint64(3) * lev))) << shift
    end = start + (np.uint64(1) << shift)
    lo = np.searchsorted(P, start, side="left")
    hi = np.where(end >= np.uint64(KEY_END), P.size, np.searchsorted(P, end, side="left"))
    assert np.array_equal(first, lo.astype(np.uint32))
    assert np.array_equal(count, (hi - lo).astype(np.uint32))
