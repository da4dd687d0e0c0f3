"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, bit for bit.

Integer / index arrays must be equal element by element; the box is compared as raw bits.
Inputs are the seeded workloads of paper_2307_06345_b200.workloads (same host buffers on both
sides).
"""
import numpy as np
import pytest

import oracle
from helpers import KEY_END
from paper_2307_06345_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cs():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2307_06345_b200 import binding
    return binding


@pytest.fixture(scope="module")
def ctx(cs):
    c = cs.Context(max_particles=1 << 22, max_leaves=1 << 21)
    yield c
    c.close()


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def assert_tree_equal(cs, got, ref, what=""):
    """got: dict of tensors from the binding; ref: dict from oracle.full_build."""
    assert got["numLeaves"] == ref["leaves"].size - 1, what
    assert got["numNodes"] == ref["numNodes"], what
    assert np.array_equal(cs.u64(got["leaves"]), ref["leaves"]), what + " leaves"
    assert np.array_equal(cs.u32(got["counts"]), ref["counts"]), what + " counts"
    assert np.array_equal(cs.u64(got["prefixes"]), ref["prefixes"]), what + " prefixes"
    for k in ("levels", "childOffsets", "parents", "levelRange", "leafToNode", "nodeToLeaf", "nodeFirst",
              "nodeCount"):
        assert np.array_equal(cs.u32(got[k]), ref[k]), what + " " + k


def stage_by_stage(cs, ctx, x, y, z, bucket):
    """Run every stage call separately and compare each output with the oracle."""
    ref = oracle.full_build(x, y, z, bucket)
    dx, dy, dz = dev(x), dev(y), dev(z)
    box = cs.computeBox(ctx, dx, dy, dz)
    assert np.array_equal(box.cpu().numpy().view(np.uint64), ref["box"].view(np.uint64)), "box"
    keys = cs.computeKeys(ctx, dx, dy, dz, box)
    assert np.array_equal(cs.u64(keys), ref["keys"]), "keys"
    perm = cs.sortKeys(ctx, keys)
    assert np.array_equal(cs.u64(keys), ref["sortedKeys"]), "sorted keys"
    assert np.array_equal(cs.u32(perm), ref["perm"]), "perm"
    leaves, counts, rounds, conv = cs.buildLeaves(ctx, keys, bucket)
    assert conv
    assert np.array_equal(cs.u64(leaves), ref["leaves"]), "leaves"
    assert np.array_equal(cs.u32(counts), ref["counts"]), "counts"
    _, _, ref_rounds, _ = oracle.leaves_iterative(ref["sortedKeys"], bucket)
    assert rounds == ref_rounds, "rounds"
    tree = cs.linkOctree(ctx, leaves)
    assert tree["numNodes"] == ref["numNodes"]
    assert np.array_equal(cs.u64(tree["prefixes"]), ref["prefixes"]), "prefixes"
    for k in ("levels", "childOffsets", "parents", "levelRange", "leafToNode", "nodeToLeaf"):
        assert np.array_equal(cs.u32(tree[k]), ref[k]), k
    # node counts: definitional (search only) and with the leaf-count accelerator
    f1, c1 = cs.nodeCounts(ctx, keys, tree["prefixes"])
    f2, c2 = cs.nodeCounts(ctx, keys, tree["prefixes"], counts, tree["nodeToLeaf"])
    for f, c in ((f1, c1), (f2, c2)):
        assert np.array_equal(cs.u32(f), ref["nodeFirst"]), "nodeFirst"
        assert np.array_equal(cs.u32(c), ref["nodeCount"]), "nodeCount"
    return ref


def fused(cs, ctx, x, y, z, bucket, ref):
    got = cs.buildOctree(ctx, dev(x), dev(y), dev(z), bucket)
    assert np.array_equal(got["box6"].cpu().numpy().view(np.uint64), ref["box"].view(np.uint64))
    assert np.array_equal(cs.u64(got["keys"]), ref["sortedKeys"])
    assert np.array_equal(cs.u32(got["perm"]), ref["perm"])
    assert_tree_equal(cs, got, ref, "fused")
    assert got["converged"]
    return got


# ------------------------------------------------------------------------------------------------
# small cases spanning several tiles and ragged tails (sort tile = 6656, leaf tile = 1024)
CASES = [
    ("uniform", 1, 64), ("uniform", 2, 1), ("uniform", 6655, 16), ("uniform", 6656, 16), ("uniform", 6657, 16),
    ("uniform", 3 * 6656 + 17, 8), ("uniform", 65536, 64), ("plummer", 100003, 64), ("plummer", 250000, 16),
    ("blobs", 300001, 64), ("blobs", 131072, 1), ("gaussian", 200000, 32),
]


def _gen(kind, n, seed=12345):
    if kind == "uniform":
        return W.uniform(n, 0.0, 1.0, seed)
    if kind == "plummer":
        return W.plummer(n, seed)
    if kind == "blobs":
        return W.blobs(n, seed, nblobs=50)
    return W.gaussian(n, seed)


@pytest.mark.parametrize("kind,n,bucket", CASES)
def test_stages_and_fused_match_oracle(cs, ctx, kind, n, bucket):
    x, y, z = _gen(kind, n)
    ref = stage_by_stage(cs, ctx, x, y, z, bucket)
    fused(cs, ctx, x, y, z, bucket, ref)


def test_config1_and_config2(cs, ctx):
    for cfg in W.CONFIGS[:2]:
        x, y, z = cfg.generate()
        for b in cfg.bucket_sizes:
            ref = stage_by_stage(cs, ctx, x, y, z, b)
            fused(cs, ctx, x, y, z, b, ref)


def test_unaligned_and_odd_inputs_take_the_scalar_path(cs, ctx):
    x, y, z = W.uniform(50001, -1.0, 1.0, 9)
    ref = oracle.full_build(x[1:], y[1:], z[1:], 16)
    dx, dy, dz = dev(x)[1:], dev(y)[1:], dev(z)[1:]          # 8-byte aligned only
    box = cs.computeBox(ctx, dx, dy, dz)
    assert np.array_equal(box.cpu().numpy().view(np.uint64), ref["box"].view(np.uint64))
    keys = cs.computeKeys(ctx, dx, dy, dz, box)
    assert np.array_equal(cs.u64(keys), ref["keys"])
    got = cs.buildOctree(ctx, dx, dy, dz, 16)
    assert_tree_equal(cs, got, ref, "unaligned fused")
    assert np.array_equal(cs.u32(got["perm"]), ref["perm"])


def test_sort_random_64bit_patterns_and_duplicates(cs, ctx):
    rng = np.random.default_rng(5)
    for n in (1, 31, 33, 5000, 6656 * 2, 100001):
        k = rng.integers(0, 1 << 63, n, dtype=np.uint64)
        if n > 100:
            k[rng.integers(0, n, n // 3)] = k[rng.integers(0, n, n // 3)]     # many duplicates
        P, perm = oracle.sort(k)
        dk = cs.from_u64(k, ctx.device)
        dperm = cs.sortKeys(ctx, dk)
        assert np.array_equal(cs.u64(dk), P)
        assert np.array_equal(cs.u32(dperm), perm)
    # few distinct keys: every digit but one is constant
    k = (rng.integers(0, 5, 60000, dtype=np.uint64) << np.uint64(37)) | np.uint64(3)
    P, perm = oracle.sort(k)
    dk = cs.from_u64(k, ctx.device)
    dperm = cs.sortKeys(ctx, dk)
    assert np.array_equal(cs.u64(dk), P) and np.array_equal(cs.u32(dperm), perm)


def test_degenerate_particle_sets(cs, ctx):
    # all particles at one point: flat box in every dimension -> key 0, leaves refine to depth 21
    n = 300
    x = np.full(n, 0.25); y = np.full(n, -3.0); z = np.full(n, 7.5)
    ref = stage_by_stage(cs, ctx, x, y, z, 64)
    assert ref["levels"].max() == 21
    fused(cs, ctx, x, y, z, 64, ref)
    # two clusters of exact duplicates + flat z
    x = np.concatenate([np.full(200, 0.1), np.full(200, 0.9), [0.5]])
    y = np.concatenate([np.full(200, 0.2), np.full(200, 0.8), [0.5]])
    z = np.zeros(401)
    ref = stage_by_stage(cs, ctx, x, y, z, 16)
    fused(cs, ctx, x, y, z, 16, ref)


def test_user_box_clamps_like_the_oracle(cs, ctx):
    x, y, z = W.uniform(20000, -2.0, 2.0, 4)
    box6 = np.array([-1.0, 1.0, -0.5, 1.5, 0.0, 0.0])       # particles outside; flat z
    ref = oracle.keys(x, y, z, box6)
    keys = cs.computeKeys(ctx, dev(x), dev(y), dev(z), dev(box6))
    assert np.array_equal(cs.u64(keys), ref)


def test_incremental_rebuild_from_previous_leaves(cs, ctx):
    """Config-5 shape at reduced N: full build, then rebuilds after a Gaussian step, each starting
    from the previous leaf array."""
    cfg = W.CONFIGS[4]
    n = 1 << 18
    x, y, z = cfg.generate(n)
    ref = oracle.full_build(x, y, z, 64)
    got = cs.buildOctree(ctx, dev(x), dev(y), dev(z), 64)
    assert_tree_equal(cs, got, ref, "step 0")
    prev = got["leaves"].clone()
    prev_ref = ref["leaves"]
    for k in range(1, 4):
        x, y, z = cfg.step(x, y, z, k)
        ref = oracle.full_build(x, y, z, 64)
        got = cs.buildOctree(ctx, dev(x), dev(y), dev(z), 64, prevLeaves=prev)
        assert_tree_equal(cs, got, ref, f"step {k}")
        b = oracle.box(x, y, z)
        P, _ = oracle.sort(oracle.keys(x, y, z, b))
        _, _, ref_rounds, _ = oracle.leaves_iterative(P, 64, K_start=prev_ref)
        assert got["rounds"] == ref_rounds
        # the paper's single-update mode: one round, compared with one oracle round
        K1, c1, r1, conv1 = oracle.leaves_iterative(P, 64, K_start=prev_ref, max_rounds=1)
        dP = cs.from_u64(P, ctx.device)
        l1, n1, rr, conv = cs.buildLeaves(ctx, dP, 64, prevLeaves=cs.from_u64(prev_ref, ctx.device), maxRounds=1,
                                          allow_not_converged=True)
        assert rr == 1 and conv == conv1
        assert np.array_equal(cs.u64(l1), K1) and np.array_equal(cs.u32(n1), c1)
        prev = got["leaves"].clone()
        prev_ref = ref["leaves"]


def test_merge_path_from_a_too_fine_previous_tree(cs, ctx):
    x, y, z = W.plummer(60000, 77)
    b = oracle.box(x, y, z)
    P, _ = oracle.sort(oracle.keys(x, y, z, b))
    Kfine, _ = oracle.leaves_topdown(P, 4)
    Kref, cref, rounds_ref, _ = oracle.leaves_iterative(P, 64, K_start=Kfine)
    Ktd, _ = oracle.leaves_topdown(P, 64)
    assert np.array_equal(Kref, Ktd)
    dP = cs.from_u64(P, ctx.device)
    leaves, counts, rounds, conv = cs.buildLeaves(ctx, dP, 64, prevLeaves=cs.from_u64(Kfine, ctx.device))
    assert conv and rounds == rounds_ref
    assert np.array_equal(cs.u64(leaves), Kref) and np.array_equal(cs.u32(counts), cref)
    # round by round
    K = Kfine
    for r in range(1, 4):
        K1, c1, _, _ = oracle.leaves_iterative(P, 64, K_start=Kfine, max_rounds=r)
        l1, n1, rr, _ = cs.buildLeaves(ctx, dP, 64, prevLeaves=cs.from_u64(Kfine, ctx.device), maxRounds=r,
                                       allow_not_converged=True)
        assert np.array_equal(cs.u64(l1), K1) and np.array_equal(cs.u32(n1), c1)


def test_empty_particle_set_gives_the_root(cs, ctx):
    e = torch.empty(0, dtype=torch.int64, device="cuda")
    leaves, counts, rounds, conv = cs.buildLeaves(ctx, e, 64)
    assert cs.u64(leaves).tolist() == [0, KEY_END] and cs.u32(counts).tolist() == [0] and rounds == 1 and conv
    tree = cs.linkOctree(ctx, leaves)
    assert tree["numNodes"] == 1 and cs.u64(tree["prefixes"]).tolist() == [1]
    assert cs.u32(tree["levelRange"]).tolist() == [0] + [1] * 22


def test_error_codes(cs, ctx):
    x, y, z = W.uniform(40000, 0.0, 1.0, 2)
    dx, dy, dz = dev(x), dev(y), dev(z)
    e = torch.empty(0, dtype=torch.float64, device="cuda")
    with pytest.raises(cs.CornerstoneError) as ei:
        cs.computeBox(ctx, e, e, e)
    assert ei.value.status == cs.ERR_INVALID_ARG
    box = cs.computeBox(ctx, dx, dy, dz)
    keys = cs.computeKeys(ctx, dx, dy, dz, box)
    cs.sortKeys(ctx, keys)
    with pytest.raises(cs.CornerstoneError) as ei:
        cs.buildLeaves(ctx, keys, 0)
    assert ei.value.status == cs.ERR_INVALID_ARG
    # capacity: outputs untouched
    leaves = torch.full((101,), -7, dtype=torch.int64, device="cuda")
    counts = torch.full((100,), -7, dtype=torch.int32, device="cuda")
    with pytest.raises(cs.CornerstoneError) as ei:
        cs.buildLeaves(ctx, keys, 16, leafCapacity=100, leaves=leaves, counts=counts)
    assert ei.value.status == cs.ERR_CAPACITY
    assert bool((leaves == -7).all()) and bool((counts == -7).all())
    # not a cornerstone array
    bad = cs.from_u64(np.array([0, 5, KEY_END], dtype=np.uint64), ctx.device)
    with pytest.raises(cs.CornerstoneError) as ei:
        cs.buildLeaves(ctx, keys, 16, prevLeaves=bad)
    assert ei.value.status == cs.ERR_NOT_CORNERSTONE
    with pytest.raises(cs.CornerstoneError) as ei:
        cs.linkOctree(ctx, cs.from_u64(np.array([0, 8 ** 20, KEY_END], dtype=np.uint64), ctx.device))
    assert ei.value.status == cs.ERR_NOT_CORNERSTONE
    # 8 leaves that are powers of 8 but do not close into an octree (misaligned sibling group)
    d = 8 ** 20
    K = np.array([0, d, 2 * d, 2 * d + d // 8] + [KEY_END], dtype=np.uint64)
    with pytest.raises(cs.CornerstoneError):
        cs.linkOctree(ctx, cs.from_u64(np.concatenate([K[:4], K[4:]]), ctx.device))
    # maxRounds reached
    leaves, counts, rounds, conv = cs.buildLeaves(ctx, keys, 16, maxRounds=2, allow_not_converged=True)
    assert rounds == 2 and not conv
    K2, c2, _, _ = oracle.leaves_iterative(cs.u64(keys), 16, max_rounds=2)
    assert np.array_equal(cs.u64(leaves), K2) and np.array_equal(cs.u32(counts), c2)
    # the context still works after errors
    leaves, counts, rounds, conv = cs.buildLeaves(ctx, keys, 16)
    Kt, ct = oracle.leaves_topdown(cs.u64(keys), 16)
    assert np.array_equal(cs.u64(leaves), Kt) and np.array_equal(cs.u32(counts), ct)


def test_host_path_matches(cs, ctx):
    x, y, z = W.blobs(150000, 8, nblobs=40)
    ref = oracle.full_build(x, y, z, 64)
    hb = cs.HostBuffers(150000, ctx.max_leaves, want=("box6", "keys", "perm", "leaves", "counts", "prefixes",
                                                        "levels", "childOffsets", "parents", "levelRange",
                                                        "leafToNode", "nodeToLeaf", "nodeFirst", "nodeCount"))
    hx, hy, hz = (torch.from_numpy(a).pin_memory() for a in (x, y, z))
    sz = cs.buildOctreeHost(ctx, hx, hy, hz, 64, hb)
    nl, nn = sz["numLeaves"], sz["numNodes"]
    assert nl == ref["leaves"].size - 1 and nn == ref["numNodes"]
    assert np.array_equal(hb.t["keys"].numpy().view(np.uint64), ref["sortedKeys"])
    assert np.array_equal(hb.t["perm"].numpy().view(np.uint32), ref["perm"])
    assert np.array_equal(hb.t["leaves"].numpy().view(np.uint64)[:nl + 1], ref["leaves"])
    assert np.array_equal(hb.t["counts"].numpy().view(np.uint32)[:nl], ref["counts"])
    assert np.array_equal(hb.t["prefixes"].numpy().view(np.uint64)[:nn], ref["prefixes"])
    for k in ("levels", "childOffsets", "parents", "nodeToLeaf", "nodeFirst", "nodeCount"):
        assert np.array_equal(hb.t[k].numpy().view(np.uint32)[:nn], ref[k]), k
    assert np.array_equal(hb.t["leafToNode"].numpy().view(np.uint32)[:nl], ref["leafToNode"])
    assert np.array_equal(hb.t["levelRange"].numpy().view(np.uint32), ref["levelRange"])


def test_host_path_with_chunked_upload(cs):
    """Above the graph limit cs_buildOctreeHost uploads in 8 pieces on a second stream and reduces the box piece by
    piece under the upload: the tree must be the oracle's, call after call (the staging buffers are reused), for a size
    whose last piece is ragged and for particles whose extremes lie in different pieces."""
    n = (1 << 22) + 12345
    x, y, z = W.plummer(n, 77)
    x[n - 1] = x.max() + 3.0                                  # extremes in the last and in the first piece
    y[0] = y.min() - 2.0
    ref = oracle.full_build(x, y, z, 64)
    ctx = cs.Context(max_particles=n, max_leaves=n // 4)
    hb = cs.HostBuffers(n, ctx.max_leaves, want=("box6", "keys", "perm", "leaves", "counts", "prefixes", "childOffsets",
                                                  "nodeFirst", "nodeCount"))
    hx, hy, hz = (torch.from_numpy(a).pin_memory() for a in (x, y, z))
    for it in range(3):
        sz = cs.buildOctreeHost(ctx, hx, hy, hz, 64, hb)
        nl, nn = sz["numLeaves"], sz["numNodes"]
        assert nl == ref["leaves"].size - 1 and nn == ref["numNodes"]
        assert np.array_equal(hb.t["box6"].numpy().view(np.uint64), ref["box"].view(np.uint64)), it
        assert np.array_equal(hb.t["keys"].numpy().view(np.uint64), ref["sortedKeys"]), it
        assert np.array_equal(hb.t["perm"].numpy().view(np.uint32), ref["perm"]), it
        assert np.array_equal(hb.t["leaves"].numpy().view(np.uint64)[:nl + 1], ref["leaves"]), it
        assert np.array_equal(hb.t["counts"].numpy().view(np.uint32)[:nl], ref["counts"]), it
        assert np.array_equal(hb.t["prefixes"].numpy().view(np.uint64)[:nn], ref["prefixes"]), it
        for k in ("childOffsets", "nodeFirst", "nodeCount"):
            assert np.array_equal(hb.t[k].numpy().view(np.uint32)[:nn], ref[k]), k
    ctx.close()


def test_two_contexts_and_a_side_stream(cs):
    """Contexts share nothing: two of them used alternately, one on a non-default stream, give the oracle's trees."""
    xa, ya, za = W.blobs(150001, 41, nblobs=20)
    xb, yb, zb = W.plummer(90000, 42)
    ra, rb = oracle.full_build(xa, ya, za, 64), oracle.full_build(xb, yb, zb, 16)
    ca = cs.Context(max_particles=200000, max_leaves=100000)
    cb = cs.Context(max_particles=100000, max_leaves=100000)
    da, db = [dev(a) for a in (xa, ya, za)], [dev(a) for a in (xb, yb, zb)]
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    for _ in range(3):
        ga = cs.buildOctree(ca, da[0], da[1], da[2], 64)
        with torch.cuda.stream(side):
            gb = cs.buildOctree(cb, db[0], db[1], db[2], 16)
        assert_tree_equal(cs, ga, ra, "context a")
        assert_tree_equal(cs, gb, rb, "context b")
        assert np.array_equal(cs.u32(ga["perm"]), ra["perm"]) and np.array_equal(cs.u32(gb["perm"]), rb["perm"])
    ca.close()
    cb.close()
