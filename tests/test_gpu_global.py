"""GPU parity of the distributed build's calls (Eq. 11) on ONE device: the particles
are cut into R shards as R ranks would hold them, every shard is counted with cs_countLeaves, the count arrays are
summed element by element (standing in for the all-reduce f_r; torch.add is plumbing here, the method's arithmetic is
in the library calls around it), cs_rebalance applies g.  Every round's N and K' equal the oracle's O11, the converged
array equals the top-down tree of the union (O4), cs_partitionLeaves equals O12, cs_nodeCountsFromLeaves equals O7."""
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
    c = cs.Context(max_particles=1 << 21, max_leaves=1 << 20)
    yield c
    c.close()


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def shards_of(cs, ctx, x, y, z, R, rng):
    """Keys with the GLOBAL box, cut into R shards of unequal size (an arbitrary distribution of the particles over
    the ranks), each sorted on its own by cs_sortKeys.  Returns device tensors and host copies."""
    box = oracle.box(x, y, z)
    dbox = dev(box)
    n = x.size
    cuts = np.sort(rng.integers(0, n + 1, R - 1))
    bounds = np.concatenate([[0], cuts, [n]]).astype(np.int64)
    order = rng.permutation(n)
    out_d, out_h = [], []
    for r in range(R):
        idx = order[bounds[r]:bounds[r + 1]]
        if idx.size == 0:
            out_d.append(torch.empty(0, dtype=torch.int64, device="cuda"))
            out_h.append(np.empty(0, dtype=np.uint64))
            continue
        k = cs.computeKeys(ctx, dev(x[idx]), dev(y[idx]), dev(z[idx]), dbox)
        cs.sortKeys(ctx, k)
        out_d.append(k)
        out_h.append(cs.u64(k).copy())
    return out_d, out_h, box


def global_counts(cs, ctx, shards, K):
    total = None
    for P in shards:
        c = cs.countLeaves(ctx, P, K)
        total = c.clone() if total is None else total + c          # f_r: element-wise sum over the ranks
    return total


@pytest.mark.parametrize("R", [2, 4, 8])
@pytest.mark.parametrize("workload,bucket", [("uniform", 16), ("plummer", 64), ("blobs", 8)])
def test_rounds_of_the_distributed_build_equal_the_oracle(cs, ctx, R, workload, bucket):
    rng = np.random.default_rng(100 * R + bucket)
    n = 60_000
    if workload == "uniform":
        x, y, z = W.uniform(n, 0.0, 1.0, W.BASE_SEED + 31)
    elif workload == "plummer":
        x, y, z = W.plummer(n, W.BASE_SEED + 32)
    else:
        x, y, z = W.blobs(n, W.BASE_SEED + 33, nblobs=20)
    shards_d, shards_h, box = shards_of(cs, ctx, x, y, z, R, rng)
    K = np.array([0, KEY_END], dtype=np.uint64)
    Kd = cs.from_u64(K, "cuda")
    rounds = 0
    while True:
        ref = oracle.global_round(shards_h, K, bucket, cap=1 << 20)
        N = global_counts(cs, ctx, shards_d, Kd)
        assert np.array_equal(cs.u32(N), ref["N"]), f"round {rounds}: summed counts"
        Knew, changed = cs.rebalance(ctx, Kd, N, bucket)
        assert np.array_equal(cs.u64(Knew), ref["K"]), f"round {rounds}: K'"
        assert changed == bool(np.any(ref["O"] != 1)), f"round {rounds}: changed"
        rounds += 1
        if not changed:
            break
        K, Kd = ref["K"], Knew.clone()
        assert rounds <= 22
    # the fixpoint of the distributed rounds is the top-down tree of the union of the shards (O4)
    Pall = np.sort(np.concatenate(shards_h), kind="stable")
    Ktop, Ntop = oracle.leaves_topdown(Pall, bucket)
    assert np.array_equal(cs.u64(Kd), Ktop)
    assert np.array_equal(cs.u32(N), Ntop)
    # SFC domain decomposition (O12) for several rank counts
    for nr in (1, 2, R, 7, 64):
        got = cs.u32(cs.partitionLeaves(ctx, N, nr))
        assert np.array_equal(got, oracle.partition(Ntop, nr)), f"partition into {nr}"
    # the replicated global octree and its node counts from the summed leaf counts (O6, O7)
    tree = cs.linkOctree(ctx, Kd)
    rtree = oracle.link(Ktop)
    first, count = cs.nodeCountsFromLeaves(ctx, Kd, N, tree["prefixes"])
    rfirst, rcount = oracle.node_counts(Ntop, rtree)
    assert np.array_equal(cs.u64(tree["prefixes"]), rtree["prefixes"])
    assert np.array_equal(cs.u32(first), rfirst)
    assert np.array_equal(cs.u32(count), rcount)


def test_one_round_with_merges_and_an_empty_rank(cs, ctx):
    """Start from a tree that is too fine (bucket 4) and rebalance with bucket 256: the round merges; one of the
    ranks holds no particles at all."""
    rng = np.random.default_rng(9)
    x, y, z = W.uniform(30_000, -1.0, 1.0, W.BASE_SEED + 41)
    box = oracle.box(x, y, z)
    P = np.sort(oracle.keys(x, y, z, box), kind="stable")
    Kfine, _ = oracle.leaves_topdown(P, 4)
    parts = np.array_split(rng.permutation(P.size), 3)
    shards_h = [np.sort(P[i], kind="stable") for i in parts] + [np.empty(0, dtype=np.uint64)]
    shards_d = [cs.from_u64(s, "cuda") for s in shards_h]
    K, Kd = Kfine, cs.from_u64(Kfine, "cuda")
    for r in range(4):
        ref = oracle.global_round(shards_h, K, 256, cap=1 << 20)
        N = global_counts(cs, ctx, shards_d, Kd)
        assert np.array_equal(cs.u32(N), ref["N"])
        Knew, changed = cs.rebalance(ctx, Kd, N, 256)
        assert np.array_equal(cs.u64(Knew), ref["K"])
        assert np.any(ref["O"] == 0) or r > 0
        K, Kd = ref["K"], Knew.clone()
        if not changed:
            break


def test_count_leaves_equals_build_leaves_counts(cs, ctx):
    """f alone on one rank reproduces the counts cs_buildLeaves returns with its leaves (Eq. 3)."""
    x, y, z = W.plummer(200_003, W.BASE_SEED + 51)
    ref = oracle.full_build(x, y, z, 64)
    P = cs.from_u64(ref["sortedKeys"], "cuda")
    K = cs.from_u64(ref["leaves"], "cuda")
    assert np.array_equal(cs.u32(cs.countLeaves(ctx, P, K)), ref["counts"])
    # no particles
    empty = torch.empty(0, dtype=torch.int64, device="cuda")
    assert not cs.u32(cs.countLeaves(ctx, empty, K)).any()


def test_rebalance_errors(cs, ctx):
    K = cs.from_u64(np.array([0, 1 << 60, KEY_END], dtype=np.uint64), "cuda")     # not a cornerstone array
    N = cs.from_u32(np.array([1, 1], dtype=np.uint32), "cuda")
    with pytest.raises(cs.CornerstoneError) as e:
        cs.rebalance(ctx, K, N, 4)
    assert e.value.status == cs.ERR_NOT_CORNERSTONE
    root = cs.from_u64(np.array([0, KEY_END], dtype=np.uint64), "cuda")
    N = cs.from_u32(np.array([100], dtype=np.uint32), "cuda")
    with pytest.raises(cs.CornerstoneError) as e:
        cs.rebalance(ctx, root, N, 4, leafCapacity=7)
    assert e.value.status == cs.ERR_CAPACITY
    Knew, changed = cs.rebalance(ctx, root, N, 4, leafCapacity=8)
    assert changed and Knew.numel() == 9


def test_partition_with_large_totals_and_many_tiles(cs, ctx):
    """Counts whose sum exceeds 2^32 (64-bit prefix sums), more than one tile of 2048 leaves, repeated boundaries."""
    rng = np.random.default_rng(77)
    N = rng.integers(0, 1 << 14, 300_000).astype(np.uint32)
    N[rng.integers(0, N.size, 2000)] = np.uint32(0xFFFFFFF0)
    N[1000:50_000] = 0
    d = cs.from_u32(N, "cuda")
    for nr in (2, 3, 8, 100, 1000, 4097):
        assert np.array_equal(cs.u32(cs.partitionLeaves(ctx, d, nr)), oracle.partition(N, nr)), nr
    z = cs.from_u32(np.zeros(5000, dtype=np.uint32), "cuda")
    assert np.array_equal(cs.u32(cs.partitionLeaves(ctx, z, 5)), oracle.partition(np.zeros(5000, dtype=np.uint32), 5))
