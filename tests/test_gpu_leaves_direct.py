"""GPU parity of the one-pass leaf build (cs_leaves_direct.cu) against the oracle.

From the root and to convergence cs_buildLeaves computes the fixpoint of f, g
in one pass over P; it must return exactly what the oracle's recursive top-down construction
(O4) and the oracle's literal iteration of Eqs. 3-9 (O5: leaves, counts AND round count) return,
and exactly what the library's own rounds return (cs_setLeafMode(ITERATIVE)).
Key sets are synthetic and seeded; they are built directly as sorted 63-bit keys so that tile
boundaries (2048 positions), window lengths (bucketSize + 1) and deep levels are hit on purpose.
"""
import numpy as np
import pytest

import oracle
from helpers import KEY_END, check_cornerstone

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
    c = cs.Context(max_particles=1 << 21, max_leaves=1 << 21)
    yield c
    c.close()


def _keys(kind, n, seed):
    rng = np.random.default_rng(seed)
    if n == 0:
        return np.zeros(0, dtype=np.uint64)
    if kind == "uniform":
        k = rng.integers(0, 1 << 63, size=n, dtype=np.uint64)
    elif kind == "dups":          # few distinct keys, each many times: leaves at level 21 above bucketSize
        pool = rng.integers(0, 1 << 63, size=max(1, n // 97), dtype=np.uint64)
        k = pool[rng.integers(0, pool.size, size=n)]
    elif kind == "same":          # one key n times
        k = np.full(n, rng.integers(0, 1 << 63, dtype=np.uint64), dtype=np.uint64)
    elif kind == "deep":          # clusters that only separate in the low digits + a sparse background
        centres = rng.integers(0, 1 << 63, size=9, dtype=np.uint64)
        width = np.uint64(1) << rng.integers(3, 40, size=9).astype(np.uint64)
        c = rng.integers(0, 9, size=n)
        k = (centres[c] & ~(width[c] - np.uint64(1))) + (rng.integers(0, 1 << 62, size=n, dtype=np.uint64) % width[c])
        bg = rng.random(n) < 0.05
        k[bg] = rng.integers(0, 1 << 63, size=int(bg.sum()), dtype=np.uint64)
    elif kind == "edges":         # first and last cell of the key space are occupied
        k = rng.integers(0, 1 << 63, size=n, dtype=np.uint64)
        k[: min(n, 5)] = 0
        k[-min(n, 7):] = (1 << 63) - 1
    else:
        raise ValueError(kind)
    return np.sort(k & np.uint64((1 << 63) - 1))


def _check(cs, ctx, P, bucket):
    ref_K, ref_N = oracle.leaves_topdown(P, bucket)
    it_K, it_N, it_rounds, it_conv = oracle.leaves_iterative(P, bucket)
    assert it_conv and np.array_equal(it_K, ref_K) and np.array_equal(it_N, ref_N)     # oracle O4 == O5
    dP = cs.from_u64(P, ctx.device) if P.size else torch.empty(0, dtype=torch.int64, device=ctx.device)
    for mode in (cs.LEAVES_AUTO, cs.LEAVES_ITERATIVE):
        ctx.setLeafMode(mode)
        try:
            leaves, counts, rounds, conv = cs.buildLeaves(ctx, dP, bucket)
        finally:
            ctx.setLeafMode(cs.LEAVES_AUTO)
        what = f"mode={mode} n={P.size} bucket={bucket}"
        assert conv, what
        assert np.array_equal(cs.u64(leaves), ref_K), what + " leaves"
        assert np.array_equal(cs.u32(counts), ref_N), what + " counts"
        assert rounds == it_rounds, what + " rounds"
    return ref_K, ref_N


SIZES = [0, 1, 2, 63, 64, 65, 66, 129, 2047, 2048, 2049, 4095, 4096, 4097, 6143, 10000, 100003]


@pytest.mark.parametrize("kind", ["uniform", "dups", "deep", "edges"])
@pytest.mark.parametrize("bucket", [1, 2, 3, 16, 63, 64, 65, 100, 1000, 1024])
def test_direct_equals_oracle(cs, ctx, kind, bucket):
    for n in SIZES:
        _check(cs, ctx, _keys(kind, n, 1000 * bucket + n), bucket)


def test_identical_keys_stop_at_depth_L(cs, ctx):
    for n, bucket in ((1, 1), (2, 1), (65, 64), (5000, 64), (4096, 7)):
        K, N = _check(cs, ctx, _keys("same", n, n), bucket)
        if n > bucket:
            assert N.max() == n and 21 in check_cornerstone(K)       # A7: a level-21 leaf may exceed bucketSize


def test_bucket_above_direct_limit_falls_back_to_rounds(cs, ctx):
    P = _keys("uniform", 50000, 7)
    _check(cs, ctx, P, 1025)
    _check(cs, ctx, P, 5000)


def test_large_clustered_set(cs, ctx):
    P = _keys("deep", 1 << 20, 99)
    K, N = _check(cs, ctx, P, 64)
    assert int(N.sum()) == P.size and K[-1] == KEY_END


def test_capacity_error_leaves_outputs_untouched(cs, ctx):
    P = _keys("uniform", 100000, 3)
    dP = cs.from_u64(P, ctx.device)
    leaves = torch.full((101,), -1, dtype=torch.int64, device=ctx.device)
    counts = torch.full((100,), -1, dtype=torch.int32, device=ctx.device)
    with pytest.raises(cs.CornerstoneError) as e:
        cs.buildLeaves(ctx, dP, 16, leafCapacity=100, leaves=leaves, counts=counts)
    assert e.value.status == cs.ERR_CAPACITY
    assert bool((leaves == -1).all()) and bool((counts == -1).all())


def test_fused_build_uses_the_same_leaves(cs, ctx):
    """cs_buildOctree (direct leaves inside) against the oracle's full build, and against itself in ITERATIVE mode."""
    from paper_2307_06345_b200 import workloads as W
    x, y, z = W.blobs(300001, 4242, nblobs=40)
    ref = oracle.full_build(x, y, z, 64)
    d = [torch.from_numpy(a).cuda() for a in (x, y, z)]
    out = {}
    for mode in (cs.LEAVES_AUTO, cs.LEAVES_ITERATIVE):
        ctx.setLeafMode(mode)
        try:
            got = cs.buildOctree(ctx, *d, 64)
        finally:
            ctx.setLeafMode(cs.LEAVES_AUTO)
        assert np.array_equal(cs.u64(got["leaves"]), ref["leaves"])
        assert np.array_equal(cs.u32(got["counts"]), ref["counts"])
        assert np.array_equal(cs.u64(got["prefixes"]), ref["prefixes"])
        for k in ("childOffsets", "parents", "levelRange", "nodeFirst", "nodeCount"):
            assert np.array_equal(cs.u32(got[k]), ref[k]), k
        out[mode] = got["rounds"]
    assert out[cs.LEAVES_AUTO] == out[cs.LEAVES_ITERATIVE]
