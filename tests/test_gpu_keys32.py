"""GPU parity of the L = 10 entry points (30-bit keys in uint32) against the oracle run
with 10 octal digits per key (oracle.key_levels(10)), bit for bit, on configurations 1-3 and on clustered inputs that
pile up at the maximum depth."""
import numpy as np
import pytest

import oracle
from paper_2307_06345_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cs():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2307_06345_b200 import binding
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def oracle32(x, y, z, bucket, curve="morton"):
    with oracle.key_levels(10):
        return oracle.full_build(x, y, z, bucket, curve=curve)


def compare(cs, got, ref, what):
    assert got["numLeaves"] == ref["leaves"].size - 1 and got["numNodes"] == ref["numNodes"], what
    assert np.array_equal(cs.u32(got["keys"]), ref["sortedKeys"].astype(np.uint32)), what + " keys"
    assert np.array_equal(cs.u32(got["perm"]), ref["perm"]), what + " perm"
    assert np.array_equal(cs.u32(got["leaves"]), ref["leaves"].astype(np.uint32)), what + " leaves"
    assert np.array_equal(cs.u32(got["counts"]), ref["counts"]), what + " counts"
    assert np.array_equal(cs.u32(got["prefixes"]), ref["prefixes"].astype(np.uint32)), what + " prefixes"
    for k in ("levels", "childOffsets", "parents", "leafToNode", "nodeToLeaf", "nodeFirst", "nodeCount"):
        assert np.array_equal(cs.u32(got[k]), ref[k]), what + " " + k
    lr = cs.u32(got["levelRange"])
    assert np.array_equal(lr[:12], ref["levelRange"][:12]) and np.all(lr[12:] == ref["numNodes"]), what + " levelRange"


@pytest.mark.parametrize("cfg_i,n,buckets", [(0, None, (64,)), (1, None, (64,)), (2, None, (16, 64)), (3, 1 << 22, (64,))])
def test_full_build_with_30_bit_keys(cs, cfg_i, n, buckets):
    cfg = W.CONFIGS[cfg_i]
    x, y, z = cfg.generate(n)
    ctx = cs.Context(max_particles=x.size, max_leaves=max(4096, x.size // 4))
    bufs = cs.TreeBuffers32(ctx, x.size)
    dx, dy, dz = dev(x), dev(y), dev(z)
    for b in buckets:
        ref = oracle32(x, y, z, b)
        got = cs.buildOctree32(ctx, dx, dy, dz, b, buffers=bufs)
        compare(cs, got, ref, f"{cfg.name} bucket {b}")
        assert int(ref["leaves"][-1]) == 1 << 30
    ctx.close()


def test_hilbert_curve_with_30_bit_keys(cs):
    x, y, z = W.plummer(300001, 5)
    ref = oracle32(x, y, z, 32, curve="hilbert")
    ctx = cs.Context(max_particles=x.size, max_leaves=x.size // 2)
    ctx.setCurve(cs.CURVE_HILBERT)
    compare(cs, cs.buildOctree32(ctx, dev(x), dev(y), dev(z), 32), ref, "hilbert")
    ctx.close()


@pytest.mark.parametrize("n", [1, 2, 100, 6656, 6657, 100003])
def test_stage_calls(cs, n):
    """cs_computeKeys32, cs_sortKeys32, cs_buildLeaves32 (one-pass, rounds, from previous leaves), cs_linkOctree32."""
    rng = np.random.default_rng(n)
    x, y, z = W.blobs(n, 77 + n, nblobs=3)
    x[: n // 3] = x[0]; y[: n // 3] = y[0]; z[: n // 3] = z[0]          # a third of the particles in one point
    ctx = cs.Context(max_particles=n, max_leaves=max(4096, n))
    with oracle.key_levels(10):
        box = oracle.box(x, y, z)
        k = oracle.keys(x, y, z, box)
        P, perm = oracle.sort(k)
        K, cnt = oracle.leaves_topdown(P, 8)
        Kit, cit, rounds, _ = oracle.leaves_iterative(P, 8)
        tree = oracle.link(K)
    dbox = dev(box)
    dk = cs.computeKeys32(ctx, dev(x), dev(y), dev(z), dbox)
    assert np.array_equal(cs.u32(dk), k.astype(np.uint32))
    dperm = cs.sortKeys32(ctx, dk)
    assert np.array_equal(cs.u32(dk), P.astype(np.uint32)) and np.array_equal(cs.u32(dperm), perm)
    for mode in (cs.LEAVES_AUTO, cs.LEAVES_ITERATIVE):
        ctx.setLeafMode(mode)
        lv, ct, r, conv = cs.buildLeaves32(ctx, dk, 8)
        assert np.array_equal(cs.u32(lv), K.astype(np.uint32)) and np.array_equal(cs.u32(ct), cnt) and conv
        assert r == rounds                                         # levels 0..10: at most 11 rounds
    # from a coarser previous array (every leaf of the bucket-64 tree): the rounds split down to the same result
    with oracle.key_levels(10):
        Kc, _ = oracle.leaves_topdown(P, 64)
    lv, ct, r, conv = cs.buildLeaves32(ctx, dk, 8, prevLeaves=dev(Kc.astype(np.uint32).view(np.int32)))
    assert np.array_equal(cs.u32(lv), K.astype(np.uint32)) and np.array_equal(cs.u32(ct), cnt) and conv
    t = cs.linkOctree32(ctx, lv)
    assert t["numNodes"] == tree["numNodes"]
    assert np.array_equal(cs.u32(t["prefixes"]), tree["prefixes"].astype(np.uint32))
    for key in ("levels", "childOffsets", "parents", "leafToNode", "nodeToLeaf"):
        assert np.array_equal(cs.u32(t[key]), tree[key]), key
    if n >= 100:
        assert int(cnt.max()) > 8 and int(K[-1]) == 1 << 30         # leaves at depth 10 keep their surplus (A7)
    ctx.close()
