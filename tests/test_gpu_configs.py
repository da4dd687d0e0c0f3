"""GPU parity on BASELINE.json's configurations, through cs_buildOctree with pre-allocated
buffers (the launch configuration bench.py times).  Bit-exact against the oracle.

c1, c2 run in test_gpu_parity.py.  c3 (2^24, buckets 16 and 64) and c4 (2^26, the headline) run
here at full size.  c5 (2^28 + 10 incremental rebuilds) runs with full oracle parity at a reduced
N by default, and at full size -- oracle checks on sampled outputs plus size-independent
properties -- when CS_TEST_FULL_C5=1 (≈ 25 GB of host memory, several minutes).
"""
import os

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


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def check_against_oracle(cs, got, ref, what):
    assert got["numLeaves"] == ref["leaves"].size - 1, what
    assert got["numNodes"] == ref["numNodes"], what
    assert np.array_equal(got["box6"].cpu().numpy().view(np.uint64), ref["box"].view(np.uint64)), what + " box"
    assert np.array_equal(cs.u64(got["keys"]), ref["sortedKeys"]), what + " sorted keys"
    assert np.array_equal(cs.u32(got["perm"]), ref["perm"]), what + " perm"
    assert np.array_equal(cs.u64(got["leaves"]), ref["leaves"]), what + " leaves"
    assert np.array_equal(cs.u32(got["counts"]), ref["counts"]), what + " counts"
    assert np.array_equal(cs.u64(got["prefixes"]), ref["prefixes"]), what + " prefixes"
    for k in ("levels", "childOffsets", "parents", "levelRange", "leafToNode", "nodeToLeaf", "nodeFirst",
              "nodeCount"):
        assert np.array_equal(cs.u32(got[k]), ref[k]), what + " " + k


def test_config3_uniform_16m_both_buckets(cs):
    cfg = W.CONFIGS[2]
    x, y, z = cfg.generate()
    ctx = cs.Context(max_particles=cfg.n, max_leaves=cfg.n // 4)
    bufs = cs.TreeBuffers(ctx, cfg.n)
    dx, dy, dz = dev(x), dev(y), dev(z)
    for b in cfg.bucket_sizes:
        ref = oracle.full_build(x, y, z, b)
        got = cs.buildOctree(ctx, dx, dy, dz, b, buffers=bufs)
        check_against_oracle(cs, got, ref, f"c3 bucket {b}")
        _, _, ref_rounds, _ = oracle.leaves_iterative(ref["sortedKeys"], b)
        assert got["rounds"] == ref_rounds and got["converged"]
    ctx.close()


def test_config4_blobs_64m_headline(cs):
    cfg = W.CONFIGS[3]
    x, y, z = cfg.generate()
    ref = oracle.full_build(x, y, z, 64)
    ctx = cs.Context(max_particles=cfg.n, max_leaves=cfg.n // 4)      # as in bench.py
    bufs = cs.TreeBuffers(ctx, cfg.n)
    got = cs.buildOctree(ctx, dev(x), dev(y), dev(z), 64, buffers=bufs)
    check_against_oracle(cs, got, ref, "c4")
    assert got["converged"]
    # duplicates exist at this density: stability is really exercised
    assert int((ref["sortedKeys"][1:] == ref["sortedKeys"][:-1]).sum()) > 0
    ctx.close()


def test_config5_plummer_incremental_reduced(cs):
    """c5's recipe at N = 2^22: full build, then 10 rebuilds each starting from the previous leaves."""
    cfg = W.CONFIGS[4]
    n = 1 << 22
    x, y, z = cfg.generate(n)
    ctx = cs.Context(max_particles=n, max_leaves=n // 4)
    bufs = cs.TreeBuffers(ctx, n)
    ref = oracle.full_build(x, y, z, 64)
    got = cs.buildOctree(ctx, dev(x), dev(y), dev(z), 64, buffers=bufs)
    check_against_oracle(cs, got, ref, "c5 step 0")
    prev = got["leaves"].clone()
    for k in range(1, cfg.incremental_steps + 1):
        x, y, z = cfg.step(x, y, z, k)
        ref = oracle.full_build(x, y, z, 64)
        got = cs.buildOctree(ctx, dev(x), dev(y), dev(z), 64, buffers=bufs, prevLeaves=prev)
        check_against_oracle(cs, got, ref, f"c5 step {k}")
        assert got["rounds"] <= 4            # a small step needs one update (+ the confirming round)
        prev = got["leaves"].clone()
    ctx.close()


@pytest.mark.skipif(os.environ.get("CS_TEST_FULL_C5") != "1", reason="set CS_TEST_FULL_C5=1 (2^28 particles)")
def test_config5_full_size_properties(cs):
    cfg = W.CONFIGS[4]
    n = cfg.n
    x, y, z = cfg.generate()
    ctx = cs.Context(max_particles=n, max_leaves=n // 4)
    bufs = cs.TreeBuffers(ctx, n)
    dx, dy, dz = dev(x), dev(y), dev(z)
    rng = np.random.default_rng(1)
    prev = None
    for step in range(0, 3):
        if step:
            x, y, z = cfg.step(x, y, z, step)
            dx, dy, dz = dev(x), dev(y), dev(z)
        got = cs.buildOctree(ctx, dx, dy, dz, 64, buffers=bufs, prevLeaves=prev)
        P = got["keys"]
        # properties that hold at any size
        assert bool((P[1:] >= P[:-1]).all())                                    # keys < 2^63: int64 order is key order
        perm = got["perm"].to(torch.int64) & 0xFFFFFFFF
        assert int(torch.bincount(perm, minlength=n).max()) == 1                # a permutation
        box = cs.computeBox(ctx, dx, dy, dz)
        unsorted = cs.computeKeys(ctx, dx, dy, dz, box)
        assert bool((unsorted[perm] == P).all())
        same = P[1:] == P[:-1]
        assert bool((perm[1:][same] > perm[:-1][same]).all())                   # stability
        K = got["leaves"]
        cnt = got["counts"].to(torch.int64)
        assert int(K[0]) == 0 and int(cs.u64(K[-1:])[0]) == KEY_END
        assert int(cnt.sum()) == n
        delta = cs.u64(K)[1:] - cs.u64(K)[:-1]
        assert np.all((delta & (delta - np.uint64(1))) == 0)                    # powers of two ...
        assert np.all((np.log2(delta.astype(np.float64)).round().astype(np.int64) % 3) == 0)   # ... of 8
        assert np.all(cs.u64(K)[:-1] % delta == 0)
        cn = cs.u32(got["counts"])
        assert np.all((cn <= 64) | (delta == 1))
        assert (got["numLeaves"] - 1) % 7 == 0 and got["numNodes"] == got["numLeaves"] + (got["numLeaves"] - 1) // 7
        co = cs.u32(got["childOffsets"]); nc = cs.u32(got["nodeCount"])
        internal = np.flatnonzero(co)
        assert np.all(nc[internal] > 64)                                        # balanced
        pick = rng.choice(internal, 2000)
        for i in pick:
            assert int(nc[co[i]:co[i] + 8].sum()) == int(nc[i])
        # oracle on sampled outputs: leaf counts and the keys of sampled particles
        Ph = cs.u64(P)
        Kh = cs.u64(K)
        sel = rng.integers(0, got["numLeaves"], 5000)
        lo = np.searchsorted(Ph, Kh[sel], side="left")
        hi = np.searchsorted(Ph, Kh[sel + 1], side="left")
        hi[Kh[sel + 1] == np.uint64(KEY_END)] = n
        assert np.array_equal((hi - lo).astype(np.uint32), cn[sel])
        ids = rng.integers(0, n, 100000)
        boxh = box.cpu().numpy()
        assert np.array_equal(oracle.keys(x[ids], y[ids], z[ids], boxh), cs.u64(unsorted[ids]))
        prev = got["leaves"].clone()
    ctx.close()
