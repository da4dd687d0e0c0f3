"""GPU parity on BASELINE.json's configurations, through cs_buildOctree with pre-allocated
buffers (the launch configuration bench.py times).  Bit-exact against the oracle.

c1, c2 run in test_gpu_parity.py.  c3 (2^24, buckets 16 and 64), c4 (2^26, the headline; also on Hilbert keys) and c5
(2^28) run here at full size, every output array compared with the oracle's.  c5's 10 incremental
rebuilds run at 2^22 by default and, at 2^28, the full build + the first rebuild; all 10 rebuilds at
2^28 when CS_TEST_FULL_C5=1 (≈ 30 GB of host memory, about a quarter of an hour of oracle time).
"""
import os

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
    del ref
    # the same particles on the Hilbert curve, every array again
    refh = oracle.full_build(x, y, z, 64, curve="hilbert")
    ctx.setCurve(cs.CURVE_HILBERT)
    got = cs.buildOctree(ctx, dev(x), dev(y), dev(z), 64, buffers=bufs)
    ctx.setCurve(cs.CURVE_MORTON)
    check_against_oracle(cs, got, refh, "c4 on Hilbert keys")
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


def _compare_and_free(cs, got, ref, what):
    """check_against_oracle for 2^28 particles: one array at a time, releasing the oracle's copy as soon as it has been
    compared (the host holds the coordinates, the oracle's arrays and one device array's copy at any moment)."""
    assert got["numLeaves"] == ref["leaves"].size - 1, what
    assert got["numNodes"] == ref["numNodes"], what
    assert np.array_equal(got["box6"].cpu().numpy().view(np.uint64), ref["box"].view(np.uint64)), what + " box"
    for k, rk, view in (("keys", "sortedKeys", cs.u64), ("perm", "perm", cs.u32), ("leaves", "leaves", cs.u64),
                        ("counts", "counts", cs.u32), ("prefixes", "prefixes", cs.u64), ("levels", "levels", cs.u32),
                        ("childOffsets", "childOffsets", cs.u32), ("parents", "parents", cs.u32),
                        ("levelRange", "levelRange", cs.u32), ("leafToNode", "leafToNode", cs.u32),
                        ("nodeToLeaf", "nodeToLeaf", cs.u32), ("nodeFirst", "nodeFirst", cs.u32),
                        ("nodeCount", "nodeCount", cs.u32)):
        assert np.array_equal(view(got[k]), ref[rk]), f"{what} {k}"
        del ref[rk]


def test_config5_full_size_every_array(cs):
    """c5 at its full size, N = 2^28 (BASELINE.json configs[4]): the full build and the incremental rebuilds that start
    from the previous leaf array, EVERY output array compared with the oracle's.  By default the full
    build and the first rebuild (the oracle needs about a minute per 2^28 build on one host core); CS_TEST_FULL_C5=1
    runs all 10 rebuilds ("still check all 11 builds"), CS_TEST_C5_N overrides the size."""
    import time
    cfg = W.CONFIGS[4]
    n = int(os.environ.get("CS_TEST_C5_N", cfg.n))
    rebuilds = cfg.incremental_steps if os.environ.get("CS_TEST_FULL_C5") == "1" else 1
    x, y, z = cfg.generate(n)
    ctx = cs.Context(max_particles=n, max_leaves=n // 4)
    bufs = cs.TreeBuffers(ctx, n)
    prev = None
    for step in range(0, rebuilds + 1):
        t0 = time.perf_counter()
        if step:
            x, y, z = cfg.step(x, y, z, step)
        dx, dy, dz = dev(x), dev(y), dev(z)
        got = cs.buildOctree(ctx, dx, dy, dz, 64, buffers=bufs, prevLeaves=prev)
        del dx, dy, dz
        t1 = time.perf_counter()
        ref = oracle.full_build(x, y, z, 64)
        t2 = time.perf_counter()
        del ref["keys"]
        nl, nn, rounds = got["numLeaves"], got["numNodes"], got["rounds"]
        _compare_and_free(cs, got, ref, f"c5 2^28 step {step}")
        assert got["converged"]
        if step:
            assert rounds <= 4           # a small step needs one update (+ the confirming round)
        print(f"c5 n={n} step {step}: leaves={nl} nodes={nn} rounds={rounds} every array equal "
              f"(gpu+copies {t1 - t0:.1f} s, oracle {t2 - t1:.1f} s, compare {time.perf_counter() - t2:.1f} s)", flush=True)
        prev = got["leaves"].clone()
    ctx.close()
