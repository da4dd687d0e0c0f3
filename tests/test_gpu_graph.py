"""cs_buildOctree replayed as one CUDA graph (cs_setGraphLimit): a call whose arguments repeat is captured and replayed;
every replay must give the oracle's tree for the data that is in the buffers AT THAT TIME (the graph holds pointers,
not data), in fresh look-back epochs, with the device-side sort decisions (gated redo) intact."""
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


def check(cs, got, ref, what):
    assert np.array_equal(cs.u64(got["keys"]), ref["sortedKeys"]), what + " keys"
    assert np.array_equal(cs.u32(got["perm"]), ref["perm"]), what + " perm"
    assert np.array_equal(cs.u64(got["leaves"]), ref["leaves"]), what + " leaves"
    assert np.array_equal(cs.u32(got["counts"]), ref["counts"]), what + " counts"
    assert np.array_equal(cs.u64(got["prefixes"]), ref["prefixes"]), what + " prefixes"
    for k in ("levels", "childOffsets", "parents", "levelRange", "leafToNode", "nodeToLeaf", "nodeFirst", "nodeCount"):
        assert np.array_equal(cs.u32(got[k]), ref[k]), what + " " + k


@pytest.mark.parametrize("n,bucket", [(1, 4), (777, 8), (65_536, 64), (300_001, 16)])
def test_replays_follow_the_data_in_the_buffers(cs, n, bucket):
    ctx = cs.Context(max_particles=n, max_leaves=8 * n + 64)
    bufs = cs.TreeBuffers(ctx, n)
    ctx.setSortMode(cs.SORT_DEFAULT)                             # one plan for all calls (the blobs are too dense for the short one)
    sets = [W.blobs(n, W.BASE_SEED + 200 + k, nblobs=16) for k in range(3)]
    dx, dy, dz = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
    launches = []
    for it in range(7):                                          # call 0 direct, call 1 captures, calls 2.. replay
        x, y, z = sets[it % 3]
        dx.copy_(torch.from_numpy(x)); dy.copy_(torch.from_numpy(y)); dz.copy_(torch.from_numpy(z))
        before = ctx.stageTimes()["launches"]
        got = cs.buildOctree(ctx, dx, dy, dz, bucket, buffers=bufs)
        launches.append(ctx.stageTimes()["launches"] - before)
        check(cs, got, oracle.full_build(x, y, z, bucket), f"call {it}")
    assert len(set(launches)) == 1 and launches[0] > 5           # a replay counts the kernels it launches
    ctx.close()


def test_graph_and_direct_calls_agree_and_modes_invalidate_the_graph(cs):
    n, bucket = 200_003, 64
    x, y, z = W.plummer(n, W.BASE_SEED + 211)
    ref = oracle.full_build(x, y, z, bucket)
    dx, dy, dz = (torch.from_numpy(a).cuda() for a in (x, y, z))
    ctx = cs.Context(max_particles=n, max_leaves=n // 2)
    bufs = cs.TreeBuffers(ctx, n)
    for it in range(3):
        check(cs, cs.buildOctree(ctx, dx, dy, dz, bucket, buffers=bufs), ref, f"graph {it}")
    ctx.setLeafMode(cs.LEAVES_ITERATIVE)                         # another mode: the captured graph no longer applies
    for it in range(3):
        got = cs.buildOctree(ctx, dx, dy, dz, bucket, buffers=bufs)
        check(cs, got, ref, f"iterative {it}")
        assert got["rounds"] == int(ref["levels"].max()) + 1
    ctx.setLeafMode(cs.LEAVES_AUTO)
    ctx.setSortMode(cs.SORT_PLAIN)
    for it in range(3):
        check(cs, cs.buildOctree(ctx, dx, dy, dz, bucket, buffers=bufs), ref, f"plain sort {it}")
    ctx.setSortMode(cs.SORT_AUTO)
    ctx.setGraphLimit(0)                                         # never replayed
    for it in range(2):
        check(cs, cs.buildOctree(ctx, dx, dy, dz, bucket, buffers=bufs), ref, f"direct {it}")
    ctx.setGraphLimit(1 << 22)
    ctx.setProfiling(True)                                       # stage timers need the separate launches
    for it in range(3):
        check(cs, cs.buildOctree(ctx, dx, dy, dz, bucket, buffers=bufs), ref, f"profiled {it}")
        assert ctx.stageTimes()["sort"] > 0
    ctx.close()


def test_replayed_builds_with_the_gated_redo_and_incremental_starts(cs):
    """Keys piled up below level 15 make the fifth pass raise its device flag: the redo kernel inside the graph must
    run, and the next call (plain plan, another graph) must agree.  Then time steps from the previous leaves."""
    n, bucket = 150_000, 32
    rng = np.random.default_rng(5)
    x = np.concatenate([rng.random(n // 2), 0.5 + 1e-7 * rng.random(n - n // 2)])
    y = np.concatenate([rng.random(n // 2), 0.5 + 1e-7 * rng.random(n - n // 2)])
    z = np.concatenate([rng.random(n // 2), 0.5 + 1e-7 * rng.random(n - n // 2)])
    ref = oracle.full_build(x, y, z, bucket)
    dx, dy, dz = (torch.from_numpy(a).cuda() for a in (x, y, z))
    ctx = cs.Context(max_particles=n, max_leaves=n)
    bufs = cs.TreeBuffers(ctx, n)
    for it in range(6):
        check(cs, cs.buildOctree(ctx, dx, dy, dz, bucket, buffers=bufs), ref, f"clustered {it}")
    # incremental: the previous leaves alias the output buffer; the number of leaves changes from step to step
    prev = None
    for it in range(5):
        x1, y1, z1 = W.displace(x, y, z, 1e-3, 900 + it)
        dx.copy_(torch.from_numpy(x1)); dy.copy_(torch.from_numpy(y1)); dz.copy_(torch.from_numpy(z1))
        got = cs.buildOctree(ctx, dx, dy, dz, bucket, buffers=bufs, prevLeaves=prev)
        check(cs, got, oracle.full_build(x1, y1, z1, bucket), f"step {it}")
        prev = got["leaves"]
    ctx.close()
