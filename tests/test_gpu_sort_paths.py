"""GPU parity of cs_sortKeys on every path of cs_sort.cu against the oracle's stable sort (O3).

Default plan: 5 radix passes over the leading 45 bits, the last of which also orders the low 18 bits inside runs of
equal leading bits; short plan: 4 passes over the leading 36 bits, the low 27 ordered inside runs; tiny plan: 3 passes
over the leading 27 bits, the low 36 ordered inside runs.  A run longer than
257 elements raises the device flag and the 7 gated plain passes redo the sort.  cs_setSortMode(PLAIN) runs the 7
plain passes directly; AUTO moves between the three.  All of them must return the same (unique) keys and permutation,
bit for bit.
"""
import numpy as np
import pytest

import oracle
from paper_2307_06345_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

MAX_RUN = 257       # longest run the fix-up takes (kFixupMaxRun + 1)


@pytest.fixture(scope="module")
def cs():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2307_06345_b200 import binding
    return binding


@pytest.fixture()
def ctx(cs):
    c = cs.Context(max_particles=1 << 21, max_leaves=1 << 18)
    yield c
    c.close()


@pytest.fixture(params=["default", "short", "tiny"])
def plan(request, cs):
    """(sort mode, LOW): the plan whose last pass orders the low LOW bits inside runs of equal leading bits: the default
    plan (5 passes over bits 18..62), the short plan (4 passes over bits 27..62), the tiny plan (3 passes over bits
    36..62)."""
    return {"default": (cs.SORT_DEFAULT, 18), "short": (cs.SORT_SHORT, 27), "tiny": (cs.SORT_TINY, 36)}[request.param]


def check(cs, ctx, k, mode=0):
    """mode (SORT_AUTO, SORT_PLAIN, SORT_DEFAULT, SORT_SHORT) is set first (which also forgets an earlier redo); None
    leaves the context as it is."""
    if mode is not None:
        ctx.setSortMode(mode)
    P, perm = oracle.sort(k)
    dk = cs.from_u64(k, ctx.device)
    dperm = cs.sortKeys(ctx, dk)
    assert np.array_equal(cs.u64(dk), P), "sorted keys"
    assert np.array_equal(cs.u32(dperm), perm), "perm"


def keys_with_runs(rng, run_lengths, LOW, low_mode="random"):
    """Keys whose bits above LOW form runs of the given lengths, shuffled."""
    tops = rng.choice(1 << min(34, 63 - LOW), size=len(run_lengths), replace=False).astype(np.uint64)
    parts = []
    for t, r in zip(tops, run_lengths):
        if low_mode == "random":
            lo = rng.integers(0, 1 << LOW, r, dtype=np.uint64)
        elif low_mode == "few":                      # many equal whole keys inside the run
            lo = rng.integers(0, 3, r, dtype=np.uint64)
        else:                                        # all equal: only stability orders them
            lo = np.zeros(r, dtype=np.uint64)
        parts.append((t << np.uint64(LOW)) | lo)
    k = np.concatenate(parts)
    rng.shuffle(k)
    return k


@pytest.mark.parametrize("low_mode", ["random", "few", "equal"])
def test_fixup_orders_short_runs(cs, ctx, plan, low_mode):
    mode, LOW = plan
    rng = np.random.default_rng(11)
    runs = list(rng.integers(1, 40, 3000)) + [MAX_RUN - 1, MAX_RUN, 200, 256]
    check(cs, ctx, keys_with_runs(rng, runs, LOW, low_mode), mode)


@pytest.mark.parametrize("longest", [MAX_RUN, MAX_RUN + 1, MAX_RUN + 2, 300, 513, 5000])
def test_run_length_boundary_and_gated_redo(cs, ctx, plan, longest):
    """Runs of exactly the limit stay on the fix-up; one element more takes the gated 7 passes."""
    mode, LOW = plan
    rng = np.random.default_rng(longest)
    runs = [1] * 20000 + [longest] + list(rng.integers(1, 9, 2000))
    check(cs, ctx, keys_with_runs(rng, runs, LOW), mode)
    # the context is reusable afterwards (flag and tickets are reset per call)
    check(cs, ctx, keys_with_runs(rng, [1] * 9000 + [17, 3], LOW), mode)


def test_runs_at_the_ends_and_across_blocks(cs, ctx, plan):
    mode, LOW = plan
    rng = np.random.default_rng(3)
    n_runs = 600
    tops = np.sort(rng.choice(1 << min(34, 63 - LOW), size=n_runs, replace=False).astype(np.uint64))
    lens = rng.integers(100, MAX_RUN + 1, n_runs)            # long runs straddle every 256-thread block
    lens[0] = MAX_RUN
    lens[-1] = MAX_RUN
    k = np.concatenate([(t << np.uint64(LOW)) | rng.integers(0, 1 << LOW, r, dtype=np.uint64)
                        for t, r in zip(tops, lens)])
    rng.shuffle(k)
    check(cs, ctx, k, mode)


def test_one_giant_run_and_all_equal_keys(cs, ctx, plan):
    mode, LOW = plan
    rng = np.random.default_rng(4)
    k = (np.uint64(12345) << np.uint64(LOW)) | rng.integers(0, 1 << LOW, 50000, dtype=np.uint64)
    check(cs, ctx, k, mode)
    check(cs, ctx, np.full(30001, 0x7FFFFFFFFFFFFFFF, dtype=np.uint64), mode)
    check(cs, ctx, np.zeros(777, dtype=np.uint64), mode)


def test_plain_mode_equals_default(cs, ctx):
    rng = np.random.default_rng(8)
    for n in (1, 257, 6656, 6657, 123457):
        k = rng.integers(0, 1 << 63, n, dtype=np.uint64)
        for mode in (cs.SORT_PLAIN, cs.SORT_AUTO, cs.SORT_DEFAULT, cs.SORT_SHORT, cs.SORT_TINY):
            check(cs, ctx, k, mode)
    with pytest.raises(cs.CornerstoneError):
        ctx.setSortMode(7)


def test_build_switches_to_plain_passes_after_a_redo(cs, ctx):
    """Deeply clustered particles (more than 257 per level-15 cell): the full build still matches
    the oracle, through the gated redo the first time and through the plain passes afterwards."""
    rng = np.random.default_rng(21)
    n = 60000
    x = np.concatenate([rng.random(n - 4000), 0.5 + 1e-7 * rng.random(4000)])
    y = np.concatenate([rng.random(n - 4000), 0.5 + 1e-7 * rng.random(4000)])
    z = np.concatenate([rng.random(n - 4000), 0.5 + 1e-7 * rng.random(4000)])
    ref = oracle.full_build(x, y, z, 64)
    d = [torch.from_numpy(a).cuda() for a in (x, y, z)]
    ctx.setSortMode(cs.SORT_AUTO)
    plans = []
    for _ in range(20):
        plans.append(ctx.sortPasses())
        got = cs.buildOctree(ctx, d[0], d[1], d[2], 64)
        assert np.array_equal(cs.u64(got["keys"]), ref["sortedKeys"])
        assert np.array_equal(cs.u32(got["perm"]), ref["perm"])
        assert np.array_equal(cs.u64(got["leaves"]), ref["leaves"])
        assert np.array_equal(cs.u32(got["nodeCount"]), ref["nodeCount"])
    # the ladder of CS_SORT_AUTO: the tiny plan (2 plain passes + the fused last one), redone on the device; the short
    # plan (3 + 1) and the default plan (4 + 1), redone as well; then the 7 plain passes for 16 builds; then the default
    # plan is tried again (and redone again): one pathological step does not cost every later one
    tiny, short, default, plain = plans[0], plans[1], plans[2], plans[3]        # 2, 3, 4 and 7 with the 9-bit digits
    assert tiny + 1 == short and short + 1 == default and plain > default + 1
    assert plans == [tiny, short, default] + [plain] * 16 + [default]
    # CS_SORT_DEFAULT never tries the finer plans
    ctx.setSortMode(cs.SORT_DEFAULT)
    plans = []
    for _ in range(3):
        plans.append(ctx.sortPasses())
        got = cs.buildOctree(ctx, d[0], d[1], d[2], 64)
        assert np.array_equal(cs.u64(got["keys"]), ref["sortedKeys"]) and np.array_equal(cs.u32(got["perm"]), ref["perm"])
    assert plans == [default, plain, plain]
    ctx.setSortMode(cs.SORT_AUTO)


def test_auto_backs_off_from_the_finer_plans(cs, ctx):
    """More than 257 particles in a level-12 cell but none in a level-15 cell: the tiny and the short plan are redone
    once each, then the default plan serves (no redo, no plain passes).  More than 257 in a level-9 cell only: the short
    plan serves.  Uniform particles stay on the tiny plan."""
    rng = np.random.default_rng(22)
    n = 50000
    k = np.concatenate([rng.integers(0, 1 << 63, n, dtype=np.uint64),
                        (np.uint64(0x765432101) << np.uint64(27)) | rng.integers(0, 1 << 27, 2000, dtype=np.uint64)])
    rng.shuffle(k)
    ctx.setSortMode(cs.SORT_AUTO)
    tiny = ctx.sortPasses()
    plans = []
    for _ in range(7):
        plans.append(ctx.sortPasses())
        check(cs, ctx, k, mode=None)
    assert plans == [tiny, tiny + 1] + [tiny + 2] * 5
    k9 = np.concatenate([rng.integers(0, 1 << 63, n, dtype=np.uint64),
                         (np.uint64(0x3654321) << np.uint64(36)) | rng.integers(0, 1 << 36, 2000, dtype=np.uint64)])
    rng.shuffle(k9)
    ctx.setSortMode(cs.SORT_AUTO)
    plans = []
    for _ in range(5):
        plans.append(ctx.sortPasses())
        check(cs, ctx, k9, mode=None)
    assert plans == [tiny] + [tiny + 1] * 4
    ctx.setSortMode(cs.SORT_AUTO)
    u = rng.integers(0, 1 << 63, 200000, dtype=np.uint64)
    plans = []
    for _ in range(4):
        plans.append(ctx.sortPasses())
        check(cs, ctx, u, mode=None)
    assert plans == [tiny] * 4


def test_sort_keys_alone_learns_of_the_redo(cs, ctx):
    """cs_sortKeys never reads the control block; the redo flag follows the stream to the host and the next sort on the
    context takes the plain passes."""
    rng = np.random.default_rng(5)
    k = np.concatenate([rng.integers(0, 1 << 63, 50000, dtype=np.uint64),
                        (np.uint64(0x1234567) << np.uint64(30)) | rng.integers(0, 1 << 18, 3000, dtype=np.uint64)])
    rng.shuffle(k)
    ctx.setSortMode(cs.SORT_AUTO)
    tiny = ctx.sortPasses()                                     # 2 with the 9-bit digits
    check(cs, ctx, k)                                           # check() synchronises when it copies the result back
    assert ctx.sortPasses() == tiny + 1                         # the short plan
    check(cs, ctx, k, mode=None)
    assert ctx.sortPasses() == tiny + 2                         # the default plan
    check(cs, ctx, k, mode=None)
    assert ctx.sortPasses() > tiny + 3                          # 7: all digits
    check(cs, ctx, k, mode=None)
    ctx.setSortMode(cs.SORT_AUTO)
    assert ctx.sortPasses() == tiny


def test_workload_shapes(cs, ctx):
    for gen in (lambda: W.blobs(300001, W.BASE_SEED + 4, nblobs=50), lambda: W.plummer(200000, W.BASE_SEED + 2)):
        x, y, z = gen()
        ref = oracle.full_build(x, y, z, 64)
        check(cs, ctx, ref["keys"])


def test_unaligned_arrays(cs, ctx):
    """keys only 8-byte aligned / perm only 4-byte aligned."""
    rng = np.random.default_rng(13)
    k = rng.integers(0, 1 << 63, 40001, dtype=np.uint64)
    k[::7] = k[1::7][: k[::7].size]
    P, perm = oracle.sort(k[1:])
    dk = cs.from_u64(k, ctx.device)[1:]
    dperm = torch.empty(k.size + 1, dtype=torch.int32, device=ctx.device)[1:k.size]
    cs.sortKeys(ctx, dk, dperm)
    assert np.array_equal(cs.u64(dk), P) and np.array_equal(cs.u32(dperm), perm)


@pytest.mark.parametrize("group", [3, 40, 200])
def test_runs_that_are_not_neighbours_before_the_last_pass(cs, ctx, plan, group):
    """Keys that agree in bits LOW..53 but differ in the top digit are interleaved in the order the last pass
    reads (it is sorted by bits LOW..53 only), so the members of a run (equal bits LOW..62) are not neighbours
    there.  The tile cuts of that pass must not separate them: with groups this long every cut falls into one."""
    mode, LOW = plan
    rng = np.random.default_rng(100 + group)
    n_groups = 300000 // group
    mid = rng.choice(1 << (54 - LOW), size=n_groups, replace=False).astype(np.uint64)    # bits LOW..53
    mid = np.repeat(mid, group)
    top = rng.integers(0, 4, mid.size, dtype=np.uint64) * np.uint64(127)                 # 4 different top digits
    low = rng.integers(0, 1 << LOW, mid.size, dtype=np.uint64)
    k = (top << np.uint64(54)) | (mid << np.uint64(LOW)) | low
    k[::11] = k[1::11][: k[::11].size]                                                   # and some equal whole keys
    rng.shuffle(k)
    check(cs, ctx, k, mode)
