"""cs_partitionLeavesStatic (include/cornerstone.h): the SFC partition for callers that must not allocate.  No context,
scratch in a fixed __device__ array of the library.  Its bounds must equal cs_partitionLeaves' (and the oracle's O12),
bit for bit, on calls in a row that share the scratch array.  Collected last on purpose (the file name): the suite
runs with pytest -x."""
import numpy as np
import pytest

import oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cs():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2307_06345_b200 import binding
    return binding


def counts_like_a_tree(rng, nl, hi):
    """leaf counts: mostly below the bucket size, some empty leaves, a few heavy ones (sum may pass 2^32)"""
    N = rng.integers(0, 65, nl, dtype=np.uint32)
    N[rng.random(nl) < 0.2] = 0
    heavy = rng.integers(0, nl, max(1, nl // 1000))
    N[heavy] = rng.integers(0, hi, heavy.size, dtype=np.uint32)
    return N


def test_static_partition_equals_the_context_path_on_calls_in_a_row(cs):
    rng = np.random.default_rng(20230706)
    ctx = cs.Context(max_particles=1024, max_leaves=1 << 22)
    # a large array (1465 tiles, total above 2^32), then small ones that leave most of the scratch stale, then large again
    cases = [(3_000_001, 1 << 24, 7), (5000, 100, 5), (1, 50, 3), (2049, 1 << 31, 64), (3_000_001, 1 << 24, 1000),
             (4096, 1, 2), (777_777, 4000, 148)]
    for it, (nl, hi, R) in enumerate(cases):
        N = counts_like_a_tree(rng, nl, hi)
        if nl == 4096:
            N[:] = 0                                             # no particles at all: every inner bound is 0
        d = torch.from_numpy(N.view(np.int32)).cuda()
        ref = cs.u32(cs.partitionLeaves(ctx, d, R))              # the existing path (context workspace)
        assert np.array_equal(ref, oracle.partition(N, R)), f"case {it}: the context path against O12"
        bounds = torch.full((R + 1,), -1, dtype=torch.int32, device="cuda")
        again = torch.full((R + 1,), -1, dtype=torch.int32, device="cuda")
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        cs.partitionLeavesStatic(d, R, bounds)                   # two calls in a row on the same stream
        cs.partitionLeavesStatic(d, R, again)
        torch.cuda.synchronize()
        if it >= 1:                                              # once the kernel is loaded, calls take no device memory
            assert torch.cuda.mem_get_info()[0] == free_before, f"case {it}: device memory changed"
        assert np.array_equal(cs.u32(bounds), ref), f"case {it}: first call"
        assert np.array_equal(cs.u32(again), ref), f"case {it}: second call"
    ctx.close()


def test_static_partition_on_another_stream_and_after_setup(cs):
    rng = np.random.default_rng(11)
    cs.partitionLeavesStaticSetup()
    N = counts_like_a_tree(rng, 123_457, 5000)
    d = torch.from_numpy(N.view(np.int32)).cuda()
    ref = oracle.partition(N, 9)
    bounds = torch.empty(10, dtype=torch.int32, device="cuda")
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        for _ in range(3):
            cs.partitionLeavesStatic(d, 9, bounds)
    s.synchronize()
    assert np.array_equal(cs.u32(bounds), ref)


def test_static_partition_rejects_what_does_not_fit(cs):
    limit = cs.partitionLeavesStaticMax()
    assert limit == 1 << 24
    d = torch.zeros(8, dtype=torch.int32, device="cuda")
    bounds = torch.full((4,), -1, dtype=torch.int32, device="cuda")

    class Huge:                                                  # numel() beyond the limit; the pointer is never read
        def data_ptr(self):
            return d.data_ptr()

        def numel(self):
            return limit + 1

    with pytest.raises(cs.CornerstoneError) as e:
        cs.partitionLeavesStatic(Huge(), 3, bounds)
    assert e.value.status == cs.ERR_CAPACITY and "exceeds the static scratch" in str(e.value)
    with pytest.raises(cs.CornerstoneError) as e:
        cs.partitionLeavesStatic(d, 0, bounds)
    assert e.value.status == cs.ERR_INVALID_ARG
    torch.cuda.synchronize()
    assert (bounds == -1).all()                                  # nothing was enqueued
    cs.partitionLeavesStatic(d, 3, bounds)                       # and the entry point still works afterwards
    assert cs.u32(bounds).tolist() == [0, 0, 0, 8]


def test_static_partition_at_its_maximum_size(cs):
    rng = np.random.default_rng(5)
    nl = cs.partitionLeavesStaticMax()                           # 8192 tiles: the whole scratch array
    N = counts_like_a_tree(rng, nl, 1 << 20)
    d = torch.from_numpy(N.view(np.int32)).cuda()
    bounds = torch.empty(33, dtype=torch.int32, device="cuda")
    cs.partitionLeavesStatic(d, 32, bounds)
    assert np.array_equal(cs.u32(bounds), oracle.partition(N, 32))
