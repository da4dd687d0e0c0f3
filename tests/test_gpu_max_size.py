"""The largest input that fits on one B200 beside its outputs and the workspace: n = 2^31 + 12345 particles (48 GiB of
coordinates, 126 GiB in all), so that particle indices use bit 31 and every 32-bit quantity of the path is near its
limit.  No oracle at this size (it would need 100 GB and ten minutes): the result is checked by the properties that
hold at any size.  The coordinates are drawn on the device (seeded torch generator): 48 GiB do not come through PCIe
in a test."""
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def test_build_of_2_to_the_31_particles_keeps_every_invariant():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    if torch.cuda.get_device_properties(0).total_memory < 170 * 2 ** 30:
        pytest.skip("needs 170 GB of device memory")
    from paper_2307_06345_b200 import binding as cs
    torch.cuda.empty_cache()
    if torch.cuda.mem_get_info()[0] < 140 * 2 ** 30:
        pytest.skip("needs 140 GB of free device memory")
    n, bucket = (1 << 31) + 12345, 64
    dev = torch.device("cuda")
    gen = torch.Generator(device=dev)
    gen.manual_seed(230706345)
    x, y, z = (torch.rand(n, dtype=torch.float64, device=dev, generator=gen) for _ in range(3))
    m = n // 16                                              # a dense clump: the tree is 19 levels deep
    x[:m] = 0.3 + 1e-3 * x[:m]; y[:m] = 0.6 + 1e-3 * y[:m]; z[:m] = 0.1 + 1e-3 * z[:m]
    ctx = cs.Context(max_particles=n, max_leaves=n // 8)
    tree = cs.buildOctree(ctx, x, y, z, bucket, buffers=cs.TreeBuffers(ctx, n))
    keys, perm = tree["keys"], tree["perm"]
    chunk = 1 << 28
    # P ascending (keys < 2^63, so the signed comparison of the bit patterns is the unsigned one)
    for a in range(0, n - 1, chunk):
        b = min(n - 1, a + chunk)
        assert bool((keys[a + 1:b + 1] >= keys[a:b]).all())
    # perm is a permutation of 0 .. n-1 (indices above 2^31 included)
    seen = torch.zeros(n, dtype=torch.bool, device=dev)
    for a in range(0, n, chunk):
        seen[perm[a:a + chunk].to(torch.int64) & 0xFFFFFFFF] = True
    assert bool(seen.all())
    del seen
    # sorted slot j holds the key of particle perm[j]: keys of a sample recomputed with cs_computeKeys
    s = torch.randint(0, n, (1 << 22,), device=dev, generator=gen)
    pi = perm[s].to(torch.int64) & 0xFFFFFFFF
    again = cs.computeKeys(ctx, x[pi].contiguous(), y[pi].contiguous(), z[pi].contiguous(), tree["box6"])
    assert bool((again == keys[s]).all())
    # stable: equal neighbours keep their original order
    eq = keys[1:chunk] == keys[0:chunk - 1]
    p0, p1 = (perm[a:a + chunk - 1].to(torch.int64) & 0xFFFFFFFF for a in (0, 1))
    assert bool((p1[eq] > p0[eq]).all())
    # Eq. 2 and the counts
    K, N = tree["leaves"], tree["counts"]
    nl, nn = tree["numLeaves"], tree["numNodes"]
    assert int(K[0]) == 0 and int(K[-1]) == -(1 << 63)        # 8^21 = 2^63 as a bit pattern
    d = (K[1:] - K[:-1])[:-1]                                 # the last gap wraps in int64; it ends at 2^63
    assert bool((d > 0).all()) and bool(((d & (d - 1)) == 0).all()) and bool(((K[:-2] & (d - 1)) == 0).all())
    cnt = N.to(torch.int64)
    assert int(cnt.sum()) == n
    assert bool(((cnt <= bucket) | (d.new_tensor(1) == torch.cat([d, d.new_ones(1)]))).all())   # except at depth 21
    assert (nl - 1) % 7 == 0 and nn == nl + (nl - 1) // 7
    nc = tree["nodeCount"].to(torch.int64) & 0xFFFFFFFF
    co = tree["childOffsets"].to(torch.int64)
    assert int(nc[0]) == n and int(tree["nodeFirst"][0]) == 0
    internal = torch.nonzero(co[: 1 << 20]).flatten()         # parents = sum of their children
    kids = nc[(co[internal].unsqueeze(1) + torch.arange(8, device=dev)).flatten()].view(-1, 8).sum(1)
    assert bool((kids == nc[internal]).all())
    assert bool((nc[internal] > bucket).all())                # internal nodes hold more than N_crit
    ctx.close()
    del tree, keys, perm, x, y, z, K, N, cnt, nc, co, d
    torch.cuda.empty_cache()
