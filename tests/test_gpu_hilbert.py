"""GPU parity of the Hilbert keys (reading A28) against the oracle's O2h, bit for
bit: the key kernel alone and the whole path on Hilbert keys (H3-H10 run unchanged on them)."""
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


@pytest.mark.parametrize("n", [1, 2, 31, 1000, 70001, (1 << 20) + 3])
def test_hilbert_keys_equal_the_oracles(cs, n):
    x, y, z = W.plummer(n, 100 + n % 97)
    ctx = cs.Context(max_particles=n, max_leaves=1024)
    dx, dy, dz = dev(x), dev(y), dev(z)
    box = cs.computeBox(ctx, dx, dy, dz)
    got = cs.u64(cs.computeKeysHilbert(ctx, dx, dy, dz, box))
    assert np.array_equal(got, oracle.hilbert_keys(x, y, z, box.cpu().numpy()))
    ctx.close()


def test_hilbert_keys_of_every_cell_of_a_small_grid(cs):
    """All 32^3 cell centres of a grid aligned with the box: the keys, shifted down to 5 levels, are a permutation of
    [0, 8^5) whose consecutive members are face neighbours (checked here on the GPU's own output)."""
    k = 5
    g = (np.arange(1 << k) + 0.5) / (1 << k)
    x, y, z = (a.ravel().copy() for a in np.meshgrid(g, g, g, indexing="ij"))
    box = np.array([0.0, 1.0, 0.0, 1.0, 0.0, 1.0])
    ctx = cs.Context(max_particles=x.size, max_leaves=1024)
    keys = cs.u64(cs.computeKeysHilbert(ctx, dev(x), dev(y), dev(z), dev(box)))
    assert np.array_equal(keys, oracle.hilbert_keys(x, y, z, box))
    cell = keys >> np.uint64(3 * (21 - k))
    assert np.array_equal(np.sort(cell), np.arange(8 ** k, dtype=np.uint64))
    order = np.argsort(cell)
    step = sum(np.abs(np.diff(c[order])) for c in (x, y, z)) * (1 << k)
    assert np.allclose(step, 1.0)
    ctx.close()


def test_unaligned_and_user_box(cs):
    n = 50001
    x, y, z = W.uniform(n + 1, -3.0, 5.0, 9)
    x, y, z = x[1:], y[1:], z[1:]                               # 8-byte aligned only: the scalar path of the kernel
    box = np.array([-1.0, 2.0, -3.0, 5.0, 0.0, 0.0])            # particles outside clamp; flat z maps to 0
    ctx = cs.Context(max_particles=n, max_leaves=1024)
    dx, dy, dz = (dev(np.concatenate([[0.0], a]))[1:] for a in (x, y, z))
    got = cs.u64(cs.computeKeysHilbert(ctx, dx, dy, dz, dev(box)))
    assert np.array_equal(got, oracle.hilbert_keys(x, y, z, box))
    ctx.close()


@pytest.mark.parametrize("cfg_i,n,bucket", [(0, None, 64), (1, None, 64), (3, 1 << 21, 16)])
def test_full_build_on_hilbert_keys(cs, cfg_i, n, bucket):
    cfg = W.CONFIGS[cfg_i]
    x, y, z = cfg.generate(n)
    ref = oracle.full_build(x, y, z, bucket, curve="hilbert")
    ctx = cs.Context(max_particles=x.size, max_leaves=max(4096, x.size // 4))
    ctx.setCurve(cs.CURVE_HILBERT)
    got = cs.buildOctree(ctx, dev(x), dev(y), dev(z), bucket)
    assert np.array_equal(cs.u64(got["keys"]), ref["sortedKeys"])
    assert np.array_equal(cs.u32(got["perm"]), ref["perm"])
    assert np.array_equal(cs.u64(got["leaves"]), ref["leaves"])
    assert np.array_equal(cs.u32(got["counts"]), ref["counts"])
    assert np.array_equal(cs.u64(got["prefixes"]), ref["prefixes"])
    for k in ("levels", "childOffsets", "parents", "levelRange", "leafToNode", "nodeToLeaf", "nodeFirst", "nodeCount"):
        assert np.array_equal(cs.u32(got[k]), ref[k]), k
    # the Morton tree of the same particles has the same shape (same cells, another order inside every level)
    ctx.setCurve(cs.CURVE_MORTON)
    mort = cs.buildOctree(ctx, dev(x), dev(y), dev(z), bucket)
    assert mort["numLeaves"] == got["numLeaves"] and mort["numNodes"] == got["numNodes"]
    assert np.array_equal(cs.u32(mort["levelRange"]), cs.u32(got["levelRange"]))
    ctx.close()


def test_node_properties_of_a_hilbert_tree(cs):
    """cs_nodeGeometryHilbert against O8h, and the rest of the node properties (centres of mass, MAC) on a tree of
    Hilbert keys: cells of deep and shallow nodes, empty leaves (they take their cell's centre)."""
    n, bucket = 150_001, 16
    x, y, z = W.blobs(n, W.BASE_SEED + 91, nblobs=12)
    ref = oracle.full_build(x, y, z, bucket, curve="hilbert")
    ctx = cs.Context(max_particles=n, max_leaves=n)
    ctx.setCurve(cs.CURVE_HILBERT)
    dx, dy, dz = dev(x), dev(y), dev(z)
    tree = cs.buildOctree(ctx, dx, dy, dz, bucket)
    assert np.array_equal(cs.u64(tree["prefixes"]), ref["prefixes"])
    centers, half = cs.nodeGeometry(ctx, tree["prefixes"], tree["box6"], curve=cs.CURVE_HILBERT)
    rc, rh = oracle.node_geometry(ref["prefixes"], ref["box"], curve="hilbert")
    assert np.array_equal(centers.cpu().numpy().view(np.uint64), rc.view(np.uint64))
    assert np.array_equal(half.cpu().numpy().view(np.uint64), rh.view(np.uint64))
    mc, _ = cs.nodeGeometry(ctx, tree["prefixes"], tree["box6"])           # read as Morton digits: other cells
    assert not np.array_equal(mc.cpu().numpy(), rc)
    xs, ys, zs = cs.gatherParticles(ctx, dx, dy, dz, tree["perm"])
    com = cs.nodeMassCenters(ctx, xs, ys, zs, tree, centers)
    rcom = oracle.centers_of_mass(x[ref["perm"]], y[ref["perm"]], z[ref["perm"]], ref["nodeFirst"], ref["nodeCount"],
                                  ref["childOffsets"], rc)
    assert np.array_equal(com.cpu().numpy().view(np.uint64), rcom.view(np.uint64))
    focus = [0.1, 0.2, 0.3, 0.4, 0.5, 0.6]
    mac = cs.macMinDistance(ctx, centers, half, focus, 0.6)
    assert np.array_equal(mac.cpu().numpy(), oracle.mac_min_distance(rc, rh, np.array(focus), 0.6))
    ctx.close()
