"""GPU parity of the node properties (cs_gatherParticles, cs_nodeGeometry, cs_nodeMassCenters, cs_macMinDistance)
against the oracle's O8-O10, bit for bit: both sides fix the same operation order (A25-A27) and no
floating-point operation is contracted.
"""
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


@pytest.fixture(scope="module")
def ctx(cs):
    c = cs.Context(max_particles=1 << 21, max_leaves=1 << 21)
    yield c
    c.close()


def bits(a):
    return np.ascontiguousarray(a, dtype=np.float64).view(np.uint64)


CASES = [("uniform", 1, 64), ("uniform", 2, 1), ("uniform", 5000, 16), ("plummer", 100003, 64), ("blobs", 300001, 64),
         ("blobs", 1 << 20, 8), ("duplicates", 40000, 4)]


def draw(kind, n):
    if kind == "uniform":
        return W.uniform(n, -1.0, 1.0, 17)
    if kind == "plummer":
        return W.plummer(n, 18)
    if kind == "blobs":
        return W.blobs(n, 19, nblobs=40)
    rng = np.random.default_rng(20)                       # few distinct points: deep, mostly empty siblings
    pts = rng.random((3, 60))
    return tuple(np.ascontiguousarray(pts[d, rng.integers(0, 60, n)]) for d in range(3))


@pytest.mark.parametrize("kind,n,bucket", CASES)
def test_node_properties_match_oracle(cs, ctx, kind, n, bucket):
    x, y, z = draw(kind, n)
    ref = oracle.full_build(x, y, z, bucket)
    d = [torch.from_numpy(a).cuda() for a in (x, y, z)]
    tree = cs.buildOctree(ctx, d[0], d[1], d[2], bucket)
    assert np.array_equal(cs.u64(tree["prefixes"]), ref["prefixes"])

    xs, ys, zs = cs.gatherParticles(ctx, d[0], d[1], d[2], tree["perm"])
    rx, ry, rz = x[ref["perm"]], y[ref["perm"]], z[ref["perm"]]
    for got, want in ((xs, rx), (ys, ry), (zs, rz)):
        assert np.array_equal(bits(got.cpu().numpy()), bits(want)), "gather"

    centers, half = cs.nodeGeometry(ctx, tree["prefixes"], tree["box6"])
    rc, rh = oracle.node_geometry(ref["prefixes"], ref["box"])
    assert np.array_equal(bits(centers.cpu().numpy()), bits(rc)), "centers"
    assert np.array_equal(bits(half.cpu().numpy()), bits(rh)), "half sizes"

    com = cs.nodeMassCenters(ctx, xs, ys, zs, tree, centers)
    rcom = oracle.centers_of_mass(rx, ry, rz, ref["nodeFirst"], ref["nodeCount"], ref["childOffsets"], rc)
    assert np.array_equal(bits(com.cpu().numpy()), bits(rcom)), "centres of mass"

    box = ref["box"]
    lo, e = box[0::2], box[1::2] - box[0::2]
    for frac0, frac1, theta in (((0.1, 0.2, 0.3), (0.3, 0.5, 0.4), 0.5), ((0.0, 0.0, 0.0), (1.0, 1.0, 1.0), 0.8),
                                ((0.7, 0.7, 0.7), (0.7, 0.7, 0.7), 0.3), ((-2.0, 0.4, 0.4), (-1.5, 0.6, 0.6), 1.0)):
        focus = np.empty(6)
        focus[0::2] = lo + np.array(frac0) * e
        focus[1::2] = lo + np.array(frac1) * e
        got = cs.macMinDistance(ctx, centers, half, focus, theta).cpu().numpy()
        want = oracle.mac_min_distance(rc, rh, focus, theta)
        assert np.array_equal(got, want), f"MAC theta={theta}"


def test_argument_checks(cs, ctx):
    x, y, z = W.uniform(1000, 0.0, 1.0, 1)
    d = [torch.from_numpy(a).cuda() for a in (x, y, z)]
    tree = cs.buildOctree(ctx, d[0], d[1], d[2], 16)
    centers, half = cs.nodeGeometry(ctx, tree["prefixes"], tree["box6"])
    with pytest.raises(cs.CornerstoneError):
        cs.macMinDistance(ctx, centers, half, [0, 1, 0, 1, 0, 1], 0.0)
    with pytest.raises(cs.CornerstoneError):                                  # in place is refused
        cs.lib().cs_gatherParticles and ctx.check(cs.lib().cs_gatherParticles(
            ctx.handle, cs._ptr(d[0]), cs._ptr(d[1]), cs._ptr(d[2]), cs._ptr(tree["perm"]), 1000, cs._ptr(d[0]),
            cs._ptr(d[1]), cs._ptr(d[2]), cs._stream()))
