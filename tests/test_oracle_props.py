"""Pins of the oracle's node properties (O8 geometry, O9 centres of mass, O10 minimum-distance MAC): the first
row past the hot path.  Each pin is something other than the
oracle's own formula: hand values for the worked example of Fig. 2, closed forms, invariants, brute force.
"""
import numpy as np
import pytest

import oracle
from helpers import decode_key
from paper_2307_06345_b200 import workloads as W

L = 21


def fig2_tree():
    """Root with its third octant subdivided: 15 leaves, 17 nodes."""
    step1 = 1 << (3 * (L - 1))
    step2 = 1 << (3 * (L - 2))
    K = [c * step1 for c in range(2)] + [2 * step1 + c * step2 for c in range(8)] + [c * step1 for c in range(3, 8)]
    K.append(1 << 63)
    return oracle.link(np.array(K, dtype=np.uint64))


def test_geometry_of_the_fig2_example_by_hand():
    t = fig2_tree()
    box = np.array([0.0, 1.0, 0.0, 2.0, -1.0, 1.0])                    # edges 1, 2, 2
    c, h = oracle.node_geometry(t["prefixes"], box)
    # root
    assert c[:, 0].tolist() == [0.5, 1.0, 0.0] and h[:, 0].tolist() == [0.5, 1.0, 1.0]
    # level 1, octant digit = 4 x + 2 y + z (A3): node 1 + digit
    for digit in range(8):
        xb, yb, zb = (digit >> 2) & 1, (digit >> 1) & 1, digit & 1
        assert c[:, 1 + digit].tolist() == [0.25 + 0.5 * xb, 0.5 + 1.0 * yb, -0.5 + 1.0 * zb]
        assert h[:, 1 + digit].tolist() == [0.25, 0.5, 0.5]
    # level 2 under octant 2 (x = 0, y = 1, z = 0): nodes 9..16, prefixes 0o120..0o127
    assert [oct(int(p)) for p in t["prefixes"][9:17]] == [oct(0o120 + d) for d in range(8)]
    for digit in range(8):
        xb, yb, zb = (digit >> 2) & 1, (digit >> 1) & 1, digit & 1
        assert c[:, 9 + digit].tolist() == [0.125 + 0.25 * xb, 1.25 + 0.5 * yb, -0.75 + 0.5 * zb]
        assert h[:, 9 + digit].tolist() == [0.125, 0.25, 0.25]


def test_geometry_contains_the_particles_of_every_leaf():
    """Ties O8 to the keys: every particle lies inside the cell of the leaf that holds it (brute force)."""
    x, y, z = W.uniform(3000, -1.0, 1.0, 5)
    r = oracle.full_build(x, y, z, 8)
    c, h = oracle.node_geometry(r["prefixes"], r["box"])
    xs, ys, zs = x[r["perm"]], y[r["perm"]], z[r["perm"]]
    leaves = np.flatnonzero(r["childOffsets"] == 0)
    for i in leaves:
        f, k = int(r["nodeFirst"][i]), int(r["nodeCount"][i])
        for a, d in ((xs, 0), (ys, 1), (zs, 2)):
            if k:
                tol = 4e-16 * max(1.0, abs(c[d, i]))
                assert np.all(a[f:f + k] >= c[d, i] - h[d, i] - tol) and np.all(a[f:f + k] <= c[d, i] + h[d, i] + tol)
    # children tile their parent: centres at +- half of the child's size, half sizes halve
    internal = np.flatnonzero(r["childOffsets"])
    for i in internal[:200]:
        co = int(r["childOffsets"][i])
        assert np.allclose(h[:, co:co + 8], h[:, i:i + 1] / 2, rtol=0, atol=0)
        assert np.allclose(np.abs(c[:, co:co + 8] - c[:, i:i + 1]), h[:, co:co + 8], rtol=1e-15, atol=1e-15)


def test_geometry_agrees_with_the_decoded_leaf_keys():
    x, y, z = W.plummer(2000, 7)
    r = oracle.full_build(x, y, z, 4)
    c, h = oracle.node_geometry(r["prefixes"], r["box"])
    e = r["box"][1::2] - r["box"][0::2]
    for j in range(0, r["leaves"].size - 1, 37):
        i = int(r["leafToNode"][j])
        lvl = int(r["levels"][i])
        g = decode_key(r["leaves"][j])                                   # 21-bit grid coordinates of the leaf's corner
        for d in range(3):
            corner = r["box"][2 * d] + (g[d] >> (L - lvl)) * (e[d] / 2 ** lvl)
            assert c[d, i] - h[d, i] == pytest.approx(corner, rel=1e-14, abs=1e-14)


def test_centre_of_mass_closed_forms():
    x, y, z = W.uniform(20000, 0.0, 1.0, 11)
    r = oracle.full_build(x, y, z, 16)
    c, _ = oracle.node_geometry(r["prefixes"], r["box"])
    xs, ys, zs = x[r["perm"]], y[r["perm"]], z[r["perm"]]
    com = oracle.centers_of_mass(xs, ys, zs, r["nodeFirst"], r["nodeCount"], r["childOffsets"], c)
    # root = mean of all particles (any summation order agrees to rounding)
    assert com[:, 0] == pytest.approx([x.mean(), y.mean(), z.mean()], rel=1e-12)
    # every node = mean of its particle range (numpy's pairwise sum: independent of the oracle's order)
    rng = np.random.default_rng(0)
    for i in rng.integers(0, r["numNodes"], 300):
        f, k = int(r["nodeFirst"][i]), int(r["nodeCount"][i])
        if k:
            assert com[:, i] == pytest.approx([xs[f:f + k].mean(), ys[f:f + k].mean(), zs[f:f + k].mean()], rel=1e-12)
        else:
            assert com[:, i].tolist() == c[:, i].tolist()               # empty node: geometric centre (A26)
    # the centre of mass lies inside the node's cell
    _, h = oracle.node_geometry(r["prefixes"], r["box"])
    assert np.all(np.abs(com - c) <= h * (1 + 1e-12))


def test_centre_of_mass_two_particles_by_hand():
    x = np.array([0.0, 1.0, 0.25]); y = np.array([0.0, 1.0, 0.75]); z = np.array([0.0, 1.0, 0.5])
    r = oracle.full_build(x, y, z, 1)
    c, _ = oracle.node_geometry(r["prefixes"], r["box"])
    com = oracle.centers_of_mass(x[r["perm"]], y[r["perm"]], z[r["perm"]], r["nodeFirst"], r["nodeCount"],
                                 r["childOffsets"], c)
    assert com[:, 0] == pytest.approx([1.25 / 3, 1.75 / 3, 0.5], rel=1e-15)


def test_mac_special_cases_and_brute_force():
    # one cubic node of edge 1 centred at the origin
    c = np.zeros((3, 1)); h = np.full((3, 1), 0.5)
    far = np.array([10.0, 11.0, -0.5, 0.5, -0.5, 0.5])                   # gap 9.5 along x
    assert oracle.mac_min_distance(c, h, far, 0.5)[0] == 1               # 9.5 > 1 / 0.5
    assert oracle.mac_min_distance(c, h, far, 0.1)[0] == 0               # 9.5 < 1 / 0.1
    touching = np.array([0.5, 1.5, -0.5, 0.5, -0.5, 0.5])
    assert oracle.mac_min_distance(c, h, touching, 1e6)[0] == 0          # r_min = 0 never passes
    inside = np.array([-0.1, 0.1, -0.1, 0.1, -0.1, 0.1])
    assert oracle.mac_min_distance(c, h, inside, 1e6)[0] == 0
    # diagonal: gaps (3, 4, 0) -> r_min = 5; l = 1: passes iff theta > 0.2
    diag = np.array([3.5, 4.0, 4.5, 5.0, -0.2, 0.2])
    assert oracle.mac_min_distance(c, h, diag, 0.21)[0] == 1 and oracle.mac_min_distance(c, h, diag, 0.19)[0] == 0
    # brute force on a small tree: minimum distance between corner / edge samples of the two boxes
    x, y, z = W.uniform(400, 0.0, 1.0, 2)
    r = oracle.full_build(x, y, z, 4)
    cc, hh = oracle.node_geometry(r["prefixes"], r["box"])
    focus = np.array([0.1, 0.3, 0.2, 0.45, 0.6, 0.9])
    theta = 0.6
    got = oracle.mac_min_distance(cc, hh, focus, theta)
    t = np.linspace(0.0, 1.0, 9)
    fx, fy, fz = (focus[0] + t * (focus[1] - focus[0]), focus[2] + t * (focus[3] - focus[2]), focus[4] + t * (focus[5] - focus[4]))
    F = np.stack(np.meshgrid(fx, fy, fz, indexing="ij"), -1).reshape(-1, 3)
    for i in range(0, r["numNodes"], 3):
        nx, ny, nz = (cc[d, i] - hh[d, i] + t * 2 * hh[d, i] for d in range(3))
        N = np.stack(np.meshgrid(nx, ny, nz, indexing="ij"), -1).reshape(-1, 3)
        dmin = np.sqrt(((N[:, None, :] - F[None, :, :]) ** 2).sum(-1)).min()   # >= true r_min, equal when faces align
        l = 2 * hh[:, i].max()
        if got[i]:
            assert dmin > l / theta * (1 - 1e-12)                        # the sampled distance can only overestimate
        lo = np.maximum(np.abs(cc[:, i] - 0.5 * (focus[0::2] + focus[1::2])) - hh[:, i] - 0.5 * (focus[1::2] - focus[0::2]), 0)
        assert bool(got[i]) == bool(np.sqrt((lo ** 2).sum()) > l / theta) or abs(np.sqrt((lo ** 2).sum()) - l / theta) < 1e-12
