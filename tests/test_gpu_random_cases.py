"""GPU parity on randomly drawn small cases: sizes around the tile sizes of every kernel, bucket sizes from 1 to
1024, and particle sets with the structures that steer the data-dependent paths (uniform, tight clusters deeper
than level 15, exact duplicates, points on a coarse lattice, a flat dimension, cells repeated across octants).  Every output of cs_buildOctree
must equal the oracle's, bit for bit.  Seeds are fixed: the cases are the same in every run.
"""
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


@pytest.fixture(scope="module")
def ctx(cs):
    c = cs.Context(max_particles=1 << 19, max_leaves=1 << 22)
    yield c
    c.close()


def draw(rng, n, kind):
    if kind == "uniform":
        p = rng.random((3, n))
    elif kind == "clusters":                       # most particles in a few cells far below level 15
        k = max(1, n // 3000)
        centres = rng.random((3, k))
        which = rng.integers(0, k, n)
        sigma = 10.0 ** rng.uniform(-8, -3, k)
        p = centres[:, which] + sigma[which] * rng.standard_normal((3, n))
        bg = rng.random(n) < 0.2
        p[:, bg] = rng.random((3, int(bg.sum())))
        p = np.clip(p, 0.0, np.nextafter(1.0, 0.0))
    elif kind == "duplicates":                     # few distinct points, many copies of each
        k = max(1, n // 50)
        pts = rng.random((3, k))
        p = pts[:, rng.integers(0, k, n)]
    elif kind == "lattice":                        # coordinates on multiples of 1/64: quotients hit integers exactly
        p = rng.integers(0, 65, (3, n)) / 64.0
    elif kind == "flat":                           # one dimension without extent
        p = rng.random((3, n))
        p[1, :] = 0.25
    elif kind == "twins":                          # same cell path on levels 4..15, other octants on levels 1..3:
        m = max(1, n // 6)                         # keys equal in bits 18..53 that differ in the top digit
        mid = rng.integers(0, 1 << 12, (3, m))     # grid bits 6..17 of each dimension
        pick = rng.integers(0, m, n)
        g = (rng.integers(0, 8, (3, n)) << 18) | (mid[:, pick] << 6) | rng.integers(0, 64, (3, n))
        p = (g + 0.5) / float(1 << 21)
        if n >= 2:                                 # pin the box to [0, 1]: the grid above is then the key grid
            p[:, 0] = 0.0
            p[:, 1] = 1.0
    else:
        raise ValueError(kind)
    return tuple(np.ascontiguousarray(p[d], dtype=np.float64) for d in range(3))


SIZES = (1, 2, 63, 64, 65, 257, 2047, 2048, 2049, 6335, 6336, 6337, 6655, 6656, 6657, 13313, 40000, 100003, 262144,
         400001)
KINDS = ("uniform", "clusters", "duplicates", "lattice", "flat", "twins")
BUCKETS = (1, 2, 8, 64, 300, 1024)


def cases():
    rng = np.random.default_rng(20230706)
    out = []
    for i, n in enumerate(SIZES):
        for kind in KINDS:
            out.append((n, kind, int(BUCKETS[int(rng.integers(0, len(BUCKETS)))]), int(rng.integers(0, 1 << 30)), i))
    return out


@pytest.mark.parametrize("n,kind,bucket,seed,_i", cases())
def test_random_case_matches_oracle(cs, ctx, n, kind, bucket, seed, _i):
    rng = np.random.default_rng(seed)
    x, y, z = draw(rng, n, kind)
    ref = oracle.full_build(x, y, z, bucket)
    d = [torch.from_numpy(a).cuda() for a in (x, y, z)]
    ctx.setSortMode(cs.SORT_AUTO)                  # a redo in an earlier case switched the context to the plain passes
    got = cs.buildOctree(ctx, d[0], d[1], d[2], bucket)
    what = f"n={n} {kind} bucket={bucket}"
    assert np.array_equal(got["box6"].cpu().numpy().view(np.uint64), ref["box"].view(np.uint64)), what + " box"
    assert np.array_equal(cs.u64(got["keys"]), ref["sortedKeys"]), what + " sorted keys"
    assert np.array_equal(cs.u32(got["perm"]), ref["perm"]), what + " perm"
    assert np.array_equal(cs.u64(got["leaves"]), ref["leaves"]), what + " leaves"
    assert np.array_equal(cs.u32(got["counts"]), ref["counts"]), what + " counts"
    assert np.array_equal(cs.u64(got["prefixes"]), ref["prefixes"]), what + " prefixes"
    for k in ("levels", "childOffsets", "parents", "levelRange", "leafToNode", "nodeToLeaf", "nodeFirst", "nodeCount"):
        assert np.array_equal(cs.u32(got[k]), ref[k]), what + " " + k
