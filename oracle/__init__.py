"""CPU oracle for the Cornerstone octree hot path -- TEST INFRASTRUCTURE ONLY.

Thin ctypes/numpy wrapper around ``cornerstone_oracle.cpp`` (plain single-threaded
C++17 written from PAPER.md).  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package;
the product (``paper_2307_06345_b200``) never does, and this package never imports
the product's CUDA binding.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build as _build

L = 21
KEY_END = 1 << 63

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.orc_box.restype = C.c_int
        _lib.orc_keys.restype = None
        _lib.orc_sort.restype = None
        _lib.orc_round.restype = C.c_int64
        _lib.orc_leaves_iterative.restype = C.c_int64
        _lib.orc_leaves_topdown.restype = C.c_int64
        _lib.orc_link.restype = C.c_int64
        _lib.orc_node_counts.restype = None
        _lib.orc_node_geometry.restype = None
        _lib.orc_node_geometry_hilbert.restype = None
        _lib.orc_centers_of_mass.restype = None
        _lib.orc_mac_min_distance.restype = None
        _lib.orc_set_L.restype = C.c_int
        _lib.orc_hilbert_keys.restype = None
        _lib.orc_hilbert_from_grid.restype = None
        _lib.orc_global_round.restype = C.c_int64
        _lib.orc_partition.restype = None
    return _lib


class key_levels:
    """``with oracle.key_levels(10): ...`` -- run the oracle with L octal digits per key (L = 10 for 32-bit
    keys, 21 for 64-bit keys).  Keys stay in uint64 arrays; 8^L is the terminal element of K."""

    def __init__(self, levels: int):
        self.levels = int(levels)

    def __enter__(self):
        global L, KEY_END
        self.old = lib().orc_set_L(self.levels)
        if self.old < 0:
            raise ValueError("L must be in 1..21")
        L, KEY_END = self.levels, 1 << (3 * self.levels)
        return self

    def __exit__(self, *a):
        global L, KEY_END
        lib().orc_set_L(self.old)
        L, KEY_END = self.old, 1 << (3 * self.old)


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _u64(a):
    return np.ascontiguousarray(a, dtype=np.uint64)


def _u32(a):
    return np.ascontiguousarray(a, dtype=np.uint32)


def box(x, y, z):
    """O1: {xmin, xmax, ymin, ymax, zmin, zmax}."""
    x, y, z = _f64(x), _f64(y), _f64(z)
    out = np.empty(6, dtype=np.float64)
    rc = lib().orc_box(_p(x), _p(y), _p(z), C.c_uint64(x.size), _p(out))
    if rc != 0:
        raise ValueError("box of an empty particle set")
    return out


def keys(x, y, z, box6):
    """O2: 64-bit Morton keys."""
    x, y, z, box6 = _f64(x), _f64(y), _f64(z), _f64(box6)
    out = np.empty(x.size, dtype=np.uint64)
    lib().orc_keys(_p(x), _p(y), _p(z), C.c_uint64(x.size), _p(box6), _p(out))
    return out


def hilbert_keys(x, y, z, box6):
    """O2h: Hilbert keys of the particles (reading A28), L octal digits."""
    x, y, z, box6 = _f64(x), _f64(y), _f64(z), _f64(box6)
    out = np.empty(x.size, dtype=np.uint64)
    lib().orc_hilbert_keys(_p(x), _p(y), _p(z), C.c_uint64(x.size), _p(box6), _p(out))
    return out


def hilbert_from_grid(gx, gy, gz, levels):
    """O2h on integer grid points of the 2^levels grid."""
    gx, gy, gz = _u32(gx), _u32(gy), _u32(gz)
    out = np.empty(gx.size, dtype=np.uint64)
    lib().orc_hilbert_from_grid(_p(gx), _p(gy), _p(gz), C.c_uint64(gx.size), C.c_int(levels), _p(out))
    return out


def sort(keys_in):
    """O3: stable sort; returns (sortedKeys, perm) with perm the gather map."""
    keys_in = _u64(keys_in)
    out = np.empty_like(keys_in)
    perm = np.empty(keys_in.size, dtype=np.uint32)
    lib().orc_sort(_p(keys_in), C.c_uint64(keys_in.size), _p(out), _p(perm))
    return out, perm


def round_(P, K, bucket_size, cap=None):
    """O5: one f + g round.  Returns dict(N, O, Oprime, K) (K is None on overflow)."""
    P, K = _u64(P), _u64(K)
    nl = K.size - 1
    if cap is None:
        cap = 8 * nl
    N = np.empty(nl, dtype=np.uint32)
    O = np.empty(nl, dtype=np.uint32)
    Op = np.empty(nl + 1, dtype=np.uint32)
    Kout = np.empty(cap + 1, dtype=np.uint64)
    nn = lib().orc_round(_p(P), C.c_uint64(P.size), _p(K), C.c_uint32(nl), C.c_uint32(bucket_size),
                         _p(N), _p(O), _p(Op), _p(Kout), C.c_uint32(cap))
    return {"N": N, "O": O, "Oprime": Op, "K": None if nn < 0 else Kout[:nn + 1].copy()}


def global_round(shards, K, bucket_size, cap=None):
    """O11: one round of the distributed build: f on every shard (each a sorted key array), the
    element-wise sum f_r, then g.  Returns dict(N, O, Oprime, K) like round_ (N = the summed counts)."""
    shards = [_u64(p) for p in shards]
    K = _u64(K)
    nl = K.size - 1
    if cap is None:
        cap = 8 * nl
    Pall = np.concatenate(shards) if shards else np.empty(0, dtype=np.uint64)
    start = np.zeros(len(shards) + 1, dtype=np.uint64)
    start[1:] = np.cumsum([p.size for p in shards])
    N = np.empty(nl, dtype=np.uint32)
    O = np.empty(nl, dtype=np.uint32)
    Op = np.empty(nl + 1, dtype=np.uint32)
    Kout = np.empty(cap + 1, dtype=np.uint64)
    nn = lib().orc_global_round(_p(Pall), _p(start), C.c_uint32(len(shards)), _p(K), C.c_uint32(nl),
                                C.c_uint32(bucket_size), _p(N), _p(O), _p(Op), _p(Kout), C.c_uint32(cap))
    return {"N": N, "O": O, "Oprime": Op, "K": None if nn < 0 else Kout[:nn + 1].copy()}


def partition(counts, n_ranks):
    """O12: leaf-index bounds b_0 = 0 <= ... <= b_{n_ranks} = n_l of the SFC domain decomposition (reading A29)."""
    counts = _u32(counts)
    out = np.empty(n_ranks + 1, dtype=np.uint32)
    lib().orc_partition(_p(counts), C.c_uint32(counts.size), C.c_uint32(n_ranks), _p(out))
    return out


def leaves_iterative(P, bucket_size, K_start=None, max_rounds=0, cap=None):
    """O5b: iterate f, g from K_start (default: the root {0, 8^21}).

    Returns (K, counts, rounds, converged)."""
    P = _u64(P)
    if K_start is None:
        K_start = np.array([0, 1 << (3 * L)], dtype=np.uint64)
    K_start = _u64(K_start)
    user_cap = cap is not None
    if cap is None:
        cap = max(64, 8 * (K_start.size - 1), P.size // 2 + 64)
    while True:
        Kout = np.empty(cap + 1, dtype=np.uint64)
        counts = np.empty(cap, dtype=np.uint32)
        rounds = C.c_uint32(0)
        conv = C.c_int(0)
        nl = lib().orc_leaves_iterative(_p(P), C.c_uint64(P.size), C.c_uint32(bucket_size), _p(K_start),
                                        C.c_uint32(K_start.size - 1), C.c_uint32(max_rounds), _p(Kout),
                                        _p(counts), C.c_uint32(cap), C.byref(rounds), C.byref(conv))
        if nl >= 0:
            return Kout[:nl + 1].copy(), counts[:nl].copy(), int(rounds.value), bool(conv.value)
        if user_cap or cap > (1 << 31):
            raise OverflowError("leaf capacity exceeded")
        cap *= 4


def leaves_topdown(P, bucket_size, cap=None):
    """O4: the balanced cornerstone array by top-down construction.  Returns (K, counts)."""
    P = _u64(P)
    user_cap = cap is not None
    if cap is None:
        cap = P.size // 4 + 64
    while True:
        Kout = np.empty(cap + 1, dtype=np.uint64)
        counts = np.empty(cap, dtype=np.uint32)
        nl = lib().orc_leaves_topdown(_p(P), C.c_uint64(P.size), C.c_uint32(bucket_size), _p(Kout),
                                      _p(counts), C.c_uint32(cap))
        if nl >= 0:
            return Kout[:nl + 1].copy(), counts[:nl].copy()
        if user_cap:
            raise OverflowError("leaf capacity exceeded")
        cap = -nl


def link(K):
    """O6: fully linked octree.  Returns a dict of arrays."""
    K = _u64(K)
    nl = K.size - 1
    if nl < 1 or (nl - 1) % 7 != 0:
        raise ValueError("not a closed octree: (n_l - 1) mod 7 != 0")
    n = nl + (nl - 1) // 7
    out = {
        "prefixes": np.empty(n, dtype=np.uint64),
        "levels": np.empty(n, dtype=np.uint32),
        "childOffsets": np.empty(n, dtype=np.uint32),
        "parents": np.empty(n, dtype=np.uint32),
        "levelRange": np.empty(L + 2, dtype=np.uint32),
        "leafToNode": np.empty(nl, dtype=np.uint32),
        "nodeToLeaf": np.empty(n, dtype=np.uint32),
    }
    nn = lib().orc_link(_p(K), C.c_uint32(nl), _p(out["prefixes"]), _p(out["levels"]), _p(out["childOffsets"]),
                        _p(out["parents"]), _p(out["levelRange"]), _p(out["leafToNode"]), _p(out["nodeToLeaf"]))
    if nn != n:
        raise ValueError("K is not a cornerstone array of a closed octree")
    out["numNodes"] = n
    return out


def node_counts(leaf_counts, tree):
    """O7: (nodeFirst, nodeCount) by recursive summation over the links."""
    leaf_counts = _u32(leaf_counts)
    n = tree["numNodes"]
    first = np.empty(n, dtype=np.uint32)
    count = np.empty(n, dtype=np.uint32)
    lib().orc_node_counts(_p(leaf_counts), C.c_uint32(leaf_counts.size), _p(_u32(tree["childOffsets"])),
                          _p(_u32(tree["nodeToLeaf"])), C.c_uint32(n), _p(first), _p(count))
    return first, count


def full_build(x, y, z, bucket_size, curve="morton"):
    """The whole path, stage by stage; returns a dict with every array."""
    b = box(x, y, z)
    k = keys(x, y, z, b) if curve == "morton" else hilbert_keys(x, y, z, b)
    P, perm = sort(k)
    K, counts = leaves_topdown(P, bucket_size)
    tree = link(K)
    first, count = node_counts(counts, tree)
    out = {"box": b, "keys": k, "sortedKeys": P, "perm": perm, "leaves": K, "counts": counts,
           "nodeFirst": first, "nodeCount": count}
    out.update(tree)
    return out


def node_geometry(prefixes, box6, curve="morton"):
    """O8 / O8h: (centers[3, n], halfSizes[3, n]) of the nodes' cells in the bounding box; the prefixes are
    placeholder-bit keys on the Morton or on the Hilbert curve (reading A28)."""
    prefixes, box6 = _u64(prefixes), _f64(box6)
    n = prefixes.size
    centers = np.empty((3, n), dtype=np.float64)
    half = np.empty((3, n), dtype=np.float64)
    fn = lib().orc_node_geometry if curve == "morton" else lib().orc_node_geometry_hilbert
    fn(_p(prefixes), C.c_uint32(n), _p(box6), _p(centers), _p(half))
    return centers, half


def centers_of_mass(xs, ys, zs, node_first, node_count, child_offsets, centers):
    """O9: com[3, n] by an upward pass over the linked tree; xs, ys, zs are the coordinates in SORTED order."""
    xs, ys, zs, centers = _f64(xs), _f64(ys), _f64(zs), _f64(centers)
    node_first, node_count, child_offsets = _u32(node_first), _u32(node_count), _u32(child_offsets)
    n = node_first.size
    com = np.empty((3, n), dtype=np.float64)
    lib().orc_centers_of_mass(_p(xs), _p(ys), _p(zs), _p(node_first), _p(node_count), _p(child_offsets), _p(centers),
                              C.c_uint32(n), _p(com))
    return com


def mac_min_distance(centers, half_sizes, focus6, theta):
    """O10: Eq. 12 against an axis-aligned focus box; uint8[n], 1 = fulfilled."""
    centers, half_sizes, focus6 = _f64(centers), _f64(half_sizes), _f64(focus6)
    n = centers.shape[1]
    out = np.empty(n, dtype=np.uint8)
    lib().orc_mac_min_distance(_p(centers), _p(half_sizes), C.c_uint32(n), _p(focus6), C.c_double(theta), _p(out))
    return out
