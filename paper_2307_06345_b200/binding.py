"""ctypes binding over the C ABI of include/cornerstone.h -- argument marshalling only.

Every function has the name of the C entry point without the ``cs_`` prefix and does nothing
but allocate output tensors (torch, on the context's device), pass raw pointers plus torch's
current CUDA stream, and translate the status code into an exception.  All computation runs
in the library's CUDA kernels.

Key / prefix arrays are ``torch.int64`` tensors holding the uint64 bit patterns; index arrays
are ``torch.int32`` tensors holding uint32 bit patterns (torch's unsigned dtypes are not needed
for plain storage).  ``u64(t)`` / ``u32(t)`` give numpy views of host copies.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
# CORNERSTONE_B200_LIB: another build of the same library (e.g. one compiled with other tile geometries)
LIB_PATH = os.environ.get("CORNERSTONE_B200_LIB") or os.path.join(_HERE, "libcornerstone_b200.so")

L = 21
KEY_END = 1 << 63
NUM_LEVEL_OFFSETS = 23
NO_LEAF = 0xFFFFFFFF
NUM_STAGES = 9
STAGE_NAMES = ("box", "keys", "sort", "leaves", "link", "counts", "sort_hist", "sort_passes", "sort_fixup")

CURVE_MORTON, CURVE_HILBERT = 0, 1
LEAVES_AUTO, LEAVES_ITERATIVE = 0, 1
SORT_AUTO, SORT_PLAIN, SORT_DEFAULT, SORT_SHORT, SORT_TINY = 0, 1, 2, 3, 4
OK, ERR_INVALID_ARG, ERR_CAPACITY, ERR_NOT_CORNERSTONE, ERR_NOT_CONVERGED, ERR_CUDA = range(6)
_STATUS_NAMES = {0: "CS_OK", 1: "CS_ERR_INVALID_ARG", 2: "CS_ERR_CAPACITY", 3: "CS_ERR_NOT_CORNERSTONE",
                 4: "CS_ERR_NOT_CONVERGED", 5: "CS_ERR_CUDA"}


class CornerstoneError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{_STATUS_NAMES.get(status, status)}: {message}")
        self.status = status


class OctreeBuffers(C.Structure):
    """Mirror of cs_octree_buffers."""
    _fields_ = [(name, C.c_void_p) for name in (
        "box6", "keys", "perm", "leaves", "counts", "prefixes", "levels", "childOffsets", "parents",
        "levelRange", "leafToNode", "nodeToLeaf", "nodeFirst", "nodeCount")] + [
        ("leafCapacity", C.c_uint32), ("nodeCapacity", C.c_uint32)]


class OctreeBuffers32(C.Structure):
    """Mirror of cs_octree_buffers32 (same members; keys, leaves and prefixes are uint32)."""
    _fields_ = OctreeBuffers._fields_


class OctreeSizes(C.Structure):
    """Mirror of cs_octree_sizes."""
    _fields_ = [("numLeaves", C.c_uint32), ("numNodes", C.c_uint32), ("rounds", C.c_uint32),
                ("converged", C.c_uint32)]


_lib = None


def lib():
    """Load libcornerstone_b200.so; there is no fallback if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build the CUDA library first "
            "(python -m paper_2307_06345_b200.build).  There is no CPU fallback.")
    l = C.CDLL(LIB_PATH)
    vp, u64, u32 = C.c_void_p, C.c_uint64, C.c_uint32
    sigs = {
        "cs_workspaceBytes": (C.c_size_t, [u64, u32]),
        "cs_create": (C.c_int, [C.POINTER(vp), C.c_int, u64, u32]),
        "cs_destroy": (None, [vp]),
        "cs_lastError": (C.c_char_p, [vp]),
        "cs_version": (C.c_char_p, []),
        "cs_setProfiling": (C.c_int, [vp, C.c_int]),
        "cs_stageTimes": (C.c_int, [vp, C.POINTER(C.c_float), C.POINTER(u64)]),
        "cs_setLeafMode": (C.c_int, [vp, C.c_int]),
        "cs_setSortMode": (C.c_int, [vp, C.c_int]),
        "cs_sortPasses": (C.c_int, [vp]),
        "cs_setGraphLimit": (C.c_int, [vp, u64]),
        "cs_computeBox": (C.c_int, [vp, vp, vp, vp, u64, vp, vp]),
        "cs_computeKeys": (C.c_int, [vp, vp, vp, vp, u64, vp, vp, vp]),
        "cs_computeKeysHilbert": (C.c_int, [vp, vp, vp, vp, u64, vp, vp, vp]),
        "cs_setCurve": (C.c_int, [vp, C.c_int]),
        "cs_sortKeys": (C.c_int, [vp, vp, vp, u64, vp]),
        "cs_buildLeaves": (C.c_int, [vp, vp, u64, u32, vp, u32, u32, vp, vp, u32, C.POINTER(u32), C.POINTER(u32), vp]),
        "cs_linkOctree": (C.c_int, [vp, vp, u32, vp, vp, vp, vp, vp, vp, vp, u32, C.POINTER(u32), vp]),
        "cs_nodeCounts": (C.c_int, [vp, vp, u64, vp, u32, vp, vp, u32, vp, vp, vp]),
        "cs_buildOctree": (C.c_int, [vp, vp, vp, vp, u64, u32, vp, u32, u32, C.POINTER(OctreeBuffers),
                                     C.POINTER(OctreeSizes), vp]),
        "cs_buildOctreeHost": (C.c_int, [vp, vp, vp, vp, u64, u32, C.POINTER(OctreeBuffers),
                                         C.POINTER(OctreeSizes), vp]),
        "cs_computeKeys32": (C.c_int, [vp, vp, vp, vp, u64, vp, C.c_int, vp, vp]),
        "cs_sortKeys32": (C.c_int, [vp, vp, vp, u64, vp]),
        "cs_buildLeaves32": (C.c_int, [vp, vp, u64, u32, vp, u32, u32, vp, vp, u32, C.POINTER(u32), C.POINTER(u32), vp]),
        "cs_linkOctree32": (C.c_int, [vp, vp, u32, vp, vp, vp, vp, vp, vp, vp, u32, C.POINTER(u32), vp]),
        "cs_buildOctree32": (C.c_int, [vp, vp, vp, vp, u64, u32, C.POINTER(OctreeBuffers32), C.POINTER(OctreeSizes), vp]),
        "cs_countLeaves": (C.c_int, [vp, vp, u64, vp, u32, vp, vp]),
        "cs_rebalance": (C.c_int, [vp, vp, vp, u32, u32, vp, u32, C.POINTER(u32), C.POINTER(u32), vp]),
        "cs_partitionLeaves": (C.c_int, [vp, vp, u32, u32, vp, vp]),
        "cs_partitionLeavesStatic": (C.c_int, [vp, u32, u32, vp, vp]),
        "cs_partitionLeavesStaticSetup": (C.c_int, []),
        "cs_partitionLeavesStaticMax": (u32, []),
        "cs_nodeCountsFromLeaves": (C.c_int, [vp, vp, vp, u32, vp, u32, vp, vp, vp]),
        "cs_gatherParticles": (C.c_int, [vp, vp, vp, vp, vp, u64, vp, vp, vp, vp]),
        "cs_nodeGeometry": (C.c_int, [vp, vp, u32, vp, vp, vp, vp]),
        "cs_nodeGeometryHilbert": (C.c_int, [vp, vp, u32, vp, vp, vp, vp]),
        "cs_nodeMassCenters": (C.c_int, [vp, vp, vp, vp, vp, vp, vp, vp, vp, u32, vp, vp]),
        "cs_macMinDistance": (C.c_int, [vp, vp, vp, u32, C.POINTER(C.c_double), C.c_double, vp, vp]),
    }
    for name, (res, args) in sigs.items():
        fn = getattr(l, name)
        fn.restype = res
        fn.argtypes = args
    _lib = l
    return l


def version() -> str:
    return lib().cs_version().decode()


def workspaceBytes(max_particles: int, max_leaves: int) -> int:
    return int(lib().cs_workspaceBytes(max_particles, max_leaves))


def _ptr(t):
    if t is None:
        return None
    return C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def u64(t) -> np.ndarray:
    """Host numpy uint64 view of an int64 tensor of key bit patterns."""
    return t.detach().cpu().numpy().view(np.uint64)


def u32(t) -> np.ndarray:
    return t.detach().cpu().numpy().view(np.uint32)


def from_u64(a, device) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.uint64).view(np.int64)).to(device)


def from_u32(a, device) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.uint32).view(np.int32)).to(device)


class Context:
    """Owns a cs_context (device workspace for up to max_particles / max_leaves)."""

    def __init__(self, max_particles: int, max_leaves: int, device: int = 0):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2307_06345_b200 needs a CUDA device (sm_100a); there is no CPU path")
        self.device = torch.device("cuda", device)
        self.max_particles = int(max_particles)
        self.max_leaves = int(max_leaves)
        self.max_nodes = self.max_leaves + (self.max_leaves - 1) // 7 + 1
        torch.cuda.init()
        with torch.cuda.device(self.device):
            torch.cuda.current_stream()          # make sure torch's primary context exists
            h = C.c_void_p()
            st = lib().cs_create(C.byref(h), device, self.max_particles, self.max_leaves)
        if st != OK:
            raise CornerstoneError(st, lib().cs_lastError(None).decode())
        self.handle = h

    def close(self):
        if getattr(self, "handle", None):
            lib().cs_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def check(self, st: int, allow=()):
        if st != OK and st not in allow:
            raise CornerstoneError(st, lib().cs_lastError(self.handle).decode())
        return st

    def setProfiling(self, enabled: bool):
        self.check(lib().cs_setProfiling(self.handle, 1 if enabled else 0))

    def setLeafMode(self, mode: int):
        """LEAVES_AUTO (one-pass fixpoint from the root) or LEAVES_ITERATIVE (always the rounds f, g)."""
        self.check(lib().cs_setLeafMode(self.handle, int(mode)))

    def setCurve(self, curve: int):
        """CURVE_MORTON (default) or CURVE_HILBERT: the curve buildOctree / buildOctreeHost compute keys on."""
        self.check(lib().cs_setCurve(self.handle, int(curve)))

    def setSortMode(self, mode: int):
        """SORT_AUTO (tiny, short, default plan, plain passes: whichever the input allows), SORT_DEFAULT (never the tiny
        or the short plan), SORT_SHORT / SORT_TINY (always that plan) or SORT_PLAIN."""
        self.check(lib().cs_setSortMode(self.handle, int(mode)))

    def setGraphLimit(self, max_particles: int):
        """buildOctree calls with at most this many particles are replayed as one CUDA graph (0: never)."""
        self.check(lib().cs_setGraphLimit(self.handle, int(max_particles)))

    def sortPasses(self) -> int:
        """Plain radix passes of the next sort (what the stage "sort_passes" times): 3, 4 or 7."""
        return int(lib().cs_sortPasses(self.handle))

    def stageTimes(self):
        ms = (C.c_float * NUM_STAGES)()
        launches = C.c_uint64(0)
        self.check(lib().cs_stageTimes(self.handle, ms, C.byref(launches)))
        d = {STAGE_NAMES[i]: float(ms[i]) for i in range(NUM_STAGES)}
        d["launches"] = int(launches.value)
        return d


def _i64(n, dev):
    return torch.empty(int(n), dtype=torch.int64, device=dev)


def _i32(n, dev):
    return torch.empty(int(n), dtype=torch.int32, device=dev)


def computeBox(ctx: Context, x, y, z, box6=None):
    if box6 is None:
        box6 = torch.empty(6, dtype=torch.float64, device=ctx.device)
    ctx.check(lib().cs_computeBox(ctx.handle, _ptr(x), _ptr(y), _ptr(z), x.numel(), _ptr(box6), _stream()))
    return box6


def computeKeys(ctx: Context, x, y, z, box6, keys=None):
    if keys is None:
        keys = _i64(x.numel(), ctx.device)
    ctx.check(lib().cs_computeKeys(ctx.handle, _ptr(x), _ptr(y), _ptr(z), x.numel(), _ptr(box6), _ptr(keys),
                                   _stream()))
    return keys


def computeKeysHilbert(ctx: Context, x, y, z, box6, keys=None):
    if keys is None:
        keys = _i64(x.numel(), ctx.device)
    ctx.check(lib().cs_computeKeysHilbert(ctx.handle, _ptr(x), _ptr(y), _ptr(z), x.numel(), _ptr(box6), _ptr(keys),
                                          _stream()))
    return keys


def sortKeys(ctx: Context, keys, perm=None):
    """Sorts ``keys`` in place; returns perm."""
    if perm is None:
        perm = _i32(keys.numel(), ctx.device)
    ctx.check(lib().cs_sortKeys(ctx.handle, _ptr(keys), _ptr(perm), keys.numel(), _stream()))
    return perm


def buildLeaves(ctx: Context, sortedKeys, bucketSize: int, prevLeaves=None, maxRounds: int = 0,
                leafCapacity: int | None = None, leaves=None, counts=None, allow_not_converged: bool = False):
    """Returns (leaves[numLeaves+1], counts[numLeaves], rounds, converged)."""
    cap = int(leafCapacity if leafCapacity is not None else ctx.max_leaves)
    if leaves is None:
        leaves = _i64(cap + 1, ctx.device)
    if counts is None:
        counts = _i32(cap, ctx.device)
    nl, rounds = C.c_uint32(0), C.c_uint32(0)
    prev_n = 0 if prevLeaves is None else prevLeaves.numel() - 1
    st = lib().cs_buildLeaves(ctx.handle, _ptr(sortedKeys), sortedKeys.numel(), bucketSize, _ptr(prevLeaves),
                              prev_n, maxRounds, _ptr(leaves), _ptr(counts), cap, C.byref(nl), C.byref(rounds),
                              _stream())
    ctx.check(st, allow=(ERR_NOT_CONVERGED,) if allow_not_converged else ())
    n = int(nl.value)
    return leaves[:n + 1], counts[:n], int(rounds.value), st == OK


def linkOctree(ctx: Context, leaves, nodeCapacity: int | None = None):
    """leaves: int64 tensor with numLeaves+1 keys.  Returns a dict of tensors (+ numNodes)."""
    nl = leaves.numel() - 1
    cap = int(nodeCapacity if nodeCapacity is not None else nl + max(nl - 1, 0) // 7 + 1)
    dev = ctx.device
    out = {"prefixes": _i64(cap, dev), "levels": _i32(cap, dev), "childOffsets": _i32(cap, dev),
           "parents": _i32(cap, dev), "levelRange": _i32(NUM_LEVEL_OFFSETS, dev), "leafToNode": _i32(max(nl, 1), dev),
           "nodeToLeaf": _i32(cap, dev)}
    nn = C.c_uint32(0)
    ctx.check(lib().cs_linkOctree(ctx.handle, _ptr(leaves), nl, _ptr(out["prefixes"]), _ptr(out["levels"]),
                                  _ptr(out["childOffsets"]), _ptr(out["parents"]), _ptr(out["levelRange"]),
                                  _ptr(out["leafToNode"]), _ptr(out["nodeToLeaf"]), cap, C.byref(nn), _stream()))
    n = int(nn.value)
    for k in ("prefixes", "levels", "childOffsets", "parents", "nodeToLeaf"):
        out[k] = out[k][:n]
    out["leafToNode"] = out["leafToNode"][:nl]
    out["numNodes"] = n
    return out


def nodeCounts(ctx: Context, sortedKeys, prefixes, leafCounts=None, nodeToLeaf=None):
    n = prefixes.numel()
    first, count = _i32(n, ctx.device), _i32(n, ctx.device)
    nl = 0 if leafCounts is None else leafCounts.numel()
    ctx.check(lib().cs_nodeCounts(ctx.handle, _ptr(sortedKeys), sortedKeys.numel(), _ptr(prefixes), n,
                                  _ptr(leafCounts), _ptr(nodeToLeaf), nl, _ptr(first), _ptr(count), _stream()))
    return first, count


class TreeBuffers:
    """Pre-allocated device outputs of a full build (so repeated builds allocate nothing)."""

    def __init__(self, ctx: Context, n: int, leafCapacity: int | None = None):
        dev = ctx.device
        self.n = int(n)
        self.leafCapacity = int(leafCapacity if leafCapacity is not None else ctx.max_leaves)
        self.nodeCapacity = self.leafCapacity + (self.leafCapacity - 1) // 7 + 1
        lc, nc = self.leafCapacity, self.nodeCapacity
        self.t = {
            "box6": torch.empty(6, dtype=torch.float64, device=dev), "keys": _i64(n, dev), "perm": _i32(n, dev),
            "leaves": _i64(lc + 1, dev), "counts": _i32(lc, dev), "prefixes": _i64(nc, dev), "levels": _i32(nc, dev),
            "childOffsets": _i32(nc, dev), "parents": _i32(nc, dev), "levelRange": _i32(NUM_LEVEL_OFFSETS, dev),
            "leafToNode": _i32(lc, dev), "nodeToLeaf": _i32(nc, dev), "nodeFirst": _i32(nc, dev),
            "nodeCount": _i32(nc, dev)}
        self.c = OctreeBuffers(**{k: v.data_ptr() for k, v in self.t.items()}, leafCapacity=lc, nodeCapacity=nc)


def buildOctree(ctx: Context, x, y, z, bucketSize: int, buffers: TreeBuffers | None = None, prevLeaves=None,
                maxRounds: int = 0, allow_not_converged: bool = False):
    """The whole path in one call (one synchronisation).  Returns a dict of tensor views."""
    n = x.numel()
    if buffers is None:
        buffers = TreeBuffers(ctx, n)
    sizes = OctreeSizes()
    prev_n = 0 if prevLeaves is None else prevLeaves.numel() - 1
    st = lib().cs_buildOctree(ctx.handle, _ptr(x), _ptr(y), _ptr(z), n, bucketSize, _ptr(prevLeaves), prev_n,
                              maxRounds, C.byref(buffers.c), C.byref(sizes), _stream())
    ctx.check(st, allow=(ERR_NOT_CONVERGED,) if allow_not_converged else ())
    nl, nn = int(sizes.numLeaves), int(sizes.numNodes)
    t = buffers.t
    out = {"box6": t["box6"], "keys": t["keys"], "perm": t["perm"], "leaves": t["leaves"][:nl + 1],
           "counts": t["counts"][:nl], "levelRange": t["levelRange"], "leafToNode": t["leafToNode"][:nl]}
    for k in ("prefixes", "levels", "childOffsets", "parents", "nodeToLeaf", "nodeFirst", "nodeCount"):
        out[k] = t[k][:nn]
    out.update(numLeaves=nl, numNodes=nn, rounds=int(sizes.rounds), converged=bool(sizes.converged))
    return out


class HostBuffers:
    """Pinned host arrays for cs_buildOctreeHost (end-to-end form)."""

    def __init__(self, n: int, leafCapacity: int, want=("leaves", "counts", "prefixes", "childOffsets",
                                                          "levelRange", "nodeFirst", "nodeCount")):
        self.leafCapacity = int(leafCapacity)
        self.nodeCapacity = self.leafCapacity + (self.leafCapacity - 1) // 7 + 1
        lc, nc = self.leafCapacity, self.nodeCapacity
        shapes = {"box6": (6, torch.float64), "keys": (n, torch.int64), "perm": (n, torch.int32),
                  "leaves": (lc + 1, torch.int64), "counts": (lc, torch.int32), "prefixes": (nc, torch.int64),
                  "levels": (nc, torch.int32), "childOffsets": (nc, torch.int32), "parents": (nc, torch.int32),
                  "levelRange": (NUM_LEVEL_OFFSETS, torch.int32), "leafToNode": (lc, torch.int32),
                  "nodeToLeaf": (nc, torch.int32), "nodeFirst": (nc, torch.int32), "nodeCount": (nc, torch.int32)}
        self.t = {k: torch.empty(shapes[k][0], dtype=shapes[k][1]).pin_memory() for k in want}
        self.c = OctreeBuffers(**{k: v.data_ptr() for k, v in self.t.items()}, leafCapacity=lc, nodeCapacity=nc)

    def bytes_back(self, n, nl, nn) -> int:
        per = {"box6": 48, "keys": 8 * n, "perm": 4 * n, "leaves": 8 * (nl + 1), "counts": 4 * nl,
               "prefixes": 8 * nn, "levels": 4 * nn, "childOffsets": 4 * nn, "parents": 4 * nn,
               "levelRange": 4 * NUM_LEVEL_OFFSETS, "leafToNode": 4 * nl, "nodeToLeaf": 4 * nn,
               "nodeFirst": 4 * nn, "nodeCount": 4 * nn}
        return sum(per[k] for k in self.t)


def buildOctreeHost(ctx: Context, x, y, z, bucketSize: int, host: HostBuffers):
    """x, y, z: HOST float64 tensors (pinned for full PCIe rate).  Results land in ``host``."""
    sizes = OctreeSizes()
    st = lib().cs_buildOctreeHost(ctx.handle, C.c_void_p(x.data_ptr()), C.c_void_p(y.data_ptr()),
                                  C.c_void_p(z.data_ptr()), x.numel(), bucketSize, C.byref(host.c),
                                  C.byref(sizes), _stream())
    ctx.check(st)
    return {"numLeaves": int(sizes.numLeaves), "numNodes": int(sizes.numNodes), "rounds": int(sizes.rounds)}


# ---- 32-bit keys, L = 10 (include/cornerstone.h, "32-bit keys") ------------------------------------------------------
# keys, leaves and prefixes are int32 tensors holding uint32 bit patterns

KEY_END32 = 1 << 30


def computeKeys32(ctx: Context, x, y, z, box6, curve: int = CURVE_MORTON, keys=None):
    if keys is None:
        keys = _i32(x.numel(), ctx.device)
    ctx.check(lib().cs_computeKeys32(ctx.handle, _ptr(x), _ptr(y), _ptr(z), x.numel(), _ptr(box6), int(curve), _ptr(keys),
                                     _stream()))
    return keys


def sortKeys32(ctx: Context, keys, perm=None):
    """Sorts ``keys`` (int32 tensor of 30-bit keys) in place; returns perm."""
    if perm is None:
        perm = _i32(keys.numel(), ctx.device)
    ctx.check(lib().cs_sortKeys32(ctx.handle, _ptr(keys), _ptr(perm), keys.numel(), _stream()))
    return perm


def buildLeaves32(ctx: Context, sortedKeys, bucketSize: int, prevLeaves=None, maxRounds: int = 0,
                  leafCapacity: int | None = None, allow_not_converged: bool = False):
    cap = int(leafCapacity if leafCapacity is not None else ctx.max_leaves)
    leaves, counts = _i32(cap + 1, ctx.device), _i32(cap, ctx.device)
    nl, rounds = C.c_uint32(0), C.c_uint32(0)
    prev_n = 0 if prevLeaves is None else prevLeaves.numel() - 1
    st = lib().cs_buildLeaves32(ctx.handle, _ptr(sortedKeys), sortedKeys.numel(), bucketSize, _ptr(prevLeaves), prev_n,
                                maxRounds, _ptr(leaves), _ptr(counts), cap, C.byref(nl), C.byref(rounds), _stream())
    ctx.check(st, allow=(ERR_NOT_CONVERGED,) if allow_not_converged else ())
    n = int(nl.value)
    return leaves[:n + 1], counts[:n], int(rounds.value), st == OK


def linkOctree32(ctx: Context, leaves):
    nl = leaves.numel() - 1
    cap = nl + max(nl - 1, 0) // 7 + 1
    dev = ctx.device
    out = {"prefixes": _i32(cap, dev), "levels": _i32(cap, dev), "childOffsets": _i32(cap, dev),
           "parents": _i32(cap, dev), "levelRange": _i32(NUM_LEVEL_OFFSETS, dev), "leafToNode": _i32(max(nl, 1), dev),
           "nodeToLeaf": _i32(cap, dev)}
    nn = C.c_uint32(0)
    ctx.check(lib().cs_linkOctree32(ctx.handle, _ptr(leaves), nl, _ptr(out["prefixes"]), _ptr(out["levels"]),
                                    _ptr(out["childOffsets"]), _ptr(out["parents"]), _ptr(out["levelRange"]),
                                    _ptr(out["leafToNode"]), _ptr(out["nodeToLeaf"]), cap, C.byref(nn), _stream()))
    n = int(nn.value)
    for k in ("prefixes", "levels", "childOffsets", "parents", "nodeToLeaf"):
        out[k] = out[k][:n]
    out["leafToNode"] = out["leafToNode"][:nl]
    out["numNodes"] = n
    return out


class TreeBuffers32:
    """Pre-allocated device outputs of cs_buildOctree32."""

    def __init__(self, ctx: Context, n: int, leafCapacity: int | None = None):
        dev = ctx.device
        self.leafCapacity = int(leafCapacity if leafCapacity is not None else ctx.max_leaves)
        self.nodeCapacity = self.leafCapacity + (self.leafCapacity - 1) // 7 + 1
        lc, nc = self.leafCapacity, self.nodeCapacity
        self.t = {
            "box6": torch.empty(6, dtype=torch.float64, device=dev), "keys": _i32(n, dev), "perm": _i32(n, dev),
            "leaves": _i32(lc + 1, dev), "counts": _i32(lc, dev), "prefixes": _i32(nc, dev), "levels": _i32(nc, dev),
            "childOffsets": _i32(nc, dev), "parents": _i32(nc, dev), "levelRange": _i32(NUM_LEVEL_OFFSETS, dev),
            "leafToNode": _i32(lc, dev), "nodeToLeaf": _i32(nc, dev), "nodeFirst": _i32(nc, dev),
            "nodeCount": _i32(nc, dev)}
        self.c = OctreeBuffers32(**{k: v.data_ptr() for k, v in self.t.items()}, leafCapacity=lc, nodeCapacity=nc)


def buildOctree32(ctx: Context, x, y, z, bucketSize: int, buffers: TreeBuffers32 | None = None):
    n = x.numel()
    if buffers is None:
        buffers = TreeBuffers32(ctx, n)
    sizes = OctreeSizes()
    ctx.check(lib().cs_buildOctree32(ctx.handle, _ptr(x), _ptr(y), _ptr(z), n, bucketSize, C.byref(buffers.c),
                                     C.byref(sizes), _stream()))
    nl, nn = int(sizes.numLeaves), int(sizes.numNodes)
    t = buffers.t
    out = {"box6": t["box6"], "keys": t["keys"], "perm": t["perm"], "leaves": t["leaves"][:nl + 1],
           "counts": t["counts"][:nl], "levelRange": t["levelRange"], "leafToNode": t["leafToNode"][:nl]}
    for k in ("prefixes", "levels", "childOffsets", "parents", "nodeToLeaf", "nodeFirst", "nodeCount"):
        out[k] = t[k][:nn]
    out.update(numLeaves=nl, numNodes=nn, rounds=int(sizes.rounds), converged=bool(sizes.converged))
    return out


# ---- the distributed build of Sec. 6: one rank's calls (include/cornerstone.h, "the distributed build") ------------------

def countLeaves(ctx: Context, sortedKeys, leaves, counts=None):
    """f alone: counts[i] = keys of sortedKeys in [leaves[i], leaves[i+1]).  No synchronisation."""
    nl = leaves.numel() - 1
    if counts is None:
        counts = _i32(nl, ctx.device)
    ctx.check(lib().cs_countLeaves(ctx.handle, _ptr(sortedKeys), sortedKeys.numel(), _ptr(leaves), nl, _ptr(counts),
                                   _stream()))
    return counts


def rebalance(ctx: Context, leaves, counts, bucketSize: int, newLeaves=None, leafCapacity: int | None = None):
    """g alone on (leaves, counts).  Returns (newLeaves[newNumLeaves + 1], changed)."""
    nl = leaves.numel() - 1
    cap = int(leafCapacity if leafCapacity is not None else ctx.max_leaves)
    if newLeaves is None:
        newLeaves = _i64(cap + 1, ctx.device)
    nn, ch = C.c_uint32(0), C.c_uint32(0)
    ctx.check(lib().cs_rebalance(ctx.handle, _ptr(leaves), _ptr(counts), nl, bucketSize, _ptr(newLeaves), cap,
                                 C.byref(nn), C.byref(ch), _stream()))
    return newLeaves[:int(nn.value) + 1], bool(ch.value)


def partitionLeaves(ctx: Context, counts, numRanks: int, bounds=None):
    """bounds[numRanks + 1]: rank r owns the leaves [bounds[r], bounds[r+1]).  No synchronisation."""
    if bounds is None:
        bounds = _i32(numRanks + 1, ctx.device)
    ctx.check(lib().cs_partitionLeaves(ctx.handle, _ptr(counts), counts.numel(), numRanks, _ptr(bounds), _stream()))
    return bounds


def partitionLeavesStaticMax() -> int:
    return int(lib().cs_partitionLeavesStaticMax())


def partitionLeavesStaticSetup():
    """Looks up the library's static scratch array on the current device (the entry point does so itself on first use)."""
    st = lib().cs_partitionLeavesStaticSetup()
    if st != OK:
        raise CornerstoneError(st, lib().cs_lastError(None).decode())


def partitionLeavesStatic(counts, numRanks: int, bounds):
    """cs_partitionLeaves without a context and without any allocation: the caller passes `bounds` (numRanks + 1 int32
    on the device of `counts`, which must be the current device); at most partitionLeavesStaticMax() leaves.  Calls
    share one scratch array in the library: do not let two of them overlap on the GPU."""
    st = lib().cs_partitionLeavesStatic(_ptr(counts), counts.numel(), numRanks, _ptr(bounds), _stream())
    if st != OK:
        raise CornerstoneError(st, lib().cs_lastError(None).decode())
    return bounds


def nodeCountsFromLeaves(ctx: Context, leaves, leafCounts, prefixes):
    n = prefixes.numel()
    first, count = _i32(n, ctx.device), _i32(n, ctx.device)
    ctx.check(lib().cs_nodeCountsFromLeaves(ctx.handle, _ptr(leaves), _ptr(leafCounts), leaves.numel() - 1, _ptr(prefixes), n,
                                            _ptr(first), _ptr(count), _stream()))
    return first, count


# ---- node properties on the linked octree (include/cornerstone.h, last section) ---------------------------

def gatherParticles(ctx: Context, x, y, z, perm):
    """Coordinates in SFC order: (xs, ys, zs) with xs[j] = x[perm[j]]."""
    out = [torch.empty_like(x) for _ in range(3)]
    ctx.check(lib().cs_gatherParticles(ctx.handle, _ptr(x), _ptr(y), _ptr(z), _ptr(perm), x.numel(), _ptr(out[0]),
                                       _ptr(out[1]), _ptr(out[2]), _stream()))
    return tuple(out)


def nodeGeometry(ctx: Context, prefixes, box6, curve: int = CURVE_MORTON):
    """(centers[3, n], halfSizes[3, n]) float64 tensors; curve = the curve the tree's keys lie on."""
    n = prefixes.numel()
    centers = torch.empty((3, n), dtype=torch.float64, device=ctx.device)
    half = torch.empty((3, n), dtype=torch.float64, device=ctx.device)
    fn = lib().cs_nodeGeometryHilbert if curve == CURVE_HILBERT else lib().cs_nodeGeometry
    ctx.check(fn(ctx.handle, _ptr(prefixes), n, _ptr(box6), _ptr(centers), _ptr(half), _stream()))
    return centers, half


def nodeMassCenters(ctx: Context, xs, ys, zs, tree, centers):
    """com[3, n] from the sorted coordinates and the dict returned by buildOctree."""
    n = tree["numNodes"]
    com = torch.empty((3, n), dtype=torch.float64, device=ctx.device)
    ctx.check(lib().cs_nodeMassCenters(ctx.handle, _ptr(xs), _ptr(ys), _ptr(zs), _ptr(tree["nodeFirst"]),
                                       _ptr(tree["nodeCount"]), _ptr(tree["childOffsets"]), _ptr(centers),
                                       _ptr(tree["levelRange"]), n, _ptr(com), _stream()))
    return com


def macMinDistance(ctx: Context, centers, halfSizes, focus6, theta: float):
    """uint8[n]: 1 where Eq. 12 holds against the focus box (6 host floats)."""
    n = centers.shape[1]
    out = torch.empty(n, dtype=torch.uint8, device=ctx.device)
    f = (C.c_double * 6)(*[float(v) for v in focus6])
    ctx.check(lib().cs_macMinDistance(ctx.handle, _ptr(centers), _ptr(halfSizes), n, f, float(theta), _ptr(out), _stream()))
    return out
