"""One rank's side of the distributed build of Sec. 6 (Eq. 11): orchestration only.

The particles are spread over the ranks of a ``torch.distributed`` process group (one process per GPU).  Every step of
the method runs in the library's kernels (``cs_countLeaves`` = f, ``cs_rebalance`` = g, ``cs_partitionLeaves``,
``cs_linkOctree``, ``cs_nodeCountsFromLeaves``); this module only strings those calls together and puts the paper's one
exchange step between them: ``f_glob = f_r o f`` with ``f_r`` "the element-wise sum of the counts arrays ... computed
with a single call to MPI_Allreduce" -- here ``dist.all_reduce(SUM)`` on the uint32 counts (NCCL on
the GPUs).  The bounding box needs a min / max all-reduce of six doubles first, and the common start array of the
rounds is broadcast from rank 0.

The kernels are passed in as callables (``count``, ``rebalance``) so that the multi-process host logic can be tested
on CPU with the ``gloo`` backend, where no CUDA kernel can run (tests/test_multirank_host_logic.py).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def world_size() -> int:
    return dist.get_world_size() if dist.is_available() and dist.is_initialized() else 1


def allreduce_box(box6: torch.Tensor) -> torch.Tensor:
    """{xmin, xmax, ymin, ymax, zmin, zmax} of all ranks' particles from the ranks' own boxes (exact: min / max)."""
    if world_size() == 1:
        return box6
    lo, hi = box6[0::2].contiguous(), box6[1::2].contiguous()
    dist.all_reduce(lo, op=dist.ReduceOp.MIN)
    dist.all_reduce(hi, op=dist.ReduceOp.MAX)
    out = torch.empty_like(box6)
    out[0::2], out[1::2] = lo, hi
    return out


def broadcast_leaves(leaves: torch.Tensor | None, device, src: int = 0) -> torch.Tensor:
    """The same start array on every rank: rank ``src``'s ``leaves`` (an int64 tensor of uint64 bit patterns)."""
    if world_size() == 1:
        return leaves
    size = torch.tensor([leaves.numel() if dist.get_rank() == src else 0], dtype=torch.int64, device=device)
    dist.broadcast(size, src=src)
    if dist.get_rank() != src:
        leaves = torch.empty(int(size.item()), dtype=torch.int64, device=device)
    else:
        leaves = leaves.contiguous()
    dist.broadcast(leaves, src=src)
    return leaves


def global_leaves(count, rebalance, start: torch.Tensor, max_rounds: int = 64):
    """Rounds of f_glob and g until a round changes nothing.

    count(K) -> this rank's counts N (an int32 tensor of uint32 bit patterns; f on the rank's own sorted keys);
    rebalance(K, N) -> (K', changed) (g on the summed counts: the same on every rank).
    Returns (K, N, rounds): the converged global leaf array, its global counts, and the number of rounds including
    the confirming one."""
    K = start
    for r in range(1, max_rounds + 1):
        N = count(K)
        if world_size() > 1:
            dist.all_reduce(N, op=dist.ReduceOp.SUM)          # f_r: uint32 sums (two's-complement wrap = uint32 wrap)
        Knew, changed = rebalance(K, N)
        if not changed:
            return K, N, r
        K = Knew
    raise RuntimeError(f"global leaf rounds did not converge in {max_rounds} rounds")


class GlobalTreeBuilder:
    """The whole distributed step on one rank: box, keys, sort (local) -> global leaves -> replicated linked octree,
    node counts and the SFC partition.  All buffers are allocated once."""

    def __init__(self, cs, ctx, n: int, bucket: int):
        self.cs, self.ctx, self.n, self.bucket = cs, ctx, int(n), int(bucket)
        dev = ctx.device
        cap = ctx.max_leaves
        self.box = torch.empty(6, dtype=torch.float64, device=dev)
        self.keys = torch.empty(self.n, dtype=torch.int64, device=dev)
        self.perm = torch.empty(self.n, dtype=torch.int32, device=dev)
        self.K = [torch.empty(cap + 1, dtype=torch.int64, device=dev) for _ in range(3)]
        self.N = torch.empty(cap, dtype=torch.int32, device=dev)
        self.localCounts = torch.empty(cap, dtype=torch.int32, device=dev)
        self.bounds = torch.empty(world_size() + 1, dtype=torch.int32, device=dev)

    def step(self, x, y, z):
        cs, ctx = self.cs, self.ctx
        rank = dist.get_rank() if world_size() > 1 else 0
        cs.computeBox(ctx, x, y, z, self.box)
        gbox = allreduce_box(self.box)
        cs.computeKeys(ctx, x, y, z, gbox, self.keys)
        cs.sortKeys(ctx, self.keys, self.perm)
        # common start: rank 0's own balanced tree (its particles are a sample of the global distribution, so the
        # global rounds only have to refine it by about log8(ranks) levels)
        start = None
        if rank == 0:
            start, _, _, _ = cs.buildLeaves(ctx, self.keys, self.bucket, leaves=self.K[2], counts=self.localCounts)
        start = broadcast_leaves(start, ctx.device)
        flip = [0]

        def count(K):
            return cs.countLeaves(ctx, self.keys, K, self.N[:K.numel() - 1])

        def rebalance(K, N):
            out = self.K[flip[0]]
            flip[0] ^= 1
            return cs.rebalance(ctx, K, N, self.bucket, newLeaves=out)

        K, N, rounds = global_leaves(count, rebalance, start)
        tree = cs.linkOctree(ctx, K)
        first, cnt = cs.nodeCountsFromLeaves(ctx, K, N, tree["prefixes"])
        bounds = cs.partitionLeaves(ctx, N, world_size(), self.bounds)
        tree.update(leaves=K, counts=N, nodeFirst=first, nodeCount=cnt, bounds=bounds, rounds=rounds,
                    numLeaves=K.numel() - 1, box6=gbox, keys=self.keys, perm=self.perm)
        return tree
