// H9 linked octree and H10 node counts.
//
// The paper generates the internal nodes from K on all levels in parallel (steps 1-2,
// PAPER.md:156-157), then radix-sorts the node keys into breadth-first order (step 3) and finds
// level offsets and first children by binary search (steps 4-5).  The result is canonical
// (ascending placeholder-bit key, reading A16), and it can be reached without the 64-bit sort
// and without searches:
//
//   * Walk the leaf boundaries j = 0..n_l-1.  The nodes whose key range STARTS at K_j are the
//     leaf j (level hi_j = L - log8(K_{j+1} - K_j)) and its ancestors that are not ancestors of
//     leaf j-1, i.e. the internal nodes of levels lo_j .. hi_j - 1 with
//     lo_j = (number of leading octal digits shared by K_j - 1 and K_j) + 1   (lo_0 = 0).
//     Every node of the tree starts at exactly one boundary, so this enumerates all n nodes, and
//     inside one level it enumerates them in SFC order.
//   * Hence index(node) = LO[level] + (number of level-`level` nodes starting at boundaries < j):
//     a 22-bin stable split, done with per-level ballots inside a warp, a scan over the warps
//     of a tile and a decoupled look-back over tiles.
//   * The children of the k-th internal node of level l (SFC order) are the 8 nodes
//     LO[l+1] + 8k .. + 8k + 7, because level l+1 consists of exactly those sibling groups in
//     the same order.  So CO = LO[l+1] + 8 * (rank among the internal nodes of level l):
//     a second set of 22 counters, no search.
//
// Pass A counts nodes per level (-> LO, numNodes) and validates Eq. 2; pass B ranks and writes.
#include "cs_device.cuh"

namespace cs {

constexpr int kLevels = kL + 1;                  // 22 levels: 0..21
constexpr int kLinkWarps = kLinkBlock / 32;

// levels of the nodes starting at boundary j: internal lo..hi-1, leaf hi.  Returns false if the
// gap violates Eq. 2.
__device__ __forceinline__ bool boundaryLevels(u64 Kj, u64 Kn, u32 j, int& lo, int& hi)
{
    const u64 delta = Kn - Kj;
    if (Kn <= Kj || !isPowerOf8(delta) || (Kj & (delta - 1))) return false;
    hi = levelOfDelta(delta);
    if (j == 0) lo = 0;
    else {
        const u64 x = (Kj - 1) ^ Kj;                          // Kj > 0 here
        lo = (__clzll((long long)x) - 1) / 3 + 1;             // 63-bit keys: bit 63 is never set
    }
    return lo <= hi;
}

__device__ __forceinline__ u32 numLeavesOf(const u32* dNumLeaves, u32 hNumLeaves)
{
    return dNumLeaves ? *dNumLeaves : hNumLeaves;
}

// ---- pass A: nodes per level --------------------------------------------------------------------
__global__ void __launch_bounds__(kLinkBlock)
    linkCountKernel(DeviceCtrl* ctrl, const u64* __restrict__ K, const u32* dNumLeaves, u32 hNumLeaves)
{
    __shared__ u32 sCnt[kLinkBins];
    __shared__ u32 sStop;
    if (threadIdx.x == 0) {                                   // one read per CTA: uniform decision
        const u32 st = *(const volatile u32*)&ctrl->status;
        sStop = (st == CS_ERR_CAPACITY || st == CS_ERR_NOT_CORNERSTONE) ? 1u : 0u;
    }
    if (threadIdx.x < kLinkBins) sCnt[threadIdx.x] = 0;
    __syncthreads();
    if (sStop) return;
    const u32 nl = numLeavesOf(dNumLeaves, hNumLeaves);
    const u32 lane = laneId();
    bool bad = false;
    const u32 stride = gridDim.x * kLinkBlock;
    const u32 rounds = (nl + stride - 1) / stride;
    for (u32 it = 0; it < rounds; ++it) {
        const u32 j = it * stride + blockIdx.x * kLinkBlock + threadIdx.x;
        int lo = 1, hi = 0;                                   // empty range for j >= nl
        if (j < nl) {
            const u64 Kj = K[j], Kn = K[j + 1];
            if (!boundaryLevels(Kj, Kn, j, lo, hi)) { bad = true; lo = 1; hi = 0; }
            if (j == 0 && Kj != 0) bad = true;
            if (j == nl - 1 && Kn != kKeyEnd) bad = true;
        }
        int wlo = lo <= hi ? lo : kLevels, whi = lo <= hi ? hi : -1;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            wlo = min(wlo, __shfl_xor_sync(kFull, wlo, o));
            whi = max(whi, __shfl_xor_sync(kFull, whi, o));
        }
        for (int l = wlo; l <= whi; ++l) {
            const u32 bAll = __ballot_sync(kFull, lo <= l && l <= hi);
            const u32 bInt = __ballot_sync(kFull, lo <= l && l < hi);
            if (lane == 0) {
                if (bAll) atomicAdd(&sCnt[l], __popc(bAll));
                if (bInt) atomicAdd(&sCnt[kLevels + l], __popc(bInt));
            }
        }
    }
    if (nl == 0) bad = true;
    __syncthreads();
    if (threadIdx.x < kLinkBins && sCnt[threadIdx.x]) atomicAdd(&ctrl->levelTotals[threadIdx.x], sCnt[threadIdx.x]);
    if (bad) ctrl->status = CS_ERR_NOT_CORNERSTONE;
}

// ---- pass B: rank and write -------------------------------------------------------------------------
struct LinkOut {
    u64* prefixes; u32* levels; u32* childOffsets; u32* parents; u32* levelRange; u32* leafToNode; u32* nodeToLeaf;
    u32 nodeCapacity;
    // optional, fused H10: with the leaves' particle offsets (prefix sum of N) at hand, every node's
    // particle range is written here too: a leaf's directly, an internal node's from the leaf
    // index where its key range ends (found by a galloping search in K, 1 probe for most nodes).
    const u32* leafOffsets; u32* nodeFirst; u32* nodeCount;
};

// index j1 of the leaf boundary K[j1] == end, given that the node starts at boundary j (j1 >= j + 8)
__device__ __forceinline__ u32 subtreeEnd(const u64* __restrict__ K, u32 j, u32 nl, u64 end)
{
    u32 cur = j + 8;
    if (cur >= nl || K[cur] >= end) return cur < nl ? cur : nl;
    u32 prev, w = 8;
    do {
        prev = cur;
        w <<= 1;
        cur = prev + w < nl ? prev + w : nl;
    } while (K[cur] < end);                      // K[nl] = 8^L >= end: terminates
    u32 lo = prev + 1, hi = cur;                 // K[prev] < end <= K[cur]
    while (lo < hi) {
        const u32 mid = lo + ((hi - lo) >> 1);
        if (K[mid] < end) lo = mid + 1;
        else hi = mid;
    }
    return lo;
}

__global__ void __launch_bounds__(kLinkBlock)
    linkEmitKernel(DeviceCtrl* ctrl, const u64* __restrict__ K, const u32* dNumLeaves, u32 hNumLeaves, LinkOut out,
                   u64* lookback, u32 epoch)
{
    __shared__ u32 sLO[kLevels + 2];                  // level offsets
    __shared__ u32 sWarp[kLinkWarps][kLinkBins];      // per-warp counts -> running exclusive prefix
    __shared__ u32 sBase[kLinkBins];                  // tile's exclusive prefix per bin
    __shared__ u32 sTile, sStop;
    const u32 tid = threadIdx.x, lane = laneId(), warp = tid >> 5;
    const u32 nl = numLeavesOf(dNumLeaves, hNumLeaves);
    if (tid == 0) {
        u32 run = 0;
        bool closed = ctrl->levelTotals[0] == 1;
        for (int l = 0; l < kLevels; ++l) {
            sLO[l] = run;
            run += ctrl->levelTotals[l];
            // every internal node has exactly 8 children
            const u32 next = l + 1 < kLevels ? ctrl->levelTotals[l + 1] : 0u;
            if (next != 8u * ctrl->levelTotals[kLevels + l]) closed = false;
        }
        sLO[kLevels] = run;
        const u32 st = ctrl->status;
        u32 stop = (st == CS_ERR_CAPACITY || st == CS_ERR_NOT_CORNERSTONE) ? 1u : 0u;
        if (!stop && !closed) { ctrl->status = CS_ERR_NOT_CORNERSTONE; stop = 1; }
        if (!stop && run > out.nodeCapacity) { ctrl->status = CS_ERR_CAPACITY; stop = 1; }
        sStop = stop;
        if (!stop && blockIdx.x == 0) {
            ctrl->numNodes = run;
            for (int l = 0; l <= kLevels; ++l) {
                ctrl->levelRange[l] = sLO[l];
                out.levelRange[l] = sLO[l];
            }
            if (out.parents) out.parents[0] = 0;           // A20
        }
    }
    __syncthreads();
    if (sStop) return;
    const u32 tiles = (nl + kLinkTile - 1) / kLinkTile;
    const u32 lt = laneMaskLt();
    for (;;) {
        __syncthreads();
        if (tid == 0) sTile = atomicAdd(&ctrl->linkTicket, 1u);
        for (int i = tid; i < kLinkWarps * kLinkBins; i += kLinkBlock) (&sWarp[0][0])[i] = 0;
        __syncthreads();
        const u32 tile = sTile;
        if (tile >= tiles) break;
        const u32 warpBase = tile * kLinkTile + warp * (32 * kLinkItems) + lane;

        // boundary levels of this thread's items (warp-striped: item order == boundary order)
        int lo[kLinkItems], hi[kLinkItems];
        u64 Kj[kLinkItems];
        int wlo = kLevels, whi = -1;
#pragma unroll
        for (int k = 0; k < kLinkItems; ++k) {
            const u32 j = warpBase + k * 32;
            lo[k] = 1; hi[k] = 0; Kj[k] = 0;
            if (j < nl) {
                Kj[k] = K[j];
                boundaryLevels(Kj[k], K[j + 1], j, lo[k], hi[k]);   // validated in pass A
                wlo = min(wlo, lo[k]);
                whi = max(whi, hi[k]);
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            wlo = min(wlo, __shfl_xor_sync(kFull, wlo, o));
            whi = max(whi, __shfl_xor_sync(kFull, whi, o));
        }
        // phase 1: per-warp counts per level
        u32* wc = sWarp[warp];
        for (int l = wlo; l <= whi; ++l) {
            u32 cAll = 0, cInt = 0;
#pragma unroll
            for (int k = 0; k < kLinkItems; ++k) {
                cAll += __popc(__ballot_sync(kFull, lo[k] <= l && l <= hi[k]));
                cInt += __popc(__ballot_sync(kFull, lo[k] <= l && l < hi[k]));
            }
            if (lane == 0) { wc[l] = cAll; wc[kLevels + l] = cInt; }
        }
        __syncthreads();
        // exclusive prefix over warps, tile totals, look-back (one thread per bin)
        if (tid < kLinkBins) {
            u32 run = 0;
#pragma unroll
            for (int w = 0; w < kLinkWarps; ++w) {
                const u32 c = sWarp[w][tid];
                sWarp[w][tid] = run;
                run += c;
            }
            u64* st = lookback + (size_t)tile * kLinkBins + tid;
            u32 excl = 0;
            if (tile == 0) lbStore(st, lbPack(epoch, kLbPrefix, run));
            else {
                lbStore(st, lbPack(epoch, kLbAggregate, run));
                excl = lbLookBack(lookback, kLinkBins, tid, tile, epoch);
                lbStore(st, lbPack(epoch, kLbPrefix, excl + run));
            }
            sBase[tid] = excl;
        }
        __syncthreads();
        // phase 2: positions and output
        for (int l = wlo; l <= whi; ++l) {
            u32 runAll = sBase[l] + wc[l];
            u32 runInt = sBase[kLevels + l] + wc[kLevels + l];
            const u32 levelStart = sLO[l];
            const u32 childStart = sLO[l + 1];
#pragma unroll
            for (int k = 0; k < kLinkItems; ++k) {
                const bool isNode = lo[k] <= l && l <= hi[k];
                const bool isInt = isNode && l < hi[k];
                const u32 bAll = __ballot_sync(kFull, isNode);
                const u32 bInt = __ballot_sync(kFull, isInt);
                if (isNode) {
                    const u32 j = warpBase + k * 32;
                    const u32 idx = levelStart + runAll + __popc(bAll & lt);
                    // placeholder-bit key: a 1 followed by l octal digits
                    out.prefixes[idx] = l == 0 ? 1ull : ((1ull << (3 * l)) | (Kj[k] >> (3 * (kL - l))));
                    if (out.levels) out.levels[idx] = (u32)l;
                    if (out.nodeFirst) {
                        const u32 firstP = out.leafOffsets[j];
                        u32 jEnd = j + 1;
                        if (isInt) jEnd = l == 0 ? nl : subtreeEnd(K, j, nl, Kj[k] + (1ull << (3 * (kL - l))));
                        out.nodeFirst[idx] = firstP;
                        out.nodeCount[idx] = out.leafOffsets[jEnd] - firstP;
                    }
                    if (isInt) {
                        const u32 co = childStart + 8u * (runInt + __popc(bInt & lt));
                        out.childOffsets[idx] = co;
                        if (out.nodeToLeaf) out.nodeToLeaf[idx] = CS_NO_LEAF;
                        if (out.parents) {
                            uint4 p4 = make_uint4(idx, idx, idx, idx);
                            uint4* dst = reinterpret_cast<uint4*>(out.parents + co);   // co = 1 + 8k: not 16B aligned
                            if ((((uintptr_t)dst) & 15u) == 0) { dst[0] = p4; dst[1] = p4; }
                            else {
#pragma unroll
                                for (int c = 0; c < 8; ++c) out.parents[co + c] = idx;
                            }
                        }
                    } else {
                        out.childOffsets[idx] = 0;               // leaf
                        if (out.nodeToLeaf) out.nodeToLeaf[idx] = j;
                        if (out.leafToNode) out.leafToNode[j] = idx;
                    }
                }
                runAll += __popc(bAll);
                runInt += __popc(bInt);
            }
        }
    }
}

cs_status enqueueLink(cs_context* ctx, const u64* leaves, const u32* dNumLeaves, u32 hNumLeaves, u32 leafBound,
                      u64* prefixes, u32* levels, u32* childOffsets, u32* parents, u32* levelRange, u32* leafToNode,
                      u32* nodeToLeaf, u32 nodeCapacity, const u32* leafOffsets, u32* nodeFirst, u32* nodeCount,
                      cudaStream_t s)
{
    StageTimer t(ctx, CS_STAGE_LINK, s);
    DeviceCtrl* ctrl = ctx->ctrl;
    // reset the link part of the control block (levelTotals, ticket)
    CS_CUDA(ctx, cudaMemsetAsync(&ctrl->linkTicket, 0, sizeof(u32), s));
    CS_CUDA(ctx, cudaMemsetAsync(ctrl->levelTotals, 0, sizeof(u32) * kLinkBins, s));
    const u32 persistentGrid = (u32)ctx->numSMs * 8;
    u32 gridA = divUp((u64)leafBound, kLinkBlock);
    if (gridA > persistentGrid) gridA = persistentGrid;
    if (gridA == 0) gridA = 1;
    linkCountKernel<<<gridA, kLinkBlock, 0, s>>>(ctrl, leaves, dNumLeaves, hNumLeaves);
    CS_LAUNCH_CHECK(ctx, "linkCountKernel");
    u32 gridB = divUp((u64)leafBound, kLinkTile);
    if (gridB > persistentGrid) gridB = persistentGrid;
    if (gridB == 0) gridB = 1;
    const u32 epoch = nextEpoch(ctx, s);
    LinkOut out{prefixes, levels, childOffsets, parents, levelRange, leafToNode, nodeToLeaf, nodeCapacity,
                leafOffsets, leafOffsets ? nodeFirst : nullptr, nodeCount};
    linkEmitKernel<<<gridB, kLinkBlock, 0, s>>>(ctrl, leaves, dNumLeaves, hNumLeaves, out, ctx->tileLookback, epoch);
    CS_LAUNCH_CHECK(ctx, "linkEmitKernel");
    return CS_OK;
}

// ---- H10: node counts ------------------------------------------------------------------------------
// nodeFirst = lower_bound(P, start), nodeCount = lower_bound(P, end) - nodeFirst.
// Leaf nodes take both from the prefix sum of the leaf counts when it is supplied (PAPER.md:258:
// leaves from the particles, which f already counted); internal nodes search P.
__global__ void __launch_bounds__(256)
    nodeCountsKernel(const DeviceCtrl* ctrl, const u64* __restrict__ P, u32 n, const u64* __restrict__ prefixes,
                     const u32* dNumNodes, u32 hNumNodes, const u32* __restrict__ leafOffsets,
                     const u32* __restrict__ nodeToLeaf, u32* __restrict__ nodeFirst, u32* __restrict__ nodeCount)
{
    if (dNumNodes && (ctrl->status == CS_ERR_CAPACITY || ctrl->status == CS_ERR_NOT_CORNERSTONE)) return;
    const u32 numNodes = dNumNodes ? *dNumNodes : hNumNodes;
    const u32 stride = gridDim.x * blockDim.x;
    for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i < numNodes; i += stride) {
        u32 first, last;
        const u32 lf = leafOffsets ? nodeToLeaf[i] : CS_NO_LEAF;
        if (lf != CS_NO_LEAF) {
            first = leafOffsets[lf];
            last = leafOffsets[lf + 1];
        } else {
            const u64 pre = prefixes[i];
            const int l = (63 - __clzll((long long)pre)) / 3;
            const int sh = 3 * (kL - l);
            const u64 start = (pre ^ (1ull << (3 * l))) << sh;
            first = lowerBound(P, 0, n, start);
            last = l == 0 ? n : lowerBound(P, first, n, start + (1ull << sh));
        }
        nodeFirst[i] = first;
        nodeCount[i] = last - first;
    }
}

cs_status enqueueNodeCounts(cs_context* ctx, const u64* P, u64 n, const u64* prefixes, const u32* dNumNodes,
                            u32 hNumNodes, u32 nodeBound, const u32* leafOffsets, const u32* nodeToLeaf,
                            u32* nodeFirst, u32* nodeCount, cudaStream_t s)
{
    StageTimer t(ctx, CS_STAGE_COUNTS, s);
    u32 grid = divUp((u64)nodeBound, 256);
    const u32 persistentGrid = (u32)ctx->numSMs * 8;
    if (grid > persistentGrid) grid = persistentGrid;
    if (grid == 0) grid = 1;
    nodeCountsKernel<<<grid, 256, 0, s>>>(ctx->ctrl, P, (u32)n, prefixes, dNumNodes, hNumNodes, leafOffsets,
                                          nodeToLeaf, nodeFirst, nodeCount);
    CS_LAUNCH_CHECK(ctx, "nodeCountsKernel");
    return CS_OK;
}

}  // namespace cs
