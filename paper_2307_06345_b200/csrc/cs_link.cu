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
//     of a tile and a prefix sum over tiles.
//   * The children of the k-th internal node of level l (SFC order) are the 8 nodes
//     LO[l+1] + 8k .. + 8k + 7, because level l+1 consists of exactly those sibling groups in
//     the same order.  So CO = LO[l+1] + 8 * (rank among the internal nodes of level l):
//     a second set of 22 counters, no search.
//
// Pass A counts nodes per level and tile and validates Eq. 2; pass A2 turns the counts into
// exclusive prefixes over tiles (-> LO, numNodes); pass C ranks inside the tile and writes.
// No pass waits on another CTA: tiles are assigned statically.
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

// ---- shared by passes A and C: this thread's boundaries and the warp's counts per level -----------
struct TileItems {
    int lo[kLinkItems], hi[kLinkItems];
    u64 Kj[kLinkItems];
    int wlo, whi;             // warp-uniform range of levels present
};

// Loads the kLinkItems boundaries of this thread (warp-striped: item order == boundary order).
// Returns false if some gap violates Eq. 2.
__device__ __forceinline__ bool loadTileItems(const u64* __restrict__ K, u32 nl, u32 warpBase, TileItems& it)
{
    bool ok = true;
    it.wlo = kLevels;
    it.whi = -1;
#pragma unroll
    for (int k = 0; k < kLinkItems; ++k) {
        const u32 j = warpBase + k * 32;
        it.lo[k] = 1; it.hi[k] = 0; it.Kj[k] = 0;                      // empty range for j >= nl
        if (j < nl) {
            it.Kj[k] = K[j];
            const u64 Kn = K[j + 1];
            if (!boundaryLevels(it.Kj[k], Kn, j, it.lo[k], it.hi[k])) { ok = false; it.lo[k] = 1; it.hi[k] = 0; }
            if (j == 0 && it.Kj[k] != 0) ok = false;
            if (j == nl - 1 && Kn != kKeyEnd) ok = false;
            if (it.lo[k] <= it.hi[k]) { it.wlo = min(it.wlo, it.lo[k]); it.whi = max(it.whi, it.hi[k]); }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        it.wlo = min(it.wlo, __shfl_xor_sync(kFull, it.wlo, o));
        it.whi = max(it.whi, __shfl_xor_sync(kFull, it.whi, o));
    }
    return ok;
}

// per-warp node counts per level (all / internal) -> wc[0..kLinkBins), written by lane 0
__device__ __forceinline__ void warpLevelCounts(const TileItems& it, u32* wc, u32 lane)
{
    for (int l = it.wlo; l <= it.whi; ++l) {
        u32 cAll = 0, cInt = 0;
#pragma unroll
        for (int k = 0; k < kLinkItems; ++k) {
            cAll += __popc(__ballot_sync(kFull, it.lo[k] <= l && l <= it.hi[k]));
            cInt += __popc(__ballot_sync(kFull, it.lo[k] <= l && l < it.hi[k]));
        }
        if (lane == 0) { wc[l] = cAll; wc[kLevels + l] = cInt; }
    }
}

// ---- pass A: nodes per level and tile; validates Eq. 2 -------------------------------------------------
__global__ void __launch_bounds__(kLinkBlock)
    linkCountKernel(DeviceCtrl* ctrl, const u64* __restrict__ K, const u32* dNumLeaves, u32 hNumLeaves,
                    u32* __restrict__ tileHist)
{
    chainEnter();
    __shared__ u32 sWarp[kLinkWarps][kLinkBins];
    __shared__ u32 sStop;
    const u32 tid = threadIdx.x, lane = laneId(), warp = tid >> 5;
    if (tid == 0) {                                           // one read per CTA: uniform decision
        const u32 st = *(const volatile u32*)&ctrl->status;
        sStop = (st == CS_ERR_CAPACITY || st == CS_ERR_NOT_CORNERSTONE) ? 1u : 0u;
    }
    __syncthreads();
    if (sStop) return;
    const u32 nl = numLeavesOf(dNumLeaves, hNumLeaves);
    const u32 tiles = (nl + kLinkTile - 1) / kLinkTile;
    bool bad = (nl == 0);
    for (u32 tile = blockIdx.x; tile < tiles; tile += gridDim.x) {
        __syncthreads();
        for (int i = tid; i < kLinkWarps * kLinkBins; i += kLinkBlock) (&sWarp[0][0])[i] = 0;
        __syncthreads();
        TileItems it;
        if (!loadTileItems(K, nl, tile * kLinkTile + warp * (32 * kLinkItems) + lane, it)) bad = true;
        warpLevelCounts(it, sWarp[warp], lane);
        __syncthreads();
        if (tid < kLinkBins) {
            u32 sum = 0;
#pragma unroll
            for (int w = 0; w < kLinkWarps; ++w) sum += sWarp[w][tid];
            tileHist[(size_t)tile * kLinkBins + tid] = sum;
        }
    }
    if (bad) ctrl->status = CS_ERR_NOT_CORNERSTONE;
}

// ---- pass A2: exclusive prefix over tiles of every (level, kind) column; column totals -----------------
constexpr int kColItems = 4;
__global__ void __launch_bounds__(256)
    linkScanKernel(DeviceCtrl* ctrl, const u32* dNumLeaves, u32 hNumLeaves, u32* __restrict__ tileHist)
{
    chainEnter();
    __shared__ u32 warpSums[256 / 32 + 1];
    const u32 st = ctrl->status;
    if (st == CS_ERR_CAPACITY || st == CS_ERR_NOT_CORNERSTONE) return;
    const u32 nl = numLeavesOf(dNumLeaves, hNumLeaves);
    const u32 tiles = (nl + kLinkTile - 1) / kLinkTile;
    const u32 bin = blockIdx.x;
    u32 running = 0;
    for (u32 t0 = 0; t0 < tiles; t0 += 256 * kColItems) {
        u32 v[kColItems], sum = 0;
#pragma unroll
        for (int k = 0; k < kColItems; ++k) {
            const u32 t = t0 + threadIdx.x * kColItems + k;
            v[k] = t < tiles ? tileHist[(size_t)t * kLinkBins + bin] : 0u;
            sum += v[k];
        }
        u32 total;
        u32 run = running + blockExclusiveScan<256>(sum, warpSums, &total);
#pragma unroll
        for (int k = 0; k < kColItems; ++k) {
            const u32 t = t0 + threadIdx.x * kColItems + k;
            if (t < tiles) tileHist[(size_t)t * kLinkBins + bin] = run;
            run += v[k];
        }
        running += total;
        __syncthreads();
    }
    if (threadIdx.x == 0) ctrl->levelTotals[bin] = running;
}

// ---- pass C: rank and write ----------------------------------------------------------------------------
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

#ifndef CS_LINK_PREFETCH
#define CS_LINK_PREFETCH 592                    // 4 CTAs per SM x 148 SMs
#endif
#ifndef CS_LINK_MINBLOCKS
#define CS_LINK_MINBLOCKS 4
#endif
__global__ void __launch_bounds__(kLinkBlock, CS_LINK_MINBLOCKS)
    linkEmitKernel(DeviceCtrl* ctrl, const u64* __restrict__ K, const u32* dNumLeaves, u32 hNumLeaves, LinkOut out,
                   const u32* __restrict__ tilePrefix)
{
    chainEnter();
    __shared__ u32 sLO[kLevels + 2];                  // level offsets
    __shared__ u32 sWarp[kLinkWarps][kLinkBins];      // per-warp counts -> running exclusive prefix
    __shared__ u32 sBase[kLinkBins];                  // tile's exclusive prefix per bin
    __shared__ u32 sStop;
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
    for (u32 tile = blockIdx.x; tile < tiles; tile += gridDim.x) {
        __syncthreads();
#if CS_LINK_PREFETCH
        if (tid == 0 && (u64)(tile + CS_LINK_PREFETCH) * kLinkTile < nl) {   // the tile one generation of CTAs ahead
            const u64 pb = (u64)(tile + CS_LINK_PREFETCH) * kLinkTile;
            const u32 cnt = (u32)((u64)nl - pb < (u64)kLinkTile ? (u64)nl - pb : (u64)kLinkTile);
            bulkPrefetchL2(K + pb, (cnt * 8u) & ~15u);
            if (out.leafOffsets) bulkPrefetchL2(out.leafOffsets + pb, (cnt * 4u) & ~15u);
        }
#endif
        for (int i = tid; i < kLinkWarps * kLinkBins; i += kLinkBlock) (&sWarp[0][0])[i] = 0;
        if (tid < kLinkBins) sBase[tid] = tilePrefix[(size_t)tile * kLinkBins + tid];
        __syncthreads();
        const u32 warpBase = tile * kLinkTile + warp * (32 * kLinkItems) + lane;
        TileItems it;
        loadTileItems(K, nl, warpBase, it);               // validated in pass A
        u32* wc = sWarp[warp];
        warpLevelCounts(it, wc, lane);
        __syncthreads();
        if (tid < kLinkBins) {                            // exclusive prefix over the warps of the tile
            u32 run = 0;
#pragma unroll
            for (int w = 0; w < kLinkWarps; ++w) {
                const u32 c = sWarp[w][tid];
                sWarp[w][tid] = run;
                run += c;
            }
        }
        __syncthreads();
        // positions and output
        for (int l = it.wlo; l <= it.whi; ++l) {
            u32 runAll = sBase[l] + wc[l];
            u32 runInt = sBase[kLevels + l] + wc[kLevels + l];
            const u32 levelStart = sLO[l];
            const u32 childStart = sLO[l + 1];
#pragma unroll
            for (int k = 0; k < kLinkItems; ++k) {
                const bool isNode = it.lo[k] <= l && l <= it.hi[k];
                const bool isInt = isNode && l < it.hi[k];
                const u32 bAll = __ballot_sync(kFull, isNode);
                const u32 bInt = __ballot_sync(kFull, isInt);
                if (isNode) {
                    const u32 j = warpBase + k * 32;
                    const u32 idx = levelStart + runAll + __popc(bAll & lt);
                    // placeholder-bit key: a 1 followed by l octal digits
                    out.prefixes[idx] = l == 0 ? 1ull : ((1ull << (3 * l)) | (it.Kj[k] >> (3 * (kL - l))));
                    if (out.levels) out.levels[idx] = (u32)l;
                    if (out.nodeFirst) {
                        const u32 firstP = out.leafOffsets[j];
                        u32 jEnd = j + 1;
                        if (isInt) jEnd = l == 0 ? nl : subtreeEnd(K, j, nl, it.Kj[k] + (1ull << (3 * (kL - l))));
                        out.nodeFirst[idx] = firstP;
                        out.nodeCount[idx] = out.leafOffsets[jEnd] - firstP;
                    }
                    if (isInt) {
                        const u32 co = childStart + 8u * (runInt + __popc(bInt & lt));
                        out.childOffsets[idx] = co;
                        if (out.nodeToLeaf) out.nodeToLeaf[idx] = CS_NO_LEAF;
                        if (out.parents) {
#pragma unroll
                            for (int c = 0; c < 8; ++c) out.parents[co + c] = idx;
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
    u32* tileHist = ctx->linkTileHist;                              // [tiles][kLinkBins]
    // one tile per CTA where possible: the tiles differ in cost (subtree-end searches), so many small CTAs
    // balance better than few persistent ones
    const u32 gridCap = (u32)ctx->numSMs * 64;
    u32 grid = divUp((u64)leafBound, kLinkTile);
    if (grid > gridCap) grid = gridCap;
    if (grid == 0) grid = 1;
    launchChained(linkCountKernel, dim3(grid), dim3(kLinkBlock), 0, s, ctrl, leaves, dNumLeaves, hNumLeaves, tileHist);
    CS_LAUNCH_CHECK(ctx, "linkCountKernel");
    launchChained(linkScanKernel, dim3(kLinkBins), dim3(256), 0, s, ctrl, dNumLeaves, hNumLeaves, tileHist);
    CS_LAUNCH_CHECK(ctx, "linkScanKernel");
    LinkOut out{prefixes, levels, childOffsets, parents, levelRange, leafToNode, nodeToLeaf, nodeCapacity,
                leafOffsets, leafOffsets ? nodeFirst : nullptr, nodeCount};
    launchChained(linkEmitKernel, dim3(grid), dim3(kLinkBlock), 0, s, ctrl, leaves, dNumLeaves, hNumLeaves, out, tileHist);
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
