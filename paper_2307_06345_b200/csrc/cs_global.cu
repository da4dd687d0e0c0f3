// The distributed build of Sec. 6 (Eq. 11), as the calls one rank makes:
//   f alone     cs_countLeaves      N_i of this rank's sorted keys for a given K (Eq. 3)
//   -- the caller sums the count arrays of all ranks element by element (f_r: "a single call to MPI_Allreduce") --
//   g alone     cs_rebalance        g3 o g2 o g1 (Eqs. 4-9) on K and the summed counts: identical on every rank
//   partition   cs_partitionLeaves  n_ranks bins of consecutive leaves with about N_tot / n_ranks particles each
//   node counts cs_nodeCountsFromLeaves  per-node sums of the (global) leaf counts, the upward pass of PAPER.md:258
// f is the merge pass of the incremental start (cs_leaves.cu: K and P are both sorted); g is written as the paper
// states it, one kernel per operator with the device-wide scan between them.
#include "cs_device.cuh"

namespace cs {

cs_status enqueueLocateLeaves(cs_context*, const u64* P, u64 n, const u64* K, u32 nl, cudaStream_t);   // cs_leaves.cu

// ---- f: counts from the located boundaries -----------------------------------------------------------------
__global__ void __launch_bounds__(256) leafCountDiffKernel(const u32* __restrict__ off, u32 nl, u32* __restrict__ counts)
{
    const u32 stride = gridDim.x * blockDim.x;
    for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i < nl; i += stride) counts[i] = off[i + 1] - off[i];
}

cs_status enqueueCountLeaves(cs_context* ctx, const u64* P, u64 n, const u64* K, u32 nl, u32* counts, cudaStream_t s)
{
    CS_CUDA(ctx, cudaMemsetAsync(ctx->ctrl, 0, sizeof(DeviceCtrl), s));
    CS_TRY(enqueueLocateLeaves(ctx, P, n, K, nl, s));
    u32 grid = divUp(nl, 256);
    const u32 persistentGrid = (u32)ctx->numSMs * 8;
    if (grid > persistentGrid) grid = persistentGrid;
    leafCountDiffKernel<<<grid, 256, 0, s>>>(ctx->leafOff[0], nl, counts);
    CS_LAUNCH_CHECK(ctx, "leafCountDiffKernel");
    return CS_OK;
}

// ---- g1 (Eq. 5): O_i in {8, 0, 1} from K and the counts N -----------------------------------------------------
// Also the Eq. 2 check of K: g is only defined on a cornerstone array.
__global__ void __launch_bounds__(256) rebalanceDecideKernel(DeviceCtrl* ctrl, const u64* __restrict__ K,
                                                             const u32* __restrict__ N, u32 nl, u32 bucket, u64 minDelta,
                                                             u32* __restrict__ O)
{
    const u32 stride = gridDim.x * blockDim.x;
    bool bad = false, changed = false;
    for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i < nl; i += stride) {
        const u64 Ki = K[i], Kn = K[i + 1];
        const u64 delta = Kn - Ki;
        if (Kn <= Ki || !isPowerOf8(delta) || (Ki & (delta - 1)) || (i == 0 && Ki != 0) || (i == nl - 1 && Kn != kKeyEnd)) {
            bad = true;
            O[i] = 1;
            continue;
        }
        u32 o = 1;
        if (N[i] > bucket && delta > minDelta) o = 8;                   // split (A7: not at depth L)
        else if (delta != kKeyEnd) {                                    // the root never merges (A9)
            const u32 j = (u32)(Ki >> (__ffsll((long long)delta) - 1)) & 7u;   // octant among the siblings
            if (j != 0 && i >= j && i - j + 8 <= nl) {
                const u32 a = i - j;
                if (K[a + 8] - K[a] == (delta << 3)) {                  // all 8 siblings are leaves of this level
                    u64 sum = 0;
#pragma unroll
                    for (u32 c = 0; c < 8; ++c) sum += N[a + c];
                    if (sum <= bucket) o = 0;                           // merged away (A8: <=)
                }
            }
        }
        if (o != 1) changed = true;
        O[i] = o;
    }
    if (bad) ctrl->status = CS_ERR_NOT_CORNERSTONE;
    if (changed) ctrl->changed[0] = 1;
}

// ---- g3 (Eqs. 7-9, A10, A11): K'[O'_i] = K_i / K'[O'_i + c] = K_i + c delta_i / 8 ---------------------------------
__global__ void __launch_bounds__(256) rebalanceScatterKernel(DeviceCtrl* ctrl, const u64* __restrict__ K,
                                                              const u32* __restrict__ O, const u32* __restrict__ Oprime,
                                                              u32 nl, u64* __restrict__ Kout, u32 cap)
{
    const u32 newTotal = Oprime[nl];
    const u32 st = ctrl->status;
    if (st == CS_ERR_NOT_CORNERSTONE) return;
    const u32 gid = blockIdx.x * blockDim.x + threadIdx.x;
    if (newTotal > cap) {
        if (gid == 0) ctrl->status = CS_ERR_CAPACITY;
        return;
    }
    const u32 stride = gridDim.x * blockDim.x;
    for (u32 i = gid; i < nl; i += stride) {
        const u32 o = O[i];
        if (o == 0) continue;
        const u32 p = Oprime[i];
        const u64 Ki = K[i];
        if (o == 1) Kout[p] = Ki;
        else {
            const u64 step = (K[i + 1] - Ki) >> 3;
#pragma unroll
            for (u32 c = 0; c < 8; ++c) Kout[p + c] = Ki + c * step;
        }
    }
    if (gid == 0) {
        Kout[newTotal] = kKeyEnd;
        ctrl->numLeaves = newTotal;
        ctrl->converged = ctrl->changed[0] ? 0u : 1u;
    }
}

cs_status enqueueRebalance(cs_context* ctx, const u64* K, const u32* N, u32 nl, u32 bucket, u32 maxLevel, u64* Kout, u32 cap,
                           cudaStream_t s)
{
    DeviceCtrl* ctrl = ctx->ctrl;
    CS_CUDA(ctx, cudaMemsetAsync(ctrl, 0, sizeof(DeviceCtrl), s));
    u32* O = ctx->leafOff[1];
    u32* Oprime = ctx->leafOffFinal;
    u32 grid = divUp(nl, 256);
    const u32 persistentGrid = (u32)ctx->numSMs * 8;
    if (grid > persistentGrid) grid = persistentGrid;
    rebalanceDecideKernel<<<grid, 256, 0, s>>>(ctrl, K, N, nl, bucket, 1ull << (3 * (kL - (int)maxLevel)), O);
    CS_LAUNCH_CHECK(ctx, "rebalanceDecideKernel");
    CS_TRY(enqueueExclusiveScan(ctx, O, Oprime, nl, s));               // g2 (Eq. 6)
    rebalanceScatterKernel<<<grid, 256, 0, s>>>(ctrl, K, O, Oprime, nl, Kout, cap);
    CS_LAUNCH_CHECK(ctx, "rebalanceScatterKernel");
    return CS_OK;
}

// ---- SFC domain decomposition (A29) ----------------------------------------------------
// C_i = N_0 + ... + N_{i-1}.  bounds[0] = 0, bounds[R] = nl, and for 0 < r < R bounds[r] is the first boundary i with
// C_i * R >= r * N_tot (compared exactly in 128 bits).  Two kernels: 64-bit sums of tiles of kPartTile counts, then one
// CTA that scans the tile sums and lets one warp per boundary find the tile and walk its counts.
constexpr int kPartTile = 2048;

__global__ void __launch_bounds__(256) partTileSumKernel(const u32* __restrict__ N, u32 nl, u64* __restrict__ tileSums)
{
    __shared__ u64 red[8];
    const u32 t0 = blockIdx.x * kPartTile;
    u64 s = 0;
    for (u32 q = threadIdx.x; q < (u32)kPartTile; q += 256) {
        const u32 i = t0 + q;
        if (i < nl) s += N[i];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(kFull, s, o);
    if ((threadIdx.x & 31u) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        u64 v = 0;
        for (int w = 0; w < 8; ++w) v += red[w];
        tileSums[blockIdx.x] = v;
    }
}

__device__ __forceinline__ bool reached(u64 C, u32 R, u32 r, u64 total)   // C * R >= r * total
{
    const u64 ah = __umul64hi(C, (u64)R), al = C * (u64)R;
    const u64 bh = __umul64hi(total, (u64)r), bl = total * (u64)r;
    return ah > bh || (ah == bh && al >= bl);
}

__global__ void __launch_bounds__(1024) partBoundsKernel(const u32* __restrict__ N, u32 nl, u64* tileSums, u32 tiles, u32 R,
                                                         u32* __restrict__ bounds)
{
    __shared__ u64 sCarry;
    __shared__ u64 warpTot[32];
    const u32 tid = threadIdx.x, lane = laneId(), warp = tid >> 5;
    if (tid == 0) sCarry = 0;
    __syncthreads();
    // exclusive scan of the tile sums, in place, 1024 at a time
    for (u32 b = 0; b < tiles; b += 1024) {
        const u32 t = b + tid;
        const u64 v = t < tiles ? tileSums[t] : 0;
        u64 inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const u64 u = __shfl_up_sync(kFull, inc, o);
            if (lane >= (u32)o) inc += u;
        }
        if (lane == 31) warpTot[warp] = inc;
        __syncthreads();
        u64 before = sCarry;
        for (u32 w = 0; w < warp; ++w) before += warpTot[w];
        if (t < tiles) tileSums[t] = before + inc - v;
        __syncthreads();
        if (tid == 1023) sCarry = before + inc;
        __syncthreads();
    }
    const u64 total = sCarry;
    if (tid == 0) {
        bounds[0] = 0;
        bounds[R] = nl;
    }
    // one warp per boundary r
    for (u32 r = 1 + warp; r < R; r += 32) {
        u32 result = 0;
        if (total != 0) {
            // last tile t with prefix[t] * R < r * total (prefix[0] = 0 qualifies)
            u32 lo = 0, hi = tiles;                                  // invariant: tile lo qualifies, tile hi does not
            while (hi - lo > 1) {
                const u32 mid = (lo + hi) >> 1;
                if (!reached(tileSums[mid], R, r, total)) lo = mid;
                else hi = mid;
            }
            u64 C = tileSums[lo];
            const u32 t0 = lo * kPartTile;
            result = nl;
            for (u32 q = 0; q < (u32)kPartTile; q += 32) {           // first i > t0 with C_i * R >= r * total
                const u32 i = t0 + q + lane;
                const u64 v = i < nl ? N[i] : 0;
                u64 inc = v;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const u64 u = __shfl_up_sync(kFull, inc, o);
                    if (lane >= (u32)o) inc += u;
                }
                const u32 m = __ballot_sync(kFull, reached(C + inc, R, r, total));   // C_{i+1}
                if (m) {
                    const u32 first = (u32)__ffs((int)m) - 1u;
                    result = t0 + q + first + 1u;
                    break;
                }
                C += __shfl_sync(kFull, inc, 31);
            }
            if (result > nl) result = nl;
        }
        if (lane == 0) bounds[r] = result;
    }
}

cs_status enqueuePartition(cs_context* ctx, const u32* N, u32 nl, u32 R, u32* bounds, cudaStream_t s)
{
    u64* tileSums = ctx->tileLookback;                                // [leafTiles] u64, tiles of >= 1024 leaves
    const u32 tiles = divUp(nl, kPartTile);
    partTileSumKernel<<<tiles, 256, 0, s>>>(N, nl, tileSums);
    CS_LAUNCH_CHECK(ctx, "partTileSumKernel");
    partBoundsKernel<<<1, 1024, 0, s>>>(N, nl, tileSums, tiles, R, bounds);
    CS_LAUNCH_CHECK(ctx, "partBoundsKernel");
    // the look-back words of later scans carry a fresh epoch, but these sums could alias one: clear them
    CS_CUDA(ctx, cudaMemsetAsync(tileSums, 0, (size_t)tiles * sizeof(u64), s));
    return CS_OK;
}

// ---- node counts from leaf counts (leaves first, internal nodes from their children) ------------------
// With off = exclusive prefix sum of the leaf counts, a node whose key range is [start, end) covers the leaves
// [a, b) with K_a = start, K_b = end: nodeFirst = off[a], nodeCount = off[b] - off[a] = the sum over its leaves,
// which is what the upward pass accumulates.
__device__ __forceinline__ u32 lowerBoundK(const u64* __restrict__ K, u32 cnt, u64 key)
{
    u32 lo = 0, hi = cnt;
    while (lo < hi) {
        const u32 mid = lo + ((hi - lo) >> 1);
        if (__ldg(K + mid) < key) lo = mid + 1;
        else hi = mid;
    }
    return lo;
}

__global__ void __launch_bounds__(256)
    nodeCountsFromLeavesKernel(const u64* __restrict__ K, const u32* __restrict__ off, u32 nl, const u64* __restrict__ prefixes,
                               u32 numNodes, u32* __restrict__ nodeFirst, u32* __restrict__ nodeCount)
{
    const u32 stride = gridDim.x * blockDim.x;
    for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i < numNodes; i += stride) {
        const u64 pre = prefixes[i];
        const int l = (63 - __clzll((long long)pre)) / 3;
        const int sh = 3 * (kL - l);
        const u64 start = (pre ^ (1ull << (3 * l))) << sh;
        const u32 a = lowerBoundK(K, nl + 1, start);
        const u32 b = l == 0 ? nl : lowerBoundK(K, nl + 1, start + (1ull << sh));
        const u32 first = off[a];
        nodeFirst[i] = first;
        nodeCount[i] = off[b] - first;
    }
}

cs_status enqueueNodeCountsFromLeaves(cs_context* ctx, const u64* K, const u32* N, u32 nl, const u64* prefixes, u32 numNodes,
                                      u32* nodeFirst, u32* nodeCount, cudaStream_t s)
{
    CS_TRY(enqueueExclusiveScan(ctx, N, ctx->leafOffFinal, nl, s));
    u32 grid = divUp(numNodes, 256);
    const u32 persistentGrid = (u32)ctx->numSMs * 8;
    if (grid > persistentGrid) grid = persistentGrid;
    nodeCountsFromLeavesKernel<<<grid, 256, 0, s>>>(K, ctx->leafOffFinal, nl, prefixes, numNodes, nodeFirst, nodeCount);
    CS_LAUNCH_CHECK(ctx, "nodeCountsFromLeavesKernel");
    return CS_OK;
}

}  // namespace cs
