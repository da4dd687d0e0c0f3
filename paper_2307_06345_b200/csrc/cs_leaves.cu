// H4-H8: cornerstone leaf array by iterating f and g = g3 o g2 o g1 (Eqs. 2-9).
//
// Two kernel launches per round do f, g1, g2, g3:
//   f   (Eq. 3)  the lower-bound position off_i of every K_i in P is carried with K from round to
//                round; N_i = off_{i+1} - off_i.  Only the 7 new boundaries of a split leaf are
//                searched, inside the parent's particle range [off_i, off_{i+1}) (second kernel).
//   g1  (Eq. 5)  O_i in {8, 0, 1} per leaf (readings A7, A8, A9).
//   g2  (Eq. 6)  exclusive prefix sum of O: in-tile scan + decoupled look-back across tiles.
//   g3  (Eqs. 7-9, A10, A11) scatter of kept keys / 8 child keys to K'.
// All sizes stay in the device control block; round r reads nl[r] and writes nl[r+1].  The rounds of
// one build are ONE cooperative launch (leafRoundsKernel): the grid loops over the rounds with a grid
// barrier between the two halves of a round and stops at the first round that changes nothing
// (ctrl->done), so a converged build pays for the rounds it needs, not for the 22 it may need, and
// there is no host round trip.  An incremental start first locates every K_i of the
// previous array in P by merging the two sorted arrays (leafLocateKernel), not by one full-range
// binary search per leaf.
#include <cooperative_groups.h>

#include "cs_device.cuh"

namespace cg = cooperative_groups;

namespace cs {

__device__ __forceinline__ u32 ldVolatile(const u32* p) { return *(const volatile u32*)p; }

// ---- start arrays -----------------------------------------------------------------------------
__global__ void leavesInitRootKernel(DeviceCtrl* ctrl, u64* K0, u32* off0, u32 n)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        K0[0] = 0;
        K0[1] = kKeyEnd;
        off0[0] = 0;
        off0[1] = n;
        ctrl->nl[0] = 1;
    }
}

// ---- incremental start: f of the previous array by a merge of K and P ---------------------------
// Copy the caller's previous cornerstone array into the workspace, check Eq. 2 and
// locate every K_i in P (Eq. 3 for the whole array: the f of the first incremental round).  K and P are
// both sorted, so this is a merge.  P is cut into tiles of kLocTile keys; tile t owns the entries of K
// whose lower-bound positions fall into it, K_i in (P[tT - 1], P[(t+1)T - 1]], a contiguous slice
// [split[t], split[t+1]) of K.  leafSplitKernel finds the slices (one binary search in K per tile, all
// tiles at once) and does the Eq. 2 check and the copy; leafLocateKernel stages each tile of P in
// shared memory once (coalesced, 8 B per particle: the only pass over P) and places each K_i of its
// slice by a binary search there.
constexpr int kLocBlock = 256;
constexpr int kLocItems = 8;
constexpr int kLocTile = kLocBlock * kLocItems;
static_assert(kLocTile == (1 << kDirectTileLog2), "split[] lives in the per-tile arrays of the one-pass build");

// first index i in [0, cnt) with A[i] > key (cnt if none), by one warp: 32 probes per dependent round trip
__device__ __forceinline__ u32 warpUpperBound32(const u64* __restrict__ A, u32 cnt, u64 key, u32 lane)
{
    u32 lo = 0, hi = cnt;                                          // answer in [lo, hi]
    while (hi - lo > 32) {
        const u32 w = hi - lo;
        const u32 s = (w + 31) / 32;
        const u32 idx = lo + (lane + 1) * s - 1;
        const bool le = idx < hi && __ldg(A + idx) <= key;
        const u32 m = __popc(__ballot_sync(kFull, le));            // probes are monotone: m leading trues
        const u32 newLo = lo + m * s;
        const u32 newHi = lo + (m + 1) * s - 1;
        lo = newLo < hi ? newLo : hi;
        hi = newHi < hi ? newHi : hi;
    }
    const u32 idx = lo + lane;
    const bool le = idx < hi && __ldg(A + idx) <= key;
    return lo + __popc(__ballot_sync(kFull, le));
}

__global__ void __launch_bounds__(256) leafSplitKernel(DeviceCtrl* ctrl, const u64* __restrict__ P, u32 n,
                                                       const u64* __restrict__ prev, u32 nlPrev, u64* K0,
                                                       u32* __restrict__ split)
{
    const u32 stride = gridDim.x * blockDim.x;
    const u32 gid = blockIdx.x * blockDim.x + threadIdx.x;
    const u32 lane = laneId();
    // one warp per tile boundary: first i with K_i > P[t T - 1]
    const u32 tiles = n ? (n + kLocTile - 1) / kLocTile : 1u;
    for (u32 t = gid >> 5; t <= tiles; t += stride >> 5) {
        u32 v = 0;
        if (t == tiles) v = nlPrev + 1;
        else if (t > 0) v = warpUpperBound32(prev, nlPrev + 1, __ldg(P + (size_t)t * kLocTile - 1), lane);
        if (lane == 0) split[t] = v;
    }
    bool bad = false;
    for (u32 i = gid; i <= nlPrev; i += stride) {
        const u64 k = prev[i];
        if (i == 0 && k != 0) bad = true;
        if (i == nlPrev) {
            if (k != kKeyEnd) bad = true;
        } else {
            const u64 kn = prev[i + 1];
            const u64 delta = kn - k;
            if (kn <= k || !isPowerOf8(delta) || (k & (delta - 1))) bad = true;
        }
        K0[i] = k;
    }
    if (bad) {
        ctrl->status = CS_ERR_NOT_CORNERSTONE;
        ctrl->done = 1;
    }
    if (gid == 0) ctrl->nl[0] = nlPrev;
}

__global__ void __launch_bounds__(kLocBlock, 4) leafLocateKernel(const u64* __restrict__ P, u32 n,
                                                                 const u64* __restrict__ prev,
                                                                 const u32* __restrict__ split, u32* __restrict__ off0)
{
    __shared__ u64 sP[kLocTile];
    const u32 tid = threadIdx.x;
    const u32 t0 = blockIdx.x * kLocTile;
    const u32 valid = n - t0 < (u32)kLocTile ? n - t0 : (u32)kLocTile;   // n == 0: one CTA with an empty tile
    const u32 a = split[blockIdx.x], b = split[blockIdx.x + 1];
    if (a == b) return;                                            // no K_i falls into this tile
    {
        u64 kr[kLocItems];
#pragma unroll
        for (int k = 0; k < kLocItems; ++k) {
            const u32 q = k * kLocBlock + tid;
            kr[k] = q < valid ? ldStreamU64(P + t0 + q) : ~0ull;
        }
#pragma unroll
        for (int k = 0; k < kLocItems; ++k) sP[k * kLocBlock + tid] = kr[k];
    }
    __syncthreads();
    for (u32 i = a + tid; i < b; i += kLocBlock) {
        const u64 k = prev[i];
        u32 lo = 0, hi = valid;                                    // first slot of the tile with P >= K_i
        while (lo < hi) {
            const u32 mid = (lo + hi) >> 1;
            if (sP[mid] < k) lo = mid + 1;
            else hi = mid;
        }
        off0[i] = t0 + lo;
    }
}

constexpr u32 kLinearMax = 1024;   // split leaves with at most this many particles: one warp reads their keys (leafSearchBody)

// ---- one round, first half: g1, g2, g3 and the task list for f ----------------------------------------
// Two phases with a grid barrier between them (all CTAs of the cooperative launch are resident):
//   decide   every tile of 2048 leaves is staged in shared memory by coalesced loads; g1 (Eq. 5) gives O_i
//            from N_i = off_{i+1} - off_i; the tile publishes sum(O) and its numbers of split leaves, every
//            thread keeps the O of its 8 leaves as 8 nibbles in a scratch word.  If no tile changed
//            anything the round is the confirming one: K' = K, nothing is written.
//   scatter  g2 (Eq. 6): position of a tile in K' = sum of the totals of the tiles before it (a plain
//            block reduction over the published totals: with the whole array in flight at once a
//            look-back chain would be as long as the array), in-tile scan; g3 (Eqs. 7-9): kept keys and
//            the 8 child keys of split leaves go to K'.  Each split leaf becomes a search task (slot of its
//            first child in K', end of its particle range): the 7 inner child boundaries are located in P
//            by leafSearchBody, spread over the whole GPU, instead of serially by the thread that owns the leaf.
struct TileInfo {
    u32 total, nLin, nSearch, pad;
};

__device__ __forceinline__ u32 leafSlot(u32 q) { return q + (q >> 3); }   // slot of tile entry q: runs of 8 in different banks

struct LeafTileSmem {
    u64 K[kLeafTile + kLeafTile / 8 + 2];
    u32 off[kLeafTile + kLeafTile / 8 + 2];
    u32 warpSums[kLeafBlock / 32 + 1];
    u32 red[3][kLeafBlock / 32];
    u32 base[3];
};

// entries tile0 .. tile0 + kLeafTile (inclusive: the entry after the tile's last leaf) of K and off
__device__ __forceinline__ void leafStageTile(LeafTileSmem& sm, const u64* Kin, const u32* offIn, u32 tile0, u32 nl, u32 n)
{
    for (u32 q = threadIdx.x; q <= (u32)kLeafTile; q += kLeafBlock) {
        const u32 i = tile0 + q;
        sm.K[leafSlot(q)] = i <= nl ? __ldcg(Kin + i) : kKeyEnd;      // .cg: written by other CTAs earlier in this launch
        sm.off[leafSlot(q)] = i <= nl ? __ldcg(offIn + i) : n;
    }
    __syncthreads();
}

// returns true (in every thread of every CTA) ... after the grid barrier that follows: see leafRoundsKernel
__device__ __forceinline__ void
    leafDecideBody(LeafTileSmem& sm, DeviceCtrl* ctrl, u32 n, u32 nl, const u64* Kin, const u32* offIn, u32* opk,
                   TileInfo* info, u32 r, u32 bucket, u64 minDelta, bool emit, u64* __restrict__ leaves, u32* __restrict__ counts,
                   u32* __restrict__ offFinal)
{
    const u32 tiles = (nl + kLeafTile - 1) / kLeafTile;
    const u32 tid = threadIdx.x;
    for (u32 tile = blockIdx.x; tile < tiles; tile += gridDim.x) {
        const u32 tile0 = tile * kLeafTile;
        leafStageTile(sm, Kin, offIn, tile0, nl, n);
        if (emit) {                                              // this round's input, in the caller's format (coalesced)
            for (u32 q = tid; q <= (u32)kLeafTile; q += kLeafBlock) {
                const u32 i = tile0 + q;
                if (i > nl || (q == (u32)kLeafTile && i != nl)) continue;   // entry kLeafTile belongs to the next tile
                const u32 o = sm.off[leafSlot(q)];
                leaves[i] = sm.K[leafSlot(q)];
                offFinal[i] = o;
                if (i < nl && counts) counts[i] = sm.off[leafSlot(q + 1)] - o;
            }
        }
        const u32 q0 = tid * kLeafItems;
        const u32 first = tile0 + q0;
        u32 Opk = 0;                                             // O of the thread's 8 leaves, 4 bits each
        u32 sum = 0, nLin = 0, nSearch = 0;
        u64 Kk = sm.K[leafSlot(q0)];
        u32 offk = sm.off[leafSlot(q0)];
#pragma unroll
        for (int k = 0; k < kLeafItems; ++k) {
            const u32 i = first + k;
            const u64 Kn = sm.K[leafSlot(q0 + k + 1)];
            const u32 offn = sm.off[leafSlot(q0 + k + 1)];
            u32 o = 0;
            if (i < nl) {
                const u64 delta = Kn - Kk;
                const u32 cnt = offn - offk;                              // f: N_i
                o = 1;
                if (cnt > bucket && delta > minDelta) o = 8;             // split (A7: not at depth L)
                else if (delta != kKeyEnd) {                             // the root never merges (A9)
                    const u32 j = (u32)(Kk >> (__ffsll((long long)delta) - 1)) & 7u;   // octant among siblings (delta = 8^m)
                    if (j != 0 && i >= j && i - j + 8 <= nl) {
                        const u32 a = i - j;
                        u64 Ka, Ka8;
                        u32 offa, offa8;
                        if (a >= tile0 && a + 8 <= tile0 + (u32)kLeafTile) {   // the siblings lie in the staged tile
                            Ka = sm.K[leafSlot(a - tile0)]; Ka8 = sm.K[leafSlot(a - tile0 + 8)];
                            offa = sm.off[leafSlot(a - tile0)]; offa8 = sm.off[leafSlot(a - tile0 + 8)];
                        } else {
                            Ka = __ldcg(Kin + a); Ka8 = __ldcg(Kin + a + 8);
                            offa = __ldcg(offIn + a); offa8 = __ldcg(offIn + a + 8);
                        }
                        if (Ka8 - Ka == (delta << 3) && offa8 - offa <= bucket) o = 0;   // all 8 siblings are leaves and
                    }                                                                    // fit into one: merged away (A8)
                }
                // split leaves become search tasks: short particle ranges are counted linearly, long ones searched
                if (o == 8) {
                    if (cnt <= kLinearMax) ++nLin;
                    else ++nSearch;
                }
            }
            Opk |= o << (4 * k);
            sum += o;
            Kk = Kn;
            offk = offn;
        }
        opk[(size_t)tile * kLeafBlock + tid] = Opk;
        // tile totals
        sum = warpReduceSum(sum); nLin = warpReduceSum(nLin); nSearch = warpReduceSum(nSearch);
        if ((tid & 31u) == 0) { sm.red[0][tid >> 5] = sum; sm.red[1][tid >> 5] = nLin; sm.red[2][tid >> 5] = nSearch; }
        __syncthreads();
        if (tid == 0) {
            TileInfo ti{0, 0, 0, 0};
            for (int w = 0; w < kLeafBlock / 32; ++w) { ti.total += sm.red[0][w]; ti.nLin += sm.red[1][w]; ti.nSearch += sm.red[2][w]; }
            info[tile] = ti;
            const u32 leavesInTile = nl - tile0 < (u32)kLeafTile ? nl - tile0 : (u32)kLeafTile;
            if (ti.total != leavesInTile || ti.nLin || ti.nSearch) atomicOr(&ctrl->changed[r], 1u);   // some O_i != 1
        }
        __syncthreads();                                     // the staged tile and sm.red are free again
    }
}

__device__ __forceinline__ void
    leafScatterBody(LeafTileSmem& sm, DeviceCtrl* ctrl, u32 n, u32 nl, const u64* Kin, const u32* offIn, u64* Kout,
                    u32* offOut, const u32* opk, const TileInfo* info, uint4* tasksLin, uint4* tasksSearch, u32 maxTasks,
                    u32 r, u32 cap, u32 lastRound)
{
    const u32 tiles = (nl + kLeafTile - 1) / kLeafTile;
    const u32 tid = threadIdx.x;
    u32 known = 0;                                               // sm.base = sums over the tiles [0, known)
    if (tid < 3) sm.base[tid] = 0;
    for (u32 tile = blockIdx.x; tile < tiles; tile += gridDim.x) {
        // g2 across tiles: add the totals of the tiles [known, tile)
        {
            u32 a0 = 0, a1 = 0, a2 = 0;
            for (u32 u = known + tid; u < tile; u += kLeafBlock) {
                const uint4 v = __ldcg(reinterpret_cast<const uint4*>(info + u));
                a0 += v.x; a1 += v.y; a2 += v.z;
            }
            a0 = warpReduceSum(a0); a1 = warpReduceSum(a1); a2 = warpReduceSum(a2);
            if ((tid & 31u) == 0) { sm.red[0][tid >> 5] = a0; sm.red[1][tid >> 5] = a1; sm.red[2][tid >> 5] = a2; }
        }
        const u32 tile0 = tile * kLeafTile;
        leafStageTile(sm, Kin, offIn, tile0, nl, n);             // ends with a barrier
        if (tid < 3) {
            u32 v = sm.base[tid];
            for (int w = 0; w < kLeafBlock / 32; ++w) v += sm.red[tid][w];
            sm.base[tid] = v;
        }
        known = tile;
        const u32 Opk = __ldcg(opk + (size_t)tile * kLeafBlock + tid);
        u32 sum = 0, splits = 0;
        const u32 q0 = tid * kLeafItems;
#pragma unroll
        for (int k = 0; k < kLeafItems; ++k) {
            const u32 o = (Opk >> (4 * k)) & 15u;
            sum += o;
            if (o == 8) splits += (sm.off[leafSlot(q0 + k + 1)] - sm.off[leafSlot(q0 + k)] <= kLinearMax) ? 1u : (1u << 16);
        }
        u32 total, totalSplits;
        const u32 excl = blockExclusiveScan<kLeafBlock>(sum, sm.warpSums, &total);          // 2 barriers: sm.base is set
        const u32 taskSlot = blockExclusiveScan<kLeafBlock>(splits, sm.warpSums, &totalSplits);
        // g3: node rebalancing (Eqs. 8, 9)
        const u32 tileBase = sm.base[0];
        u32 p = tileBase + excl;
        u32 linSlot = sm.base[1] + (taskSlot & 0xFFFFu), searchSlot = sm.base[2] + (taskSlot >> 16);
#pragma unroll
        for (int k = 0; k < kLeafItems; ++k) {
            const u32 o = (Opk >> (4 * k)) & 15u;
            if (o == 1) {
                if (p < cap) {
                    Kout[p] = sm.K[leafSlot(q0 + k)];
                    offOut[p] = sm.off[leafSlot(q0 + k)];
                }
                p += 1;
            } else if (o == 8) {
                const u64 K0 = sm.K[leafSlot(q0 + k)];
                const u64 step = (sm.K[leafSlot(q0 + k + 1)] - K0) >> 3;
                const u32 lo = sm.off[leafSlot(q0 + k)], hi = sm.off[leafSlot(q0 + k + 1)];
                if (p + 8 <= cap) {
#pragma unroll
                    for (u32 c = 0; c < 8; ++c) Kout[p + c] = K0 + c * step;
                    offOut[p] = lo;
                }
                const bool lin = hi - lo <= kLinearMax;
                u32& tslot = lin ? linSlot : searchSlot;
                if (p + 8 <= cap && tslot < maxTasks)             // first child slot, particle range, shift of the child digit
                    (lin ? tasksLin : tasksSearch)[tslot] = make_uint4(p, lo, hi, (u32)__ffsll((long long)step) - 1u);
                ++tslot;
                p += 8;
            }
        }
        if (tile == tiles - 1 && tid == 0) {                 // the last tile closes the round
            const u32 newTotal = tileBase + total;
            const u32 linTotal = sm.base[1] + (totalSplits & 0xFFFFu), searchTotal = sm.base[2] + (totalSplits >> 16);
            ctrl->taskCount[r] = linTotal;
            ctrl->searchCount[r] = searchTotal;
            ctrl->nl[r + 1] = newTotal;
            ctrl->rounds = r + 1;
            if (newTotal > cap) {
                ctrl->status = CS_ERR_CAPACITY;
                ctrl->done = 1;
            } else {
                Kout[newTotal] = kKeyEnd;                    // A11: terminal element of K'
                offOut[newTotal] = n;
                ctrl->numLeaves = newTotal;
                ctrl->converged = 0;
                if (r == lastRound) {
                    ctrl->status = CS_ERR_NOT_CONVERGED;
                    ctrl->done = 1;
                }
            }
        }
        __syncthreads();                                     // everyone is done with the staged tile and sm.base
    }
}

// ---- one round, second half: f for the new boundaries (Eq. 3) ------------------------------------------
// A split leaf with particle range [lo, hi) needs lower_bound(P, K'[p + c]) for c = 1..7, all inside [lo, hi):
//   * short ranges (<= kLinearMax keys; nearly all: a leaf that splits holds little more than N_crit
//     particles unless the tree is still coarse): one warp per leaf reads the range's keys once, coalesced,
//     and counts the keys below every child boundary with ballots (the keys' child octants are
//     non-decreasing, so boundary c lies after the keys of octants < c);
//   * long ranges: one warp per (leaf, boundary), a 32-ary search: 32 probes per step, 5 bits of the range
//     per dependent memory round trip instead of 1.
__device__ __forceinline__ u32 warpLowerBound32(const u64* __restrict__ P, u32 lo, u32 hi, u64 key, u32 lane)
{
    // invariant: answer in [lo, hi]; P[lo-1] < key (or lo is the range start), P[hi] >= key (or hi is the end)
    while (hi - lo > 32) {
        const u32 w = hi - lo;
        const u32 s = (w + 31) / 32;                               // probe stride
        const u32 idx = lo + (lane + 1) * s - 1;                   // last probe may fall beyond hi - 1
        const bool below = idx < hi && __ldg(P + idx) < key;
        const u32 m = __popc(__ballot_sync(kFull, below));         // probes are monotone: m leading trues
        const u32 newLo = lo + m * s;
        const u32 newHi = lo + (m + 1) * s - 1;
        lo = newLo < hi ? newLo : hi;
        hi = newHi < hi ? newHi : hi;
    }
    const u32 idx = lo + lane;
    const bool below = idx < hi && __ldg(P + idx) < key;
    return lo + __popc(__ballot_sync(kFull, below));
}

__device__ __forceinline__ void
    leafSearchBody(const DeviceCtrl* ctrl, const u64* __restrict__ P, const u64* Kout, u32* offOut, const uint4* tasksLin,
                   const uint4* tasksSearch, u32 maxTasks, u32 r)
{
    const u32 st = ldVolatile(&ctrl->status);
    if (st == CS_ERR_CAPACITY || st == CS_ERR_NOT_CORNERSTONE) return;   // task lists incomplete
    u32 numLin = ldVolatile(&ctrl->taskCount[r]), numSearch = ldVolatile(&ctrl->searchCount[r]);
    if (numLin > maxTasks) numLin = maxTasks;
    if (numSearch > maxTasks) numSearch = maxTasks;
    const u32 lane = laneId();
    const u32 warpsPerGrid = gridDim.x * (blockDim.x >> 5);
    const u32 warpId = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);

    // ---- short ranges: one warp per split leaf, 128 keys (4 per lane, loaded together) per step; the next
    // leaf's descriptor is fetched while this one's keys are on their way -------------------------------------
    uint4 next = make_uint4(0, 0, 0, 0);
    if (warpId < numLin) next = __ldcg(tasksLin + warpId);               // .cg: written earlier in this launch
    for (u32 t = warpId; t < numLin; t += warpsPerGrid) {
        const uint4 task = next;
        if (t + warpsPerGrid < numLin) next = __ldcg(tasksLin + t + warpsPerGrid);
        const u32 p = task.x, lo = task.y, hi = task.z, sh = task.w;     // child length = 8^(sh/3)
        u32 below = 0;                                                   // lane c: keys of the range in child octants < c
        for (u32 base = lo; base < hi; base += 128) {
            u32 d[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const u32 idx = base + q * 32 + lane;
                d[q] = idx < hi ? (u32)(__ldg(P + idx) >> sh) & 7u : 8u;
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
#pragma unroll
                for (u32 c = 1; c < 8; ++c) {
                    const u32 m = __popc(__ballot_sync(kFull, d[q] < c));
                    if (lane == c) below += m;
                }
            }
        }
        if (lane >= 1 && lane < 8) offOut[p + lane] = lo + below;
    }

    // ---- long ranges: one warp per (task, child boundary), 32-ary search -----------------------------
    const u32 units = numSearch * 7u;
    for (u32 u = warpId; u < units; u += warpsPerGrid) {
        const u32 t = u / 7u, c = u % 7u + 1u;
        const uint4 task = __ldcg(tasksSearch + t);
        const u32 p = task.x, lo = task.y, hi = task.z;
        const u64 key = __ldcg(Kout + p) + ((u64)c << task.w);
        const u32 pos = warpLowerBound32(P, lo, hi, key, lane);
        if (lane == 0) offOut[p + c] = pos;
    }
}

// ---- hand the result to the caller: leaves, counts (f of the returned K), and off[] ---------------
__device__ __forceinline__ void leavesEmitBody(const u64* K, const u32* off, u32 nl, u64* __restrict__ leaves,
                                               u32* __restrict__ counts, u32* __restrict__ offFinal)
{
    const u32 stride = gridDim.x * blockDim.x;
    for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i <= nl; i += stride) {
        const u32 o = __ldcg(off + i);
        leaves[i] = __ldcg(K + i);
        offFinal[i] = o;
        if (i < nl && counts) counts[i] = __ldcg(off + i + 1) - o;
    }
}

// the one-pass build (cs_leaves_direct.cu) leaves its result in K0 / off0
__global__ void __launch_bounds__(256) leavesEmitKernel(const DeviceCtrl* ctrl, const u64* K0, const u32* off0, u64* leaves,
                                                        u32* counts, u32* offFinal)
{
    chainEnter();
    const u32 st = ctrl->status;
    if (st == CS_ERR_CAPACITY || st == CS_ERR_NOT_CORNERSTONE) return;   // outputs untouched
    leavesEmitBody(K0, off0, ctrl->nl[ctrl->rounds], leaves, counts, offFinal);
}

// ---- all rounds of a build in one cooperative launch ---------------------------------------------------
// Round r: decide (g1) | grid barrier | scatter (g2, g3) | grid barrier | f for the new boundaries
// (leafSearchBody) | grid barrier.  What one phase writes for the next is read with .cg loads after the
// barrier.  After the first barrier every CTA sees whether any O_i != 1: if none, this was the confirming
// round, K' = K and the loop ends for the whole grid at once; the last tile of the scatter phase
// closes a round that did change something (sizes, capacity, round limit) before the second barrier.
// The result is then handed to the caller by the same grid.
struct RoundsArgs {
    DeviceCtrl* ctrl;
    const u64* P;
    u32 n;
    u64* K[2];
    u32* off[2];
    u32* opk;                   // [tiles][kLeafBlock] O of 8 leaves per word
    TileInfo* info;             // [tiles]
    uint4* tasksLin;
    uint4* tasksSearch;
    u32 maxTasks;
    u32 bucket, cap, roundsToLaunch;
    u64 minDelta;               // key range of a leaf at the maximum depth: 1, or 8^11 for 30-bit keys held in the top digits
    bool emitEarly;             // rounds after the first also hand their input array to the caller: if such a round turns out to
                                // be the confirming one, the result is already in place (incremental starts: round 1, normally)
    u64* leaves;
    u32* counts;
    u32* offFinal;
};

__global__ void __launch_bounds__(kLeafBlock, 5) leafRoundsKernel(const RoundsArgs a)
{
    __shared__ LeafTileSmem sm;
    cg::grid_group grid = cg::this_grid();
    DeviceCtrl* ctrl = a.ctrl;
    if (ldVolatile(&ctrl->done)) return;                     // the start array was refused (written before this launch)
    u32 nl = ldVolatile(&ctrl->nl[0]);
    u32 final = 0;                                           // buffer pair that holds the result
    for (u32 r = 0; r < a.roundsToLaunch; ++r) {
        const u32 in = r & 1, out = in ^ 1;
        const bool emitNow = a.emitEarly && r > 0;
        leafDecideBody(sm, ctrl, a.n, nl, a.K[in], a.off[in], a.opk, a.info, r, a.bucket, a.minDelta, emitNow, a.leaves, a.counts,
                       a.offFinal);
        grid.sync();
        if (ldVolatile(&ctrl->changed[r]) == 0) {            // O_i = 1 for all i: converged, K' = K
            if (blockIdx.x == 0 && threadIdx.x == 0) {
                ctrl->rounds = r + 1;
                ctrl->nl[r + 1] = nl;
                ctrl->numLeaves = nl;
                ctrl->converged = 1;
                ctrl->done = 1;
            }
            if (emitNow) return;                             // the result is in the caller's arrays already
            final = in;
            break;
        }
        leafScatterBody(sm, ctrl, a.n, nl, a.K[in], a.off[in], a.K[out], a.off[out], a.opk, a.info, a.tasksLin,
                        a.tasksSearch, a.maxTasks, r, a.cap, a.roundsToLaunch - 1);
        grid.sync();
        if (ldVolatile(&ctrl->taskCount[r]) | ldVolatile(&ctrl->searchCount[r])) {   // some leaf was split
            leafSearchBody(ctrl, a.P, a.K[out], a.off[out], a.tasksLin, a.tasksSearch, a.maxTasks, r);
            grid.sync();
        }
        final = out;
        nl = ldVolatile(&ctrl->nl[r + 1]);
        if (ldVolatile(&ctrl->done)) break;                  // capacity exceeded, or the round limit reached
    }
    if (ldVolatile(&ctrl->status) == CS_ERR_CAPACITY) return;   // outputs untouched
    leavesEmitBody(a.K[final], a.off[final], nl, a.leaves, a.counts, a.offFinal);
}

// co-resident CTAs of leafRoundsKernel per SM (per device: once per cs_create)
cs_status leavesInit(cs_context* ctx)
{
    int perSM = 0;
    CS_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&perSM, leafRoundsKernel, kLeafBlock, 0));
    if (perSM < 1) return fail(ctx, CS_ERR_CUDA, "leafRoundsKernel does not fit on an SM");
    ctx->roundsGrid = (u32)perSM * (u32)ctx->numSMs;
    return CS_OK;
}

// f (Eq. 3) of a whole array K by the merge pass: ctx->leafK[0] = K (checked against Eq. 2: a violation sets
// ctrl->status), ctx->leafOff[0][i] = lower_bound(P, K_i) for i = 0 .. nl.  The caller has cleared the control block.
cs_status enqueueLocateLeaves(cs_context* ctx, const u64* P, u64 n, const u64* K, u32 nl, cudaStream_t s)
{
    const u32 persistentGrid = (u32)ctx->numSMs * 8;
    const u32 locTiles = n ? divUp(n, kLocTile) : 1u;
    u32 gs = divUp((u64)(nl > locTiles ? nl : locTiles) + 1, 256);
    if (gs > persistentGrid) gs = persistentGrid;
    leafSplitKernel<<<gs, 256, 0, s>>>(ctx->ctrl, P, (u32)n, K, nl, ctx->leafK[0], ctx->dirTotals);
    CS_LAUNCH_CHECK(ctx, "leafSplitKernel");
    leafLocateKernel<<<locTiles, kLocBlock, 0, s>>>(P, (u32)n, K, ctx->dirTotals, ctx->leafOff[0]);
    CS_LAUNCH_CHECK(ctx, "leafLocateKernel");
    return CS_OK;
}

cs_status enqueueLeaves(cs_context* ctx, const u64* P, u64 n, u32 bucket, const u64* prevLeaves, u32 prevNumLeaves,
                        u32 maxRounds, u64* leaves, u32* counts, u32 leafCapacity, u32 maxLevel, cudaStream_t s)
{
    StageTimer t(ctx, CS_STAGE_LEAVES, s);
    const u32 cap = leafCapacity < ctx->maxLeaves ? leafCapacity : ctx->maxLeaves;
    DeviceCtrl* ctrl = ctx->ctrl;
    CS_CUDA(ctx, cudaMemsetAsync(ctrl, 0, sizeof(DeviceCtrl), s));
    const u32 persistentGrid = (u32)ctx->numSMs * 8;
    // From the root and to convergence the fixpoint is built in one pass over P (cs_leaves_direct.cu);
    // the rounds below serve incremental starts, bounded round counts and cs_setLeafMode(ITERATIVE).
    if (!prevLeaves && maxRounds == 0 && ctx->leafMode != CS_LEAVES_ITERATIVE && leavesDirectSupported(ctx, bucket)) {
        CS_TRY(enqueueLeavesDirect(ctx, P, n, bucket, cap, maxLevel, s));
        u32 g = divUp((u64)cap + 1, 256);
        if (g > persistentGrid) g = persistentGrid;
        launchChained(leavesEmitKernel, dim3(g), dim3(256), 0, s, ctrl, ctx->leafK[0], ctx->leafOff[0], leaves, counts, ctx->leafOffFinal);
        CS_LAUNCH_CHECK(ctx, "leavesEmitKernel");
        return CS_OK;
    }
    if (prevLeaves) {
        // f of the previous array by one merge pass over P
        CS_TRY(enqueueLocateLeaves(ctx, P, n, prevLeaves, prevNumLeaves, s));
    } else {
        leavesInitRootKernel<<<1, 32, 0, s>>>(ctrl, ctx->leafK[0], ctx->leafOff[0], (u32)n);
        CS_LAUNCH_CHECK(ctx, "leavesInitRootKernel");
    }
    RoundsArgs a;
    a.ctrl = ctrl; a.P = P; a.n = (u32)n;
    a.K[0] = ctx->leafK[0]; a.K[1] = ctx->leafK[1]; a.off[0] = ctx->leafOff[0]; a.off[1] = ctx->leafOff[1];
    a.tasksLin = ctx->leafTasks; a.tasksSearch = ctx->leafTasks + ctx->maxTasks; a.maxTasks = ctx->maxTasks;
    a.opk = ctx->leafOpk; a.info = reinterpret_cast<TileInfo*>(ctx->leafTileInfo);
    a.roundsToLaunch = (maxRounds == 0 || maxRounds > (u32)kMaxRounds) ? (u32)kMaxRounds : maxRounds;
    a.bucket = bucket; a.cap = cap;
    a.minDelta = 1ull << (3 * (kL - (int)maxLevel));
    a.emitEarly = prevLeaves != nullptr;
    a.leaves = leaves; a.counts = counts; a.offFinal = ctx->leafOffFinal;
    // every CTA must be resident (grid barriers): at most what the device holds, at most one CTA per tile
    // of the largest array this call can produce
    u32 grid = divUp((u64)cap + 1, kLeafTile);
    if (grid > ctx->roundsGrid) grid = ctx->roundsGrid;
    void* args[] = {(void*)&a};
    CS_CUDA(ctx, cudaLaunchCooperativeKernel((const void*)leafRoundsKernel, dim3(grid), dim3(kLeafBlock), args, 0, s));
    CS_LAUNCH_CHECK(ctx, "leafRoundsKernel");
    return CS_OK;
}

}  // namespace cs
