// H4-H8: cornerstone leaf array by iterating f and g = g3 o g2 o g1 (Eqs. 2-9).
//
// Two kernel launches per round do f, g1, g2, g3:
//   f   (Eq. 3)  the lower-bound position off_i of every K_i in P is carried with K from round to
//                round; N_i = off_{i+1} - off_i.  Only the 7 new boundaries of a split leaf are
//                searched, inside the parent's particle range [off_i, off_{i+1}) (second kernel).
//   g1  (Eq. 5)  O_i in {8, 0, 1} per leaf (readings A7, A8, A9).
//   g2  (Eq. 6)  exclusive prefix sum of O: in-tile scan + decoupled look-back across tiles.
//   g3  (Eqs. 7-9, A10, A11) scatter of kept keys / 8 child keys to K'.
// All sizes stay in the device control block; round r reads nl[r] and writes nl[r+1], so the
// host can enqueue the maximum number of rounds without reading anything back: rounds after
// convergence return at once (ctrl->done).
#include "cs_device.cuh"

namespace cs {

__device__ __forceinline__ u32 ldVolatile(const u32* p) { return *(const volatile u32*)p; }

// ---- divergence levels ----------------------------------------------------------------------------
// D[i] = number of leading octal digits that the sorted neighbours P[i-1] and P[i] share (21 for
// equal keys; D[0] = 0).  Inside a node of level l every D is >= l, and the positions with
// D == l are exactly the places where the node's particles change child octant.  One byte per
// particle, written once per sorted array: the refinement rounds then locate the child
// boundaries of short leaves by scanning bytes instead of re-reading 8-byte keys every round.
__global__ void __launch_bounds__(256) divergenceKernel(const u64* __restrict__ P, u32 n, unsigned char* __restrict__ D)
{
    const u32 lane = laneId();
    const u32 pairs = (n + 1) >> 1;
    const u32 stride = gridDim.x * blockDim.x;
    const u32 rounds = (pairs + stride - 1) / stride;            // warp-uniform trip count (shuffles inside)
    for (u32 it = 0; it < rounds; ++it) {
        const u32 t = it * stride + blockIdx.x * blockDim.x + threadIdx.x;
        const u32 i = 2 * t;
        u64 a = 0, b = 0;
        if (i + 1 < n) {
            const ulonglong2 v = ldStreamU2(P + i);
            a = v.x;
            b = v.y;
        } else if (i < n) a = ldStreamU64(P + i);
        u64 prev = __shfl_up_sync(kFull, b, 1);
        if (lane == 0) prev = (i > 0 && i < n) ? P[i - 1] : a;
        if (i < n) {
            const u32 d0 = i == 0 ? 0u : (u32)(__clzll((long long)(prev ^ a)) - 1) / 3u;
            const u32 d1 = (u32)(__clzll((long long)(a ^ b)) - 1) / 3u;
            if (i + 1 < n) *reinterpret_cast<unsigned short*>(D + i) = (unsigned short)(d0 | (d1 << 8));
            else D[i] = (unsigned char)d0;
        }
    }
}

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

// Copy the caller's previous cornerstone array into the workspace, check Eq. 2
// and locate every K_i in P (the full f of the first incremental round).
__global__ void __launch_bounds__(256) leavesInitPrevKernel(DeviceCtrl* ctrl, const u64* __restrict__ P, u32 n,
                                                            const u64* __restrict__ prev, u32 nlPrev, u64* K0,
                                                            u32* off0)
{
    const u32 stride = gridDim.x * blockDim.x;
    bool bad = false;
    for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i <= nlPrev; i += stride) {
        const u64 k = prev[i];
        if (i == 0 && k != 0) bad = true;
        if (i == nlPrev) {
            if (k != kKeyEnd) bad = true;
            off0[i] = n;
        } else {
            const u64 kn = prev[i + 1];
            const u64 delta = kn - k;
            if (kn <= k || !isPowerOf8(delta) || (k & (delta - 1))) bad = true;
            off0[i] = lowerBound(P, 0, n, k);
        }
        K0[i] = k;
    }
    if (bad) {
        ctrl->status = CS_ERR_NOT_CORNERSTONE;
        ctrl->done = 1;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) ctrl->nl[0] = nlPrev;
}

constexpr u32 kLinearMax = 1024;   // split leaves with at most this many particles are counted linearly

// ---- one round, kernel 1: g1, g2, g3 and the task list for f ----------------------------------------
// Each split leaf becomes a search task (slot of its first child in K', end of its particle
// range): the 7 inner child boundaries are located in P by leafSearchKernel, spread over the
// whole GPU, instead of serially by the thread that owns the leaf.
__global__ void __launch_bounds__(kLeafBlock)
    leafRoundKernel(DeviceCtrl* ctrl, u32 n, const u64* __restrict__ Kin, const u32* __restrict__ offIn,
                    u64* __restrict__ Kout, u32* __restrict__ offOut, uint2* __restrict__ tasksLin,
                    uint2* __restrict__ tasksSearch, u32 maxTasks, u64* lookback, u32 epoch, u32 r, u32 bucket, u32 cap,
                    u32 lastRound)
{
    __shared__ u32 sTile, sPrefix, sDone, sLinBase, sSearchBase;
    __shared__ u32 warpSums[kLeafBlock / 32 + 1];
    __shared__ u32 warpSums2[kLeafBlock / 32 + 1];
    if (threadIdx.x == 0) sDone = ldVolatile(&ctrl->done);   // one read per CTA: the decision must be uniform
    __syncthreads();
    if (sDone) return;
    const u32 nl = ctrl->nl[r];
    const u32 tiles = (nl + kLeafTile - 1) / kLeafTile;
    const u32 tid = threadIdx.x;
    // Tiles are handed out by an atomic ticket (a tile only waits for tiles that already run).  The
    // ticket of the NEXT tile is drawn by the last thread while the current tile is in flight, so
    // its round trip is off the critical path.
    u32 nextTicket = 0;
    if (tid == kLeafBlock - 1) sTile = atomicAdd(&ctrl->ticket[r], 1u);
    for (;;) {
        __syncthreads();
        const u32 tile = sTile;
        if (tile >= tiles) break;
        const u32 first = tile * kLeafTile + tid * kLeafItems;

        u64 K[kLeafItems + 1];
        u32 off[kLeafItems + 1];
#pragma unroll
        for (int k = 0; k <= kLeafItems; ++k) {
            u32 i = first + k;
            K[k] = i <= nl ? Kin[i] : kKeyEnd;
            off[k] = i <= nl ? offIn[i] : n;
        }
        if (tid == kLeafBlock - 1) nextTicket = atomicAdd(&ctrl->ticket[r], 1u);
        // g1: rebalance decision (Eq. 5)
        u32 O[kLeafItems];
        u32 sum = 0, splits = 0;
        bool anyChange = false;
#pragma unroll
        for (int k = 0; k < kLeafItems; ++k) {
            const u32 i = first + k;
            u32 o = 0;
            if (i < nl) {
                const u64 delta = K[k + 1] - K[k];
                const u32 cnt = off[k + 1] - off[k];                      // f: N_i
                o = 1;
                if (cnt > bucket && delta > 1) o = 8;                    // split (A7: not at depth L)
                else if (delta != kKeyEnd) {                             // the root never merges (A9)
                    const u32 j = (u32)(K[k] >> (__ffsll((long long)delta) - 1)) & 7u;   // octant among siblings (delta = 8^m)
                    if (j != 0 && i >= j && i - j + 8 <= nl) {
                        const u32 a = i - j;
                        if (Kin[a + 8] - Kin[a] == (delta << 3)) {       // all 8 siblings are leaves
                            const u32 combined = offIn[a + 8] - offIn[a];
                            if (combined <= bucket) o = 0;               // merged away (A8)
                        }
                    }
                }
                anyChange |= (o != 1);
            }
            O[k] = o;
            sum += o;
            // split leaves become search tasks: short particle ranges are counted linearly, long ones searched
            if (o == 8) splits += (off[k + 1] - off[k] <= kLinearMax) ? 1u : (1u << 16);
        }
        // g2: exclusive prefix sum (Eq. 6): tile scan + look-back
        u32 total, totalSplits;
        const u32 excl = blockExclusiveScan<kLeafBlock>(sum, warpSums, &total);
        u32 taskSlot = blockExclusiveScan<kLeafBlock>(splits, warpSums2, &totalSplits);
        if (tid < 32) {                               // warp 0: publish, then warp-wide look-back
            u64* st = lookback + tile;
            u32 p = 0;
            if (tile == 0) {
                if (tid == 0) lbStore(st, lbPack(epoch, kLbPrefix, total));
            } else {
                if (tid == 0) lbStore(st, lbPack(epoch, kLbAggregate, total));
                p = lbLookBackWarp(lookback, tile, epoch);
                if (tid == 0) lbStore(st, lbPack(epoch, kLbPrefix, p + total));
            }
            if (tid == 0) {
                sPrefix = p;
                const u32 nLin = totalSplits & 0xFFFFu, nSearch = totalSplits >> 16;
                sLinBase = nLin ? atomicAdd(&ctrl->taskCount[r], nLin) : 0u;
                sSearchBase = nSearch ? atomicAdd(&ctrl->searchCount[r], nSearch) : 0u;
            }
        }
        const int tileChanged = __syncthreads_or(anyChange ? 1 : 0);
        // g3: node rebalancing (Eqs. 8, 9)
        u32 p = sPrefix + excl;
        u32 linSlot = sLinBase + (taskSlot & 0xFFFFu), searchSlot = sSearchBase + (taskSlot >> 16);
#pragma unroll
        for (int k = 0; k < kLeafItems; ++k) {
            if (O[k] == 1) {
                if (p < cap) {
                    Kout[p] = K[k];
                    offOut[p] = off[k];
                }
                p += 1;
            } else if (O[k] == 8) {
                const u64 step = (K[k + 1] - K[k]) >> 3;
                if (p + 8 <= cap) {
#pragma unroll
                    for (u32 c = 0; c < 8; ++c) Kout[p + c] = K[k] + c * step;
                    offOut[p] = off[k];
                }
                const bool lin = off[k + 1] - off[k] <= kLinearMax;
                u32& slot = lin ? linSlot : searchSlot;
                if (p + 8 <= cap && slot < maxTasks) (lin ? tasksLin : tasksSearch)[slot] = make_uint2(p, off[k + 1]);
                ++slot;
                p += 8;
            }
        }
        if (tid == 0) {
            const u32 newTotal = sPrefix + total;
            if (tile == tiles - 1) {                         // A11: terminal element of K'
                if (newTotal <= cap) {
                    Kout[newTotal] = kKeyEnd;
                    offOut[newTotal] = n;
                }
                ctrl->nl[r + 1] = newTotal;
            }
            if (tileChanged) atomicOr(&ctrl->changed[r], 1u);
            __threadfence();
            const u32 finished = atomicAdd(&ctrl->tilesDone[r], 1u) + 1u;
            if (finished == tiles) {                         // last tile to finish closes the round
                __threadfence();
                const u32 nlNew = ldVolatile(&ctrl->nl[r + 1]);
                const u32 ch = ldVolatile(&ctrl->changed[r]);
                ctrl->rounds = r + 1;
                if (nlNew > cap) {
                    ctrl->status = CS_ERR_CAPACITY;
                    ctrl->done = 1;
                } else {
                    ctrl->numLeaves = nlNew;
                    ctrl->converged = ch ? 0u : 1u;
                    if (!ch) ctrl->done = 1;                 // O_i = 1 for all i
                    else if (r == lastRound) {
                        ctrl->status = CS_ERR_NOT_CONVERGED;
                        ctrl->done = 1;
                    }
                }
            }
        }
        __syncthreads();                                     // everyone is done with sTile / sPrefix
        if (tid == kLeafBlock - 1) sTile = nextTicket;
    }
}

// ---- one round, kernel 2: f for the new boundaries (Eq. 3) ------------------------------------------
// A split leaf with particle range [lo, hi) needs lower_bound(P, K'[p + c]) for c = 1..7, all
// inside [lo, hi).  Work unit = (task, c), one warp each:
//   * short ranges (<= kLinearMax keys): 8 lanes scan the range's divergence bytes (see
//     divergenceKernel) for changes of child octant; only the hits touch the keys.
//   * long ranges: a 32-ary search, 32 probes per step (5 bits of the range per dependent
//     memory round trip instead of 1).
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

__global__ void __launch_bounds__(256)
    leafSearchKernel(const DeviceCtrl* ctrl, const u64* __restrict__ P, const unsigned char* __restrict__ D,
                     const u64* __restrict__ Kout, u32* __restrict__ offOut, const uint2* __restrict__ tasksLin,
                     const uint2* __restrict__ tasksSearch, u32 maxTasks, u32 r)
{
    if (ctrl->status == CS_ERR_CAPACITY || ctrl->status == CS_ERR_NOT_CORNERSTONE) return;   // task lists incomplete
    u32 numLin = ctrl->taskCount[r], numSearch = ctrl->searchCount[r];
    if (numLin > maxTasks) numLin = maxTasks;
    if (numSearch > maxTasks) numSearch = maxTasks;
    const u32 lane = laneId();
    const u32 warpsPerGrid = gridDim.x * (blockDim.x >> 5);
    const u32 warpId = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);

    // ---- short ranges: 8 lanes per task, 4 tasks per warp.  The lanes scan the divergence bytes of
    // the range, 16 per load, for D == level (a change of child octant); the few hits read the two
    // neighbouring keys and record the boundary for every child index the change skips ------------
    const u32 gl = lane & 7u;
    for (u32 t0 = warpId * 4u; t0 < numLin; t0 += warpsPerGrid * 4u) {
        const u32 t = t0 + (lane >> 3);
        const bool valid = t < numLin;
        u32 p = 0, lo = 0, hi = 0, level = 0;
        int sh = 0;
        if (valid) {
            const uint2 task = tasksLin[t];
            p = task.x;
            hi = task.y;
            lo = offOut[p];
            sh = __ffsll((long long)(Kout[p + 1] - Kout[p])) - 1;         // child length = 8^(sh/3)
            level = (u32)kL - 1u - (u32)sh / 3u;                          // level of the split leaf
        }
        const bool nonEmpty = hi > lo;                                    // a split leaf always has particles
        if (valid && nonEmpty && gl == 0) {                               // ends of the range
            const u32 cf = (u32)(__ldg(P + lo) >> sh) & 7u;
            const u32 cl = (u32)(__ldg(P + hi - 1) >> sh) & 7u;
            for (u32 c = 1; c <= cf; ++c) offOut[p + c] = lo;
            for (u32 c = cl + 1; c < 8; ++c) offOut[p + c] = hi;
        }
        // interior positions lo < i < hi with D[i] == level
        const u32 a0 = (lo + 1u) & ~15u;                                  // 16-byte aligned start
        u32 iters = (valid && hi > lo + 1u) ? (hi - a0 + 127u) / 128u : 0u;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) iters = max(iters, __shfl_xor_sync(kFull, iters, o));
        const u32 want = level * 0x01010101u;
        for (u32 it = 0; it < iters; ++it) {
            const u32 i0 = a0 + it * 128u + gl * 16u;
            if (!valid || i0 >= hi) continue;
            const uint4 v = *reinterpret_cast<const uint4*>(D + i0);
            const u32 w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                u32 eq = __vcmpeq4(w[q], want);                           // 0xFF in every byte equal to level
                while (eq) {
                    const u32 byte = (__ffs((int)eq) - 1) >> 3;
                    eq &= ~(0xFFu << (byte * 8));
                    const u32 i = i0 + q * 4u + byte;
                    if (i > lo && i < hi) {
                        const u32 c0 = (u32)(__ldg(P + i - 1) >> sh) & 7u;
                        const u32 c1 = (u32)(__ldg(P + i) >> sh) & 7u;
                        for (u32 c = c0 + 1; c <= c1; ++c) offOut[p + c] = i;
                    }
                }
            }
        }
    }

    // ---- long ranges: one warp per (task, child boundary), 32-ary search -----------------------------
    const u32 units = numSearch * 7u;
    for (u32 u = warpId; u < units; u += warpsPerGrid) {
        const u32 t = u / 7u, c = u % 7u + 1u;
        const uint2 task = tasksSearch[t];
        const u32 p = task.x, hi = task.y;
        const u32 lo = offOut[p];
        const u32 pos = warpLowerBound32(P, lo, hi, Kout[p + c], lane);
        if (lane == 0) offOut[p + c] = pos;
    }
}

// ---- hand the result to the caller: leaves, counts (f of the returned K), and off[] ---------------
__global__ void __launch_bounds__(256) leavesEmitKernel(const DeviceCtrl* ctrl, const u64* K0, const u64* K1,
                                                        const u32* off0, const u32* off1, u64* leaves, u32* counts,
                                                        u32* offFinal)
{
    const u32 st = ctrl->status;
    if (st == CS_ERR_CAPACITY || st == CS_ERR_NOT_CORNERSTONE) return;   // outputs untouched
    const u32 rounds = ctrl->rounds;
    const u32 nl = ctrl->nl[rounds];
    const bool second = (rounds & 1) && !ctrl->directBuild;      // the one-pass build always writes K0 / off0
    const u64* K = second ? K1 : K0;
    const u32* off = second ? off1 : off0;
    const u32 stride = gridDim.x * blockDim.x;
    for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i <= nl; i += stride) {
        const u32 o = off[i];
        leaves[i] = K[i];
        offFinal[i] = o;
        if (i < nl && counts) counts[i] = off[i + 1] - o;
    }
}

cs_status enqueueLeaves(cs_context* ctx, const u64* P, u64 n, u32 bucket, const u64* prevLeaves, u32 prevNumLeaves,
                        u32 maxRounds, u64* leaves, u32* counts, u32 leafCapacity, cudaStream_t s)
{
    StageTimer t(ctx, CS_STAGE_LEAVES, s);
    const u32 cap = leafCapacity < ctx->maxLeaves ? leafCapacity : ctx->maxLeaves;
    DeviceCtrl* ctrl = ctx->ctrl;
    CS_CUDA(ctx, cudaMemsetAsync(ctrl, 0, sizeof(DeviceCtrl), s));
    const u32 persistentGrid = (u32)ctx->numSMs * 8;
    // From the root and to convergence the fixpoint is built in one pass over P (cs_leaves_direct.cu);
    // the rounds below serve incremental starts, bounded round counts and cs_setLeafMode(ITERATIVE).
    if (!prevLeaves && maxRounds == 0 && ctx->leafMode != CS_LEAVES_ITERATIVE && leavesDirectSupported(ctx, bucket)) {
        CS_TRY(enqueueLeavesDirect(ctx, P, n, bucket, cap, s));
        u32 g = divUp((u64)cap + 1, 256);
        if (g > persistentGrid) g = persistentGrid;
        leavesEmitKernel<<<g, 256, 0, s>>>(ctrl, ctx->leafK[0], ctx->leafK[1], ctx->leafOff[0], ctx->leafOff[1], leaves,
                                           counts, ctx->leafOffFinal);
        CS_LAUNCH_CHECK(ctx, "leavesEmitKernel");
        return CS_OK;
    }
    if (n) {
        u32 g = divUp((n + 1) / 2, 256);
        if (g > persistentGrid) g = persistentGrid;
        divergenceKernel<<<g, 256, 0, s>>>(P, (u32)n, ctx->divLevel);
        CS_LAUNCH_CHECK(ctx, "divergenceKernel");
    }
    if (prevLeaves) {
        u32 grid = divUp((u64)prevNumLeaves + 1, 256);
        if (grid > persistentGrid) grid = persistentGrid;
        leavesInitPrevKernel<<<grid, 256, 0, s>>>(ctrl, P, (u32)n, prevLeaves, prevNumLeaves, ctx->leafK[0],
                                                  ctx->leafOff[0]);
        CS_LAUNCH_CHECK(ctx, "leavesInitPrevKernel");
    } else {
        leavesInitRootKernel<<<1, 32, 0, s>>>(ctrl, ctx->leafK[0], ctx->leafOff[0], (u32)n);
        CS_LAUNCH_CHECK(ctx, "leavesInitRootKernel");
    }
    const u32 roundsToLaunch = (maxRounds == 0 || maxRounds > (u32)kMaxRounds) ? (u32)kMaxRounds : maxRounds;
    // grid: enough CTAs for the largest array this context can hold, capped at a persistent size
    u32 grid = divUp((u64)cap + 1, kLeafTile);
    if (grid > persistentGrid) grid = persistentGrid;
    for (u32 r = 0; r < roundsToLaunch; ++r) {
        const u32 epoch = nextEpoch(ctx, s);
        // early rounds from the root touch at most 8^r leaves: do not launch more CTAs than that
        u32 g = grid;
        if (!prevLeaves && r < 8) {
            u32 bound = divUp(1ull << (3 * r), kLeafTile);
            if (bound < g) g = bound;
        }
        leafRoundKernel<<<g, kLeafBlock, 0, s>>>(ctrl, (u32)n, ctx->leafK[r & 1], ctx->leafOff[r & 1],
                                                 ctx->leafK[(r + 1) & 1], ctx->leafOff[(r + 1) & 1], ctx->leafTasks,
                                                 ctx->leafTasks + ctx->maxTasks, ctx->maxTasks, ctx->tileLookback,
                                                 epoch, r, bucket, cap, roundsToLaunch - 1);
        CS_LAUNCH_CHECK(ctx, "leafRoundKernel");
        // searches of this round's split leaves: at most 7 * 8^r warps of work in the early rounds
        u32 gs = persistentGrid;
        if (!prevLeaves && r < 4) {
            u32 bound = divUp(7ull << (3 * r), 8);
            if (bound < gs) gs = bound;
        }
        leafSearchKernel<<<gs, 256, 0, s>>>(ctrl, P, ctx->divLevel, ctx->leafK[(r + 1) & 1], ctx->leafOff[(r + 1) & 1],
                                            ctx->leafTasks, ctx->leafTasks + ctx->maxTasks, ctx->maxTasks, r);
        CS_LAUNCH_CHECK(ctx, "leafSearchKernel");
    }
    leavesEmitKernel<<<grid, 256, 0, s>>>(ctrl, ctx->leafK[0], ctx->leafK[1], ctx->leafOff[0], ctx->leafOff[1],
                                          leaves, counts, ctx->leafOffFinal);
    CS_LAUNCH_CHECK(ctx, "leavesEmitKernel");
    return CS_OK;
}

}  // namespace cs
