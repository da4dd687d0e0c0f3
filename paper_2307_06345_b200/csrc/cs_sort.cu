// H3: stable LSD radix sort of (u64 key, u32 index) pairs -- PAPER.md:70, 168; A5.
//
// "Onesweep" organisation: one histogram pass over the keys gives the global digit counts of
// all 8 passes; every pass then reads each element once and writes it once.  A pass tile is
// ranked inside the CTA (warp-level match + per-warp digit counters), the tile's position in
// each digit's output run comes from a decoupled look-back over the preceding tiles' digit
// counts, and the tile is written out through shared memory so that each digit's run is a
// contiguous burst.  Tiles take their index from an atomic ticket, so a tile only ever waits
// for tiles that are already running (forward progress).
//
// Model bytes per particle: histogram 8 + pass 0 (8 read, 12 written) + 7 x 24 = 196.
#include "cs_device.cuh"

namespace cs {

constexpr int kHistBlock = 512;
constexpr int kSortWarps = kSortBlock / 32;

__device__ __forceinline__ u32 digitOf(u64 key, int shift) { return (u32)(key >> shift) & (kRadix - 1); }

// ---- global digit histograms of all passes ----------------------------------------------------
__global__ void __launch_bounds__(kHistBlock) sortHistKernel(const u64* __restrict__ keys, u64 n, u32* gHist)
{
    __shared__ u32 sh[kSortPasses * kRadix];
    for (int i = threadIdx.x; i < kSortPasses * kRadix; i += kHistBlock) sh[i] = 0;
    __syncthreads();
    const u64 tid = (u64)blockIdx.x * kHistBlock + threadIdx.x;
    const u64 nthreads = (u64)gridDim.x * kHistBlock;
    const bool vec = (((uintptr_t)keys) & 15u) == 0;
    auto add = [&](u64 k) {
#pragma unroll
        for (int p = 0; p < kSortPasses; ++p) atomicAdd(&sh[p * kRadix + digitOf(k, p * kRadixBits)], 1u);
    };
    if (vec) {
        const u64 pairs = n >> 1;
        u64 i = tid;
        for (; i + 3 * nthreads < pairs; i += 4 * nthreads) {
            ulonglong2 a = ldStreamU2(keys + 2 * i);
            ulonglong2 b = ldStreamU2(keys + 2 * (i + nthreads));
            ulonglong2 c = ldStreamU2(keys + 2 * (i + 2 * nthreads));
            ulonglong2 d = ldStreamU2(keys + 2 * (i + 3 * nthreads));
            add(a.x); add(a.y); add(b.x); add(b.y); add(c.x); add(c.y); add(d.x); add(d.y);
        }
        for (; i < pairs; i += nthreads) {
            ulonglong2 a = ldStreamU2(keys + 2 * i);
            add(a.x); add(a.y);
        }
        if ((n & 1) && tid == 0) add(keys[n - 1]);
    } else {
        for (u64 i = tid; i < n; i += nthreads) add(ldStreamU64(keys + i));
    }
    __syncthreads();
    for (int i = threadIdx.x; i < kSortPasses * kRadix; i += kHistBlock) {
        u32 v = sh[i];
        if (v) atomicAdd(&gHist[i], v);
    }
}

// exclusive scan of each pass's 256 digit counts, in place (one CTA)
__global__ void __launch_bounds__(kRadix) sortScanHistKernel(u32* gHist)
{
    __shared__ u32 warpSums[kRadix / 32 + 1];
    for (int p = 0; p < kSortPasses; ++p) {
        u32 v = gHist[p * kRadix + threadIdx.x];
        u32 total;
        u32 excl = blockExclusiveScan<kRadix>(v, warpSums, &total);
        gHist[p * kRadix + threadIdx.x] = excl;
        __syncthreads();
    }
}

// ---- one radix pass ------------------------------------------------------------------------------
struct SortSmem {
    u64 keys[kSortTile];                 // tile in digit order
    u32 vals[kSortTile];
    u32 warpHist[kSortWarps][kRadix];    // per-warp digit counts, then exclusive prefix over warps
    u32 digitStart[kRadix];              // first tile-local slot of each digit
    u32 globalBase[kRadix];              // global slot of (digit d, tile-local slot i) = globalBase[d] + i
    u32 warpSums[kSortWarps + 1];
    u32 tile;
};

#ifndef CS_SORT_LOOKBATCH
#define CS_SORT_LOOKBATCH 4
#endif
#ifndef CS_SORT_LATELB
#define CS_SORT_LATELB 0
#endif
#ifndef CS_SORT_PREFETCH
#define CS_SORT_PREFETCH 0
#endif
constexpr int kLookBatch = CS_SORT_LOOKBATCH;   // predecessors fetched per look-back round trip

// Exclusive prefix of counter c over tiles < tile.  The words of kLookBatch predecessors are
// requested together, so one memory round trip covers kLookBatch tiles.
__device__ __forceinline__ u32 lookBackBatched(const u64* state, u32 c, u32 tile, u32 epoch)
{
    u32 excl = 0;
    int p = (int)tile - 1;
    while (p >= 0) {
        u64 w[kLookBatch];
#pragma unroll
        for (int i = 0; i < kLookBatch; ++i)
            if (p - i >= 0) w[i] = lbLoad(state + (size_t)(p - i) * kRadix + c);
#pragma unroll
        for (int i = 0; i < kLookBatch; ++i) {
            if (p - i < 0) return excl;
            while ((u32)(w[i] >> 34) != (epoch & 0x3FFFFFFFu)) {
                __nanosleep(32);
                w[i] = lbLoad(state + (size_t)(p - i) * kRadix + c);
            }
            excl += (u32)w[i];
            if (((u32)(w[i] >> 32) & 3u) == kLbPrefix) return excl;
        }
        p -= kLookBatch;
    }
    return excl;
}

// Lanes of the warp whose 8-bit digit equals this lane's: one ballot per digit bit (the native match.any
// is far slower).  Per bit: s = bit ? ~0 : 0 (bfe.s32), p = (s != 0), v = ballot(p), peers &= ~(v ^ s).
__device__ __forceinline__ u32 matchDigit(u32 d)
{
    u32 peers = kFull;
#pragma unroll
    for (int b = 0; b < kRadixBits; ++b) {
        asm("{\n\t"
            ".reg .pred p;\n\t"
            ".reg .b32 s, v;\n\t"
            "bfe.s32 s, %1, %2, 1;\n\t"
            "setp.ne.s32 p, s, 0;\n\t"
            "vote.sync.ballot.b32 v, p, 0xffffffff;\n\t"
            "lop3.b32 %0, %0, v, s, 0x90;\n\t"
            "}"
            : "+r"(peers)
            : "r"(d), "r"(b));
    }
    return peers;
}

template <bool FIRST, bool FULL>
__device__ __forceinline__ void onesweepTile(SortSmem& sm, const u64* __restrict__ keysIn, const u32* __restrict__ valsIn,
                                             u64* __restrict__ keysOut, u32* __restrict__ valsOut, u32 tile, u32 valid,
                                             int shift, const u32* __restrict__ digitBase, u64* lookback, u32 epoch)
{
    const u32 tid = threadIdx.x, lane = laneId(), warp = tid >> 5;
    const u64 base = (u64)tile * kSortTile;

    // ---- load: warp-striped, so that (warp, item, lane) order == memory order (stability) ----
    u64 key[kSortItems];
    const u32 warpOff = warp * (32 * kSortItems) + lane;
#if CS_SORT_PREFETCH
    if (!FIRST && tid < kSortTile * 4 / 128)
        asm volatile("prefetch.global.L2 [%0];" ::"l"(valsIn + base + tid * 32));
#endif
    const u64* src = keysIn + base + warpOff;
#pragma unroll
    for (int j = 0; j < kSortItems; ++j)
        key[j] = (FULL || warpOff + j * 32 < valid) ? ldStreamU64(src + j * 32) : ~0ull;   // pads sort last

    // ---- rank inside the warp: every peer reads the warp's running count of its digit (a
    // shared-memory broadcast) and the lowest peer bumps it once ------------------------------------
    u32 rankPk[(kSortItems + 1) / 2];                                        // two 16-bit ranks per register
#pragma unroll
    for (int j = 0; j < (kSortItems + 1) / 2; ++j) rankPk[j] = 0;
    u32* wh = sm.warpHist[warp];
    const u32 lt = laneMaskLt();
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
        const u32 d = digitOf(key[j], shift);
        const u32 peers = matchDigit(d);
        const u32 lower = __popc(peers & lt);
        const u32 prev = wh[d];
        __syncwarp();
        if (lower == 0) wh[d] = prev + __popc(peers);
        __syncwarp();
        rankPk[j >> 1] |= (prev + lower) << ((j & 1) * 16);
    }
    __syncthreads();

    // ---- per digit: exclusive prefix over warps, tile count, tile-local start ------------------
    u32 count = 0;
    if (tid < kRadix) {
        u32 run = 0;
#pragma unroll
        for (int w = 0; w < kSortWarps; ++w) {
            u32 c = sm.warpHist[w][tid];
            sm.warpHist[w][tid] = run;
            run += c;
        }
        count = run;
        // publish this tile's count at once: the tiles behind it can start their look-back
        const u32 real = (!FULL && tid == kRadix - 1) ? count - (kSortTile - valid) : count;   // pads are not elements
        lbStore(lookback + (size_t)tile * kRadix + tid, lbPack(epoch, tile == 0 ? kLbPrefix : kLbAggregate, real));
    }
    u32 total;
    u32 start = blockExclusiveScan<kSortBlock>(count, sm.warpSums, &total);
    if (tid < kRadix) {
        sm.digitStart[tid] = start;
#if !CS_SORT_LATELB
        // ---- decoupled look-back over preceding tiles, one thread per digit ----------------------
        u32 excl = 0;
        if (tile != 0) {
            const u32 real = (!FULL && tid == kRadix - 1) ? count - (kSortTile - valid) : count;
            excl = lookBackBatched(lookback, tid, tile, epoch);
            lbStore(lookback + (size_t)tile * kRadix + tid, lbPack(epoch, kLbPrefix, excl + real));
        }
        sm.globalBase[tid] = digitBase[tid] + excl - start;
#endif
    }
    __syncthreads();

    // ---- scatter keys, then values, into digit order in shared memory -----------------------------
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
        u32 d = digitOf(key[j], shift);
        const u32 r = (rankPk[j >> 1] >> ((j & 1) * 16)) & 0xFFFFu;
        const u32 pos = sm.digitStart[d] + wh[d] + r;
        sm.keys[pos] = key[j];
        if (j & 1) rankPk[j >> 1] = (rankPk[j >> 1] & 0xFFFFu) | (pos << 16);
        else rankPk[j >> 1] = (rankPk[j >> 1] & 0xFFFF0000u) | pos;
    }
    // values: pass 0 synthesises the identity permutation instead of reading it
    asm volatile("" ::: "memory");        // keep the value loads behind the key scatter (register pressure)
    u32 val[kSortItems];
    const u32* vsrc = valsIn + base + warpOff;
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
        if (FIRST) val[j] = (u32)base + warpOff + j * 32;
        else val[j] = (FULL || warpOff + j * 32 < valid) ? ldStreamU32(vsrc + j * 32) : 0u;
    }
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) sm.vals[(rankPk[j >> 1] >> ((j & 1) * 16)) & 0xFFFFu] = val[j];
#if CS_SORT_LATELB
    // ---- decoupled look-back, after the shared-memory scatter: the predecessors have had that much
    // longer to publish their prefixes, and the other warps are not kept waiting at a barrier ---------
    if (tid < kRadix) {
        u32 excl = 0;
        if (tile != 0) {
            const u32 real = (!FULL && tid == kRadix - 1) ? count - (kSortTile - valid) : count;
            excl = lookBackBatched(lookback, tid, tile, epoch);
            lbStore(lookback + (size_t)tile * kRadix + tid, lbPack(epoch, kLbPrefix, excl + real));
        }
        sm.globalBase[tid] = digitBase[tid] + excl - start;
    }
#endif
    __syncthreads();

    // ---- write out: consecutive threads -> consecutive slots of a digit's run ----------------------
#pragma unroll
    for (int k = 0; k < kSortItems; ++k) {
        const u32 i = tid + k * kSortBlock;
        if (FULL || i < valid) {
            const u64 kk = sm.keys[i];
            const u32 dst = sm.globalBase[digitOf(kk, shift)] + i;
            keysOut[dst] = kk;
            valsOut[dst] = sm.vals[i];
        }
    }
}

template <bool FIRST>
__global__ void __launch_bounds__(kSortBlock, kSortMinBlocks)
    onesweepKernel(const u64* __restrict__ keysIn, const u32* __restrict__ valsIn, u64* __restrict__ keysOut,
                   u32* __restrict__ valsOut, u32 n, int shift, const u32* __restrict__ digitBase /*scanned hist*/,
                   u32* ticket, u64* lookback, u32 epoch)
{
    extern __shared__ __align__(16) unsigned char smemRaw[];
    SortSmem& sm = *reinterpret_cast<SortSmem*>(smemRaw);
    const u32 tid = threadIdx.x;
    if (tid == 0) sm.tile = atomicAdd(ticket, 1u);
    for (int i = tid; i < kSortWarps * kRadix; i += kSortBlock) (&sm.warpHist[0][0])[i] = 0;
    __syncthreads();
    const u32 tile = sm.tile;
    const u64 base = (u64)tile * kSortTile;
    const u32 valid = (u32)((n - base) < (u64)kSortTile ? (n - base) : (u64)kSortTile);
    if (valid == kSortTile)
        onesweepTile<FIRST, true>(sm, keysIn, valsIn, keysOut, valsOut, tile, valid, shift, digitBase, lookback, epoch);
    else
        onesweepTile<FIRST, false>(sm, keysIn, valsIn, keysOut, valsOut, tile, valid, shift, digitBase, lookback, epoch);
}

cs_status enqueueSortReset(cs_context* ctx, cudaStream_t s)
{
    CS_CUDA(ctx, cudaMemsetAsync(ctx->sortHist, 0, (kSortPasses * kRadix + 64) * sizeof(u32), s));
    return CS_OK;
}

cs_status enqueueSort(cs_context* ctx, u64* keys, u32* perm, u64 n, bool histReady, cudaStream_t s)
{
    StageTimer t(ctx, CS_STAGE_SORT, s);
    if (n == 0) return CS_OK;
    static bool attrSet = false;
    if (!attrSet) {
        CS_CUDA(ctx, cudaFuncSetAttribute(onesweepKernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)sizeof(SortSmem)));
        CS_CUDA(ctx, cudaFuncSetAttribute(onesweepKernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)sizeof(SortSmem)));
        attrSet = true;
    }
    {
        StageTimer th(ctx, CS_STAGE_SORT_HIST, s);
        if (!histReady) {
            CS_TRY(enqueueSortReset(ctx, s));
            u32 grid = (u32)ctx->numSMs * 4;
            u32 need = divUp((n + 1) / 2, kHistBlock);
            if (need < grid) grid = need ? need : 1;
            sortHistKernel<<<grid, kHistBlock, 0, s>>>(keys, n, ctx->sortHist);
            CS_LAUNCH_CHECK(ctx, "sortHistKernel");
        }
        sortScanHistKernel<<<1, kRadix, 0, s>>>(ctx->sortHist);
        CS_LAUNCH_CHECK(ctx, "sortScanHistKernel");
    }
    StageTimer tp(ctx, CS_STAGE_SORT_PASSES, s);
    const u32 tiles = divUp(n, kSortTile);
    u64* kbuf[2] = {keys, ctx->keysAlt};
    u32* vbuf[2] = {perm, ctx->permAlt};
    for (int p = 0; p < kSortPasses; ++p) {
        const u32 epoch = nextEpoch(ctx, s);
        const int in = p & 1, out = in ^ 1;
        if (p == 0)
            onesweepKernel<true><<<tiles, kSortBlock, sizeof(SortSmem), s>>>(
                kbuf[in], nullptr, kbuf[out], vbuf[out], (u32)n, p * kRadixBits, ctx->sortHist + p * kRadix,
                ctx->sortTickets + p, ctx->sortLookback, epoch);
        else
            onesweepKernel<false><<<tiles, kSortBlock, sizeof(SortSmem), s>>>(
                kbuf[in], vbuf[in], kbuf[out], vbuf[out], (u32)n, p * kRadixBits, ctx->sortHist + p * kRadix,
                ctx->sortTickets + p, ctx->sortLookback, epoch);
        CS_LAUNCH_CHECK(ctx, "onesweepKernel");
    }
    return CS_OK;
}

}  // namespace cs
