// H3: stable LSD radix sort of (u64 key, u32 index) pairs -- PAPER.md:70, 168; A5.
//
// "Onesweep" organisation: one histogram pass over the keys gives the global digit counts of
// all passes; every pass then reads each element once and writes it once.  63 key bits = 7
// digits of 9 bits.  A pass tile is ranked inside the CTA (warp-level ballot matching + per-warp
// digit counters), the tile's position in each digit's output run comes from a decoupled
// look-back over the preceding tiles' digit counts (one thread per digit, all 512 threads of the
// CTA), and the tile is written out through shared memory so that each digit's run is a
// contiguous burst.  Tiles take their index from an atomic ticket, so a tile only ever waits
// for tiles that are already running (forward progress); the CTAs are persistent.
//
// Short cut: SFC keys of N particles are all but decided by their leading
// digits.  The default path sorts by the 5 leading digits (bits 18..62) with 5 passes and then
// orders the low 18 bits inside every run of equal leading digits directly (sortFixupKernel:
// rank = elements of the run that must precede, counted by scanning the run, O(run length) per
// element).  A run longer than kFixupMaxRun + 1 raises a device flag instead; the 7 plain passes
// that follow in the stream are gated on that flag and redo the sort from the (still complete)
// output of pass 5.  Either way the result is the stable sort: parity does not depend on the path.
//
// Model bytes per particle (SURVEY 8d, 8 passes of 8 bits): 196; moved by the default path:
// pass 0 (8 read, 12 written) + 4 x 24 + fix-up 24 = 140 (histograms come from the key kernel).
#include "cs_device.cuh"

namespace cs {

constexpr int kHistBlock = 512;
constexpr int kSortWarps = kSortBlock / 32;
static_assert(kSortBlock >= kRadix, "one thread per digit in the per-digit phases of a radix pass");
static_assert(kSortItems * 32 < 65536 && kSortTile < 65536, "16-bit per-warp digit counters and tile-local slots");

__device__ __forceinline__ u32 digitOf(u64 key, int shift) { return (u32)(key >> shift) & (kRadix - 1); }

// ---- global digit histograms of all passes ----------------------------------------------------
// copyTo (nullable): the keys are also copied there (the buffer the first pass reads, see sortSource)
__global__ void __launch_bounds__(kHistBlock) sortHistKernel(const u64* __restrict__ keys, u64 n, u32* gHist,
                                                             u64* __restrict__ copyTo)
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
            if (copyTo) {
                stStreamU2(copyTo + 2 * i, a.x, a.y);
                stStreamU2(copyTo + 2 * (i + nthreads), b.x, b.y);
                stStreamU2(copyTo + 2 * (i + 2 * nthreads), c.x, c.y);
                stStreamU2(copyTo + 2 * (i + 3 * nthreads), d.x, d.y);
            }
        }
        for (; i < pairs; i += nthreads) {
            ulonglong2 a = ldStreamU2(keys + 2 * i);
            add(a.x); add(a.y);
            if (copyTo) stStreamU2(copyTo + 2 * i, a.x, a.y);
        }
        if ((n & 1) && tid == 0) {
            add(keys[n - 1]);
            if (copyTo) copyTo[n - 1] = keys[n - 1];
        }
    } else {
        for (u64 i = tid; i < n; i += nthreads) {
            const u64 k = ldStreamU64(keys + i);
            add(k);
            if (copyTo) copyTo[i] = k;
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < kSortPasses * kRadix; i += kHistBlock) {
        u32 v = sh[i];
        if (v) atomicAdd(&gHist[i], v);
    }
}

// exclusive scan of each pass's digit counts, in place (one CTA)
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
    u64 keys[kSortTile];                           // tile in digit order
    u32 vals[kSortTile];
    unsigned short warpHist[kSortWarps][kRadix];   // per-warp digit counts, then first tile-local slot of (warp, digit)
    u32 globalBase[kRadix];                        // global slot of (digit d, tile-local slot i) = globalBase[d] + i
    u32 warpSums[kSortWarps + 1];
    u32 tile;
};

#ifndef CS_SORT_LOOKBATCH
#define CS_SORT_LOOKBATCH 4
#endif
constexpr int kLookBatch = CS_SORT_LOOKBATCH;   // predecessors fetched per look-back round trip

// Exclusive prefix of counter c over tiles < tile (tile > 0).  The words of kLookBatch predecessors
// are requested together, so one memory round trip covers kLookBatch tiles.  Tile 0 always holds a
// prefix word, so indices clamped to 0 are never summed twice.
__device__ __forceinline__ u32 lookBackBatched(const u64* state, u32 c, u32 tile, u32 epoch)
{
    const u32 want = epoch & 0x3FFFFFFFu;
    u32 excl = 0;
    int p = (int)tile - 1;
    for (;;) {
        u64 w[kLookBatch];
#pragma unroll
        for (int i = 0; i < kLookBatch; ++i) w[i] = lbLoad(state + (size_t)max(p - i, 0) * kRadix + c);
#pragma unroll
        for (int i = 0; i < kLookBatch; ++i) {
            u64 x = w[i];
            while ((u32)(x >> 34) != want) {
                __nanosleep(32);
                x = lbLoad(state + (size_t)max(p - i, 0) * kRadix + c);
            }
            excl += (u32)x;
            if (((u32)(x >> 32) & 3u) == kLbPrefix) return excl;
        }
        p -= kLookBatch;
    }
}

// Lanes of the warp whose digit equals this lane's: one ballot per digit bit (the native match.any is far
// slower).  Per bit: p = bit set, v = ballot(p); a &= v where p, o |= v where !p; peers = a & ~o.
// SASS per bit: VOTE + 2 predicated LOP3; the predicates of 7 bits come from one R2P.
__device__ __forceinline__ u32 matchDigit(u32 d)
{
    u32 a = kFull, o = 0;
#pragma unroll
    for (int b = 0; b < kRadixBits; ++b) {
        asm("{\n\t"
            ".reg .pred p;\n\t"
            ".reg .b32 t, v;\n\t"
            "and.b32 t, %2, %3;\n\t"
            "setp.ne.u32 p, t, 0;\n\t"
            "vote.sync.ballot.b32 v, p, 0xffffffff;\n\t"
            "@p and.b32 %0, %0, v;\n\t"
            "@!p or.b32 %1, %1, v;\n\t"
            "}"
            : "+r"(a), "+r"(o)
            : "r"(d), "r"(1u << b));
    }
    return a & ~o;
}

// keys of one tile: warp-striped, so that (warp, item, lane) order == memory order (stability); pads sort last
template <bool FULL>
__device__ __forceinline__ void tileLoadKeys(u64 (&key)[kSortItems], const u64* __restrict__ keysIn, u32 tile, u32 valid)
{
    const u32 warpOff = (threadIdx.x >> 5) * (32 * kSortItems) + laneId();
    const u64* src = keysIn + (u64)tile * kSortTile + warpOff;
#pragma unroll
    for (int j = 0; j < kSortItems; ++j)
        key[j] = (FULL || warpOff + j * 32 < valid) ? ldStreamU64(src + j * 32) : ~0ull;
}

// From the loaded keys to the tile staged in digit order in shared memory, with globalBase[] set
// (ranking, per-digit prefixes, scatter of keys and values, look-back).  Ends with a barrier.
template <int SHIFT, bool FIRST, bool FULL>
__device__ __forceinline__ void tileStage(SortSmem& sm, u64 (&key)[kSortItems], const u32* __restrict__ valsIn, u32 tile,
                                          u32 valid, const u32* __restrict__ digitBase, u64* lookback, u32 epoch)
{
    const u32 tid = threadIdx.x, lane = laneId(), warp = tid >> 5;
    const u64 base = (u64)tile * kSortTile;
    const u32 warpOff = warp * (32 * kSortItems) + lane;

    // ---- rank inside the warp: every peer reads the warp's running count of its digit (a
    // shared-memory broadcast) and the lowest peer bumps it once ------------------------------------
    u32 rankPk[(kSortItems + 1) / 2];                                        // two 16-bit ranks per register
#pragma unroll
    for (int j = 0; j < (kSortItems + 1) / 2; ++j) rankPk[j] = 0;
    unsigned short* wh = sm.warpHist[warp];
    const u32 lt = laneMaskLt();
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
        const u32 d = digitOf(key[j], SHIFT);
        const u32 peers = matchDigit(d);
        const u32 lower = __popc(peers & lt);
        const u32 prev = wh[d];
        __syncwarp();
        if (lower == 0) wh[d] = (unsigned short)(prev + __popc(peers));
        __syncwarp();
        rankPk[j >> 1] |= (prev + lower) << ((j & 1) * 16);
    }
    // values: requested now, used after the key scatter (their latency hides behind the per-digit phase);
    // the first pass synthesises the identity permutation instead of reading it
    u32 val[kSortItems];
    {
        const u32* vsrc = valsIn + base + warpOff;
#pragma unroll
        for (int j = 0; j < kSortItems; ++j) {
            if (FIRST) val[j] = (u32)base + warpOff + j * 32;
            else val[j] = (FULL || warpOff + j * 32 < valid) ? ldStreamU32(vsrc + j * 32) : 0u;
        }
    }
    __syncthreads();

    // ---- per digit (one thread each): tile count, tile-local start, first slot of every warp ------
    u32 count = 0;
    if (tid < kRadix) {
#pragma unroll
        for (int w = 0; w < kSortWarps; ++w) count += sm.warpHist[w][tid];
        // publish this tile's count at once: the tiles behind it can start their look-back
        const u32 real = (!FULL && tid == kRadix - 1) ? count - (kSortTile - valid) : count;   // pads are not elements
        lbStore(lookback + (size_t)tile * kRadix + tid, lbPack(epoch, tile == 0 ? kLbPrefix : kLbAggregate, real));
    }
    u32 total;
    const u32 start = blockExclusiveScan<kSortBlock>(count, sm.warpSums, &total);
    if (tid < kRadix) {
        u32 run = start;
#pragma unroll
        for (int w = 0; w < kSortWarps; ++w) {
            const u32 c = sm.warpHist[w][tid];
            sm.warpHist[w][tid] = (unsigned short)run;
            run += c;
        }
    }
    __syncthreads();

    // ---- scatter keys, then values, into digit order in shared memory -----------------------------
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
        const u32 d = digitOf(key[j], SHIFT);
        const u32 r = (rankPk[j >> 1] >> ((j & 1) * 16)) & 0xFFFFu;
        const u32 pos = wh[d] + r;
        sm.keys[pos] = key[j];
        if (j & 1) rankPk[j >> 1] = (rankPk[j >> 1] & 0xFFFFu) | (pos << 16);
        else rankPk[j >> 1] = (rankPk[j >> 1] & 0xFFFF0000u) | pos;
    }
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) sm.vals[(rankPk[j >> 1] >> ((j & 1) * 16)) & 0xFFFFu] = val[j];

    // ---- decoupled look-back, after the shared-memory scatter: the predecessors have had that much
    // longer to publish their prefixes ---------------------------------------------------------------
    if (tid < kRadix) {
        u32 excl = 0;
        if (tile != 0) {
            const u32 real = (!FULL && tid == kRadix - 1) ? count - (kSortTile - valid) : count;
            excl = lookBackBatched(lookback, tid, tile, epoch);
            lbStore(lookback + (size_t)tile * kRadix + tid, lbPack(epoch, kLbPrefix, excl + real));
        }
        sm.globalBase[tid] = digitBase[tid] + excl - start;
    }
    __syncthreads();

}

// write out: consecutive threads -> consecutive slots of a digit's run
template <int SHIFT, bool FULL>
__device__ __forceinline__ void tileWriteOut(const SortSmem& sm, u64* __restrict__ keysOut, u32* __restrict__ valsOut, u32 valid)
{
    const u32 tid = threadIdx.x;
#pragma unroll
    for (int k = 0; k < kSortItems; ++k) {
        const u32 i = tid + k * kSortBlock;
        if (FULL || i < valid) {
            const u64 kk = sm.keys[i];
            const u32 dst = sm.globalBase[digitOf(kk, SHIFT)] + i;
            keysOut[dst] = kk;
            valsOut[dst] = sm.vals[i];
        }
    }
}

template <int SHIFT, bool FIRST, bool FULL>
__device__ __forceinline__ void onesweepTile(SortSmem& sm, const u64* __restrict__ keysIn, const u32* __restrict__ valsIn,
                                             u64* __restrict__ keysOut, u32* __restrict__ valsOut, u32 tile, u32 valid,
                                             const u32* __restrict__ digitBase, u64* lookback, u32 epoch)
{
    u64 key[kSortItems];
    tileLoadKeys<FULL>(key, keysIn, tile, valid);
    tileStage<SHIFT, FIRST, FULL>(sm, key, valsIn, tile, valid, digitBase, lookback, epoch);
    tileWriteOut<SHIFT, FULL>(sm, keysOut, valsOut, valid);
}

// One tile per CTA (grid = tiles): the passes of the default path and of cs_setSortMode(PLAIN).
template <int SHIFT, bool FIRST>
__global__ void __launch_bounds__(kSortBlock, kSortMinBlocks)
    onesweepKernel(const u64* __restrict__ keysIn, const u32* __restrict__ valsIn, u64* __restrict__ keysOut,
                   u32* __restrict__ valsOut, u32 n, const u32* __restrict__ digitBase /*scanned hist*/, u32* ticket,
                   u64* lookback, u32 epoch)
{
    extern __shared__ __align__(16) unsigned char smemRaw[];
    SortSmem& sm = *reinterpret_cast<SortSmem*>(smemRaw);
    const u32 tid = threadIdx.x;
    if (tid == 0) sm.tile = atomicAdd(ticket, 1u);
    u32* whWords = reinterpret_cast<u32*>(&sm.warpHist[0][0]);
    for (int i = tid; i < kSortWarps * kRadix / 2; i += kSortBlock) whWords[i] = 0;
    __syncthreads();
    const u32 tile = sm.tile;
    const u64 base = (u64)tile * kSortTile;
    const u32 valid = (u32)((n - base) < (u64)kSortTile ? (n - base) : (u64)kSortTile);
    if (valid == kSortTile)
        onesweepTile<SHIFT, FIRST, true>(sm, keysIn, valsIn, keysOut, valsOut, tile, valid, digitBase, lookback, epoch);
    else
        onesweepTile<SHIFT, FIRST, false>(sm, keysIn, valsIn, keysOut, valsOut, tile, valid, digitBase, lookback, epoch);
}

// The redo passes behind the fix-up: persistent CTAs that leave at once unless *gate != 0, so that
// the default path pays a few microseconds for them, not a wave of empty CTAs per pass.
template <int SHIFT>
__global__ void __launch_bounds__(kSortBlock, kSortMinBlocks)
    onesweepGatedKernel(const u64* __restrict__ keysIn, const u32* __restrict__ valsIn, u64* __restrict__ keysOut,
                        u32* __restrict__ valsOut, u32 n, const u32* __restrict__ digitBase, u32* ticket, u64* lookback,
                        u32 epoch, const u32* gate)
{
    extern __shared__ __align__(16) unsigned char smemRaw[];
    SortSmem& sm = *reinterpret_cast<SortSmem*>(smemRaw);
    const u32 tid = threadIdx.x;
    if (*reinterpret_cast<const volatile u32*>(gate) == 0) return;
    const u32 tiles = (n + kSortTile - 1) / kSortTile;
    u32* whWords = reinterpret_cast<u32*>(&sm.warpHist[0][0]);
    for (;;) {
        __syncthreads();                                   // the previous tile is written out
        if (tid == 0) sm.tile = atomicAdd(ticket, 1u);
        for (int i = tid; i < kSortWarps * kRadix / 2; i += kSortBlock) whWords[i] = 0;
        __syncthreads();
        const u32 tile = sm.tile;
        if (tile >= tiles) break;
        const u64 base = (u64)tile * kSortTile;
        const u32 valid = (u32)((n - base) < (u64)kSortTile ? (n - base) : (u64)kSortTile);
        if (valid == kSortTile)
            onesweepTile<SHIFT, false, true>(sm, keysIn, valsIn, keysOut, valsOut, tile, valid, digitBase, lookback, epoch);
        else
            onesweepTile<SHIFT, false, false>(sm, keysIn, valsIn, keysOut, valsOut, tile, valid, digitBase, lookback, epoch);
    }
}

// ---- fix-up of the low bits inside runs of equal leading digits ----------------------------------------
// In: elements stably sorted by key >> LOW.  Out: stably sorted by the whole key.  An element moves
// inside its run only: to runStart + (elements of the run with smaller low bits) + (elements of the run
// before it with equal low bits).  Neighbours are read through L1 (the lines were just loaded by the
// adjacent threads).  Runs longer than kFixupMaxRun + 1: *redo = 1 and the kernel gives up.
constexpr int kFixupBlock = 256;
constexpr u32 kFixupMaxRun = 256;

template <int LOW>
__global__ void __launch_bounds__(kFixupBlock)
    sortFixupKernel(const u64* __restrict__ keysIn, const u32* __restrict__ valsIn, u64* __restrict__ keysOut,
                    u32* __restrict__ valsOut, u32 n, u32* redo)
{
    const u32 stride = gridDim.x * kFixupBlock;
    u32 it = 0;
    for (u32 i = blockIdx.x * kFixupBlock + threadIdx.x; i < n; i += stride, ++it) {
        const u64 key = keysIn[i];
        const u32 val = ldStreamU32(valsIn + i);
        // same run <=> the keys agree above bit LOW; inside a run the key order is the order of the low bits
        const u64 kl = keysIn[i > 0 ? i - 1 : 0], kr = keysIn[i + 1 < n ? i + 1 : i];
        const bool runL = i > 0 && ((kl ^ key) >> LOW) == 0, runR = i + 1 < n && ((kr ^ key) >> LOW) == 0;
        u32 dst = i;
        if (runL || runR) {                                 // not alone in its run: count what precedes it
            // The input is ordered by the leading bits, so the run [a, e) is where runLo <= k < runHi.  Its
            // ends are found by doubling steps + bisection (all lanes of a run walk the same addresses).
            const u64 runLo = key & ~((1ull << LOW) - 1), runHi = runLo + (1ull << LOW);
            u32 a = i, e = i + 1;
            if (runL) {
                u32 d = 2;                                  // keysIn[i - 1] is inside
                while (d <= i && d <= 2 * kFixupMaxRun && keysIn[i - d] >= runLo) d *= 2;
                u32 lo = d <= i ? i - d + 1 : 0, hi = i - d / 2;   // keysIn[hi] inside; first inside index in [lo, hi]
                if (d <= i && d > 2 * kFixupMaxRun) lo = hi;      // beyond the limit anyway
                while (lo < hi) {
                    const u32 mid = lo + ((hi - lo) >> 1);
                    if (keysIn[mid] >= runLo) hi = mid;
                    else lo = mid + 1;
                }
                a = lo;
            }
            if (runR) {
                u32 d = 2;                                  // keysIn[i + 1] is inside
                while (d < n - i && d <= 2 * kFixupMaxRun && keysIn[i + d] < runHi) d *= 2;
                u32 lo = i + d / 2 + 1, hi = d < n - i ? i + d : n;   // keysIn[lo - 1] inside; first outside index in [lo, hi]
                if (d < n - i && d > 2 * kFixupMaxRun) hi = lo;
                while (lo < hi) {
                    const u32 mid = lo + ((hi - lo) >> 1);
                    if (keysIn[mid] < runHi) lo = mid + 1;
                    else hi = mid;
                }
                e = lo;
            }
            if (i - a > kFixupMaxRun || e - i - 1 > kFixupMaxRun) {   // longer than the limit: the gated passes redo the sort
                *reinterpret_cast<volatile u32*>(redo) = 1u;
                return;
            }
            // inside the run the leading bits agree, so the low words order it; ties keep their input order
            const u32* lowWord = reinterpret_cast<const u32*>(keysIn);
            const u32 mine = (u32)key;
            u32 before = 0;
            for (u32 m = a; m < e; ++m) {
                const u32 w = lowWord[2 * (size_t)m];
                before += (w < mine) || (w == mine && m < i);
            }
            dst = a + before;
        }
        keysOut[dst] = key;
        valsOut[dst] = val;
        // now and then: no point in finishing once another thread has given up
        if ((it & 15u) == 15u && *reinterpret_cast<const volatile u32*>(redo)) return;
    }
}

cs_status enqueueSortReset(cs_context* ctx, cudaStream_t s)
{
    CS_CUDA(ctx, cudaMemsetAsync(ctx->sortHist, 0, (kSortPasses * kRadix + 64) * sizeof(u32), s));
    return CS_OK;
}

constexpr int kTopPasses = 5;                               // digits 2..6 (bits 18..62) before the fix-up
constexpr int kFixupLow = (kSortPasses - kTopPasses) * kRadixBits;
static_assert(kSortPasses == 7 && kRadixBits == 9, "the pass plan below is written for 7 digits of 9 bits");

struct PassPlan {
    u64* k[2];
    u32* v[2];
    int cur;                                                // buffers holding the current order
    u32 n, tiles;
    int ticketSlot;
};

template <int SHIFT, bool FIRST>
static cs_status launchPass(cs_context* ctx, PassPlan& pl, cudaStream_t s)
{
    static bool attrSet = false;
    if (!attrSet) {
        CS_CUDA(ctx, cudaFuncSetAttribute(onesweepKernel<SHIFT, FIRST>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)sizeof(SortSmem)));
        attrSet = true;
    }
    const u32 epoch = nextEpoch(ctx, s);
    const int in = pl.cur, out = in ^ 1;
    onesweepKernel<SHIFT, FIRST><<<pl.tiles, kSortBlock, sizeof(SortSmem), s>>>(
        pl.k[in], FIRST ? nullptr : pl.v[in], pl.k[out], pl.v[out], pl.n, ctx->sortHist + (SHIFT / kRadixBits) * kRadix,
        ctx->sortTickets + pl.ticketSlot++, ctx->sortLookback, epoch);
    CS_LAUNCH_CHECK(ctx, "onesweepKernel");
    pl.cur = out;
    return CS_OK;
}

template <int SHIFT>
static cs_status launchGatedPass(cs_context* ctx, PassPlan& pl, const u32* gate, cudaStream_t s)
{
    static bool attrSet = false;
    if (!attrSet) {
        CS_CUDA(ctx, cudaFuncSetAttribute(onesweepGatedKernel<SHIFT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)sizeof(SortSmem)));
        attrSet = true;
    }
    const u32 epoch = nextEpoch(ctx, s);
    const int in = pl.cur, out = in ^ 1;
    const u32 resident = (u32)ctx->numSMs * kSortMinBlocks;
    onesweepGatedKernel<SHIFT><<<pl.tiles < resident ? pl.tiles : resident, kSortBlock, sizeof(SortSmem), s>>>(
        pl.k[in], pl.v[in], pl.k[out], pl.v[out], pl.n, ctx->sortHist + (SHIFT / kRadixBits) * kRadix,
        ctx->sortTickets + pl.ticketSlot++, ctx->sortLookback, epoch, gate);
    CS_LAUNCH_CHECK(ctx, "onesweepGatedKernel");
    pl.cur = out;
    return CS_OK;
}

// Where the first radix pass reads the unsorted keys.  The passes alternate between the caller's
// arrays and the workspace's: the default path (5 passes + fix-up, and 7 more if redone) ends where
// it started; the plain 7 passes end in the other pair.
u64* sortSource(cs_context* ctx, u64* keys) { return ctx->sortPlain ? ctx->keysAlt : keys; }

// fused: the unsorted keys already lie in sortSource(ctx, keys) and ctx->sortHist holds their digit counts
// (cs_buildOctree: the key kernel wrote both); otherwise they are in `keys`.
cs_status enqueueSort(cs_context* ctx, u64* keys, u32* perm, u64 n, bool fused, cudaStream_t s)
{
    StageTimer t(ctx, CS_STAGE_SORT, s);
    if (n == 0) return CS_OK;
    u64* first = sortSource(ctx, keys);
    {
        StageTimer th(ctx, CS_STAGE_SORT_HIST, s);
        if (!fused) {
            CS_TRY(enqueueSortReset(ctx, s));
            u32 grid = (u32)ctx->numSMs * 4;
            u32 need = divUp((n + 1) / 2, kHistBlock);
            if (need < grid) grid = need ? need : 1;
            sortHistKernel<<<grid, kHistBlock, 0, s>>>(keys, n, ctx->sortHist, first == keys ? nullptr : first);
            CS_LAUNCH_CHECK(ctx, "sortHistKernel");
        }
        sortScanHistKernel<<<1, kRadix, 0, s>>>(ctx->sortHist);
        CS_LAUNCH_CHECK(ctx, "sortScanHistKernel");
    }
    ctx->evUsed[CS_STAGE_SORT_FIXUP] = false;
    PassPlan pl;
    const bool own = first == keys;
    pl.k[0] = first; pl.k[1] = own ? ctx->keysAlt : keys;
    pl.v[0] = own ? perm : ctx->permAlt; pl.v[1] = own ? ctx->permAlt : perm;
    pl.cur = 0;
    pl.n = (u32)n;
    pl.tiles = divUp(n, kSortTile);
    pl.ticketSlot = 0;
    if (ctx->sortPlain) {                                   // all 7 digits, least significant first
        StageTimer tp(ctx, CS_STAGE_SORT_PASSES, s);
        CS_TRY((launchPass<0, true>(ctx, pl, s)));
        CS_TRY((launchPass<9, false>(ctx, pl, s)));
        CS_TRY((launchPass<18, false>(ctx, pl, s)));
        CS_TRY((launchPass<27, false>(ctx, pl, s)));
        CS_TRY((launchPass<36, false>(ctx, pl, s)));
        CS_TRY((launchPass<45, false>(ctx, pl, s)));
        return launchPass<54, false>(ctx, pl, s);
    }
    {   // leading digits, most of the order
        StageTimer tp(ctx, CS_STAGE_SORT_PASSES, s);
        CS_TRY((launchPass<18, true>(ctx, pl, s)));
        CS_TRY((launchPass<27, false>(ctx, pl, s)));
        CS_TRY((launchPass<36, false>(ctx, pl, s)));
        CS_TRY((launchPass<45, false>(ctx, pl, s)));
        CS_TRY((launchPass<54, false>(ctx, pl, s)));
    }
    StageTimer tf(ctx, CS_STAGE_SORT_FIXUP, s);
    // low bits inside the runs; out of place, so the input stays intact for a redo
    u32* redo = ctx->sortTickets + kSortRedoSlot;
    {
        u32 grid = divUp(n, kFixupBlock);
        const u32 cap = (u32)ctx->numSMs * 32;
        if (grid > cap) grid = cap;
        const int in = pl.cur, out = in ^ 1;
        sortFixupKernel<kFixupLow><<<grid, kFixupBlock, 0, s>>>(pl.k[in], pl.v[in], pl.k[out], pl.v[out], pl.n, redo);
        CS_LAUNCH_CHECK(ctx, "sortFixupKernel");
    }
    // gated redo from the output of the fifth pass (pl.cur still names it): 7 passes end in the other pair,
    // which is where the fix-up wrote
    CS_TRY((launchGatedPass<0>(ctx, pl, redo, s)));
    CS_TRY((launchGatedPass<9>(ctx, pl, redo, s)));
    CS_TRY((launchGatedPass<18>(ctx, pl, redo, s)));
    CS_TRY((launchGatedPass<27>(ctx, pl, redo, s)));
    CS_TRY((launchGatedPass<36>(ctx, pl, redo, s)));
    CS_TRY((launchGatedPass<45>(ctx, pl, redo, s)));
    return launchGatedPass<54>(ctx, pl, redo, s);
}

}  // namespace cs
