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
// orders the low 18 bits inside every run of equal leading digits directly, in the shared-memory
// stage of the fifth pass (onesweepLastKernel: rank = elements of the run that must precede,
// counted by scanning the run, O(run length) per element).  A run longer than kFixupMaxRun + 1
// raises a device flag instead; the 7 plain passes that follow in the stream are gated on that
// flag and redo the sort from the (still complete) input of the fifth pass.  Either way the
// result is the stable sort: parity does not depend on the path.
//
// Model bytes per particle (SURVEY 8d, 8 passes of 8 bits): 196; moved by the default path:
// pass 0 (8 read, 12 written) + 4 x 24 = 116 (histograms come from the key kernel).
#include <cooperative_groups.h>

#include "cs_device.cuh"

namespace cg = cooperative_groups;

namespace cs {

constexpr int kHistBlock = 512;
constexpr int kSortWarps = kSortBlock / 32;
static_assert(kSortBlock >= kRadix, "one thread per digit in the per-digit phases of a radix pass");
static_assert(kSortItems * 32 < 65536 && kSortTile < 65536, "16-bit per-warp digit counters and tile-local slots");

__device__ __forceinline__ u32 digitOf(u64 key, int shift) { return (u32)(key >> shift) & (kRadix - 1); }
__device__ __forceinline__ u32 digitOf(u32 key, int shift) { return (key >> shift) & (kRadix - 1); }
__device__ __forceinline__ u64 ldStreamKey(const u64* p) { return ldStreamU64(p); }
__device__ __forceinline__ u32 ldStreamKey(const u32* p) { return ldStreamU32(p); }

// ---- global digit histograms of all passes ----------------------------------------------------
// copyTo (nullable): the keys are also copied there (the buffer the first pass reads, see sortSource)
// firstPass: digits below it are not counted (their counts stay zero: the default path does not sort by them)
__global__ void __launch_bounds__(kHistBlock) sortHistKernel(const u64* __restrict__ keys, u64 n, u32* gHist,
                                                             u64* __restrict__ copyTo, int firstPass)
{
    __shared__ u32 sh[kSortPasses * kRadix];
    for (int i = threadIdx.x; i < kSortPasses * kRadix; i += kHistBlock) sh[i] = 0;
    __syncthreads();
    const u64 tid = (u64)blockIdx.x * kHistBlock + threadIdx.x;
    const u64 nthreads = (u64)gridDim.x * kHistBlock;
    const bool vec = (((uintptr_t)keys) & 15u) == 0;
    auto add = [&](u64 k) {
#pragma unroll
        for (int p = 0; p < kSortPasses; ++p)
            if (p >= firstPass) atomicAdd(&sh[p * kRadix + digitOf(k, p * kRadixBits)], 1u);
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

// exclusive scan of each pass's digit counts, in place (one CTA per pass)
__global__ void __launch_bounds__(kRadix) sortScanHistKernel(u32* gHist)
{
    chainEnter();
    __shared__ u32 warpSums[kRadix / 32 + 1];
    const u32 i = blockIdx.x * kRadix + threadIdx.x;
    u32 total;
    gHist[i] = blockExclusiveScan<kRadix>(gHist[i], warpSums, &total);
}

// ---- one radix pass ------------------------------------------------------------------------------
#ifndef CS_SORT_PREFETCH
#define CS_SORT_PREFETCH 296
#endif
constexpr int kHistWords = kSortWarps * kRadix / 2;

template <typename KeyT>
struct SortSmemT {
    KeyT keys[kSortTile];                          // tile in digit order
    u32 vals[kSortTile];
    unsigned short warpHist[kSortWarps][kRadix];   // per-warp digit counts, then first tile-local slot of (warp, digit)
    u32 globalBase[kRadix];                        // global slot of (digit d, tile-local slot i) = globalBase[d] + i
    u32 warpSums[kSortWarps + 1];
    u32 tile;
};
typedef SortSmemT<u64> SortSmem;                   // 63-bit keys (L = 21); SortSmemT<u32>: 30-bit keys (L = 10)

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
template <bool FULL, typename KeyT>
__device__ __forceinline__ void tileLoadKeys(KeyT (&key)[kSortItems], const KeyT* __restrict__ keysIn, u64 base, u32 valid)
{
    const u32 warpOff = (threadIdx.x >> 5) * (32 * kSortItems) + laneId();
    const KeyT* src = keysIn + base + warpOff;
#pragma unroll
    for (int j = 0; j < kSortItems; ++j)
        key[j] = (FULL || warpOff + j * 32 < valid) ? ldStreamKey(src + j * 32) : (KeyT)~(KeyT)0;
}

// From the loaded keys to the tile staged in digit order in shared memory, with globalBase[] set
// (ranking, per-digit prefixes, scatter of keys and values, look-back).  Ends with a barrier.
template <int SHIFT, bool FIRST, bool FULL, typename KeyT, bool COLD = false>
__device__ __forceinline__ void tileStage(SortSmemT<KeyT>& sm, KeyT (&key)[kSortItems], const u32* __restrict__ valsIn, u32 tile,
                                          u64 base, u32 valid, const u32* __restrict__ digitBase, u64* lookback, u32 epoch)
{
    const u32 tid = threadIdx.x, lane = laneId(), warp = tid >> 5;
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
        const u32 peers = COLD ? __match_any_sync(kFull, d) : matchDigit(d);   // COLD: the redo path, where ptxas runs out of
                                                                                // predicates for the hand-written match
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
template <int SHIFT, bool FULL, typename KeyT>
__device__ __forceinline__ void tileWriteOut(const SortSmemT<KeyT>& sm, KeyT* __restrict__ keysOut, u32* __restrict__ valsOut, u32 valid)
{
    const u32 tid = threadIdx.x;
#pragma unroll
    for (int k = 0; k < kSortItems; ++k) {
        const u32 i = tid + k * kSortBlock;
        if (FULL || i < valid) {
            const KeyT kk = sm.keys[i];
            const u32 dst = sm.globalBase[digitOf(kk, SHIFT)] + i;
            keysOut[dst] = kk;
            valsOut[dst] = sm.vals[i];
        }
    }
}

template <int SHIFT, bool FIRST, bool FULL, typename KeyT, bool COLD = false>
__device__ __forceinline__ void onesweepTile(SortSmemT<KeyT>& sm, const KeyT* __restrict__ keysIn, const u32* __restrict__ valsIn,
                                             KeyT* __restrict__ keysOut, u32* __restrict__ valsOut, u32 tile, u32 valid,
                                             const u32* __restrict__ digitBase, u64* lookback, u32 epoch)
{
    KeyT key[kSortItems];
    const u64 base = (u64)tile * kSortTile;
    tileLoadKeys<FULL>(key, keysIn, base, valid);
    tileStage<SHIFT, FIRST, FULL, KeyT, COLD>(sm, key, valsIn, tile, base, valid, digitBase, lookback, epoch);
    tileWriteOut<SHIFT, FULL>(sm, keysOut, valsOut, valid);
}

// One tile per CTA (grid = tiles): the passes of the default path and of cs_setSortMode(PLAIN).
template <int SHIFT, bool FIRST, typename KeyT>
__global__ void __launch_bounds__(kSortBlock, kSortMinBlocks)
    onesweepKernel(const KeyT* __restrict__ keysIn, const u32* __restrict__ valsIn, KeyT* __restrict__ keysOut,
                   u32* __restrict__ valsOut, u32 n, const u32* __restrict__ digitBase /*scanned hist*/, u32* ticket,
                   u64* lookback, u32 epoch, const u32* __restrict__ epochBase)
{
    chainEnter();
    epoch += *epochBase;
    extern __shared__ __align__(16) unsigned char smemRaw[];
    SortSmemT<KeyT>& sm = *reinterpret_cast<SortSmemT<KeyT>*>(smemRaw);
    const u32 tid = threadIdx.x;
    u32* whWords = reinterpret_cast<u32*>(sm.warpHist);
    if (tid == 0) {
        const u32 t = atomicAdd(ticket, 1u);
        sm.tile = t;
#if CS_SORT_PREFETCH
        // the tile that a CTA will pick up one generation of resident CTAs from now: on its way into L2 already
        const u64 pb = ((u64)t + CS_SORT_PREFETCH) * kSortTile;
        if (pb < n) {
            const u32 cnt = (u32)((n - pb) < (u64)kSortTile ? (n - pb) : (u64)kSortTile);
            bulkPrefetchL2(keysIn + pb, (cnt * (u32)sizeof(KeyT)) & ~15u);
            if (!FIRST) bulkPrefetchL2(valsIn + pb, (cnt * 4u) & ~15u);
        }
#endif
    }
    for (int i = tid; i < kHistWords; i += kSortBlock) whWords[i] = 0;
    __syncthreads();
    const u32 tile = sm.tile;
    const u64 base = (u64)tile * kSortTile;
    const u32 valid = (u32)((n - base) < (u64)kSortTile ? (n - base) : (u64)kSortTile);
    if (valid == kSortTile)
        onesweepTile<SHIFT, FIRST, true>(sm, keysIn, valsIn, keysOut, valsOut, tile, valid, digitBase, lookback, epoch);
    else
        onesweepTile<SHIFT, FIRST, false>(sm, keysIn, valsIn, keysOut, valsOut, tile, valid, digitBase, lookback, epoch);
}

// ---- last pass of the default path: radix pass over the top digit + fix-up of the low bits ---------------
// Input: stably sorted by bits LOW..53.  After this pass's stable split by the top digit the elements
// are sorted by all bits >= LOW; what is left is the order of the low bits inside every run of equal
// leading bits.  The elements of such a run are adjacent in the input's order within one top digit, so if
// no run straddles a tile, every run lies contiguous in the tile staged in shared memory and can be
// ordered there, on the way out.  Hence the tiles are cut between groups of elements that agree in the
// bits LOW..53 (the input's order; a run is part of one group): nominal boundaries every kLastTile
// elements, each moved back to the start of the group it falls into (at most kFixupMaxRun elements).  An element of a run goes to runStart + (run elements with smaller low bits) + (earlier run
// elements with equal low bits).  A run longer than kFixupMaxRun + 1 raises *redo instead (the gated passes
// that follow redo the sort from this pass's input).
constexpr u32 kFixupMaxRun = 256;
constexpr u32 kLastTile = kSortLastTile;                  // nominal tile: room for a boundary run, multiple of 64
static_assert(kLastTile % 64 == 0 && kLastTile > 2 * kFixupMaxRun, "nominal tile of the last pass");

// Where to cut the input at or before element `b` (0 < b < n) so that no run is split: the input is ordered
// by the bits LOW .. TOP-1 only, so the members of a run (equal bits >= LOW) need not be neighbours there; the
// elements that agree in the bits LOW .. TOP-1 are (a "group": every run lies inside one).  Returns the start
// of the group of element b, found by one warp.  *tooLong is set if it starts more than kFixupMaxRun elements
// before b (then b itself is returned).
template <int LOW, int TOP>
__device__ __forceinline__ u32 groupStartBefore(const u64* __restrict__ keysIn, u32 b, bool* tooLong)
{
    constexpr u64 kGroupBits = ((1ull << TOP) - 1) & ~((1ull << LOW) - 1);
    const u32 lane = laneId();
    const u64 kb = keysIn[b];
    u32 back = 0;
    for (;;) {
        const u32 off = back + lane + 1;                    // element b - off
        const bool same = off <= b && ((keysIn[b - (off <= b ? off : 0)] ^ kb) & kGroupBits) == 0;
        const u32 m = __ballot_sync(kFull, same);
        const u32 c = m == kFull ? 32u : (u32)__ffs((int)~m) - 1u;   // lanes 0..c-1 are in the group
        back += c;
        if (c < 32) break;
        if (back > kFixupMaxRun) break;
    }
    if (back > kFixupMaxRun) {
        *tooLong = true;
        return b;
    }
    return b - back;
}

// Write out with the fix-up.  The staged tile is ordered by the bits >= LOW, so a run (equal bits >= LOW) is a
// contiguous range of slots; "head" = first slot of a run.  First every thread marks the heads among its slots
// into a bit mask in shared memory (headMask, bit i <-> slot i; the slots from `valid` on count as heads).  Then,
// as in the plain write-out, consecutive lanes take consecutive slots, 32 slots (one mask word) per warp step.
// A lane finds its run [runStart, runEnd) from the mask words (nearest head at or below it, nearest head above it; a
// word of heads only goes straight out) and counts the members that must precede it by reading the run's low words
// from shared memory: slot of an element = run start + (members with smaller low bits) + (earlier members with equal
// low bits); it is stored straight to its place in the output.  (Counting with shuffles inside the 32 slots plus
// shared-memory loops for the parts outside measured 1.6 % slower.)  A run longer than kFixupMaxRun + 1 raises *redo
// instead.
constexpr int kHeadWords = kSortTile / 32 + 2 + (kFixupMaxRun + 64) / 32;   // + sentinels past the tile

template <int SHIFT, int LOW>
__device__ __forceinline__ void tileWriteOutFixup(const SortSmem& sm, u32* headMask, u64* __restrict__ keysOut,
                                                  u32* __restrict__ valsOut, u32 valid, u32* redo)
{
    const u32 tid = threadIdx.x, lane = laneId();
    const u64* keys = sm.keys;
    const u32* low = reinterpret_cast<const u32*>(sm.keys);
    // ---- head bits: consecutive threads <-> consecutive slots, one ballot per 32 slots -----------------
    bool someRun = false;                                    // a slot that is not a head: a run of two or more elements
#pragma unroll
    for (int k = 0; k < kSortItems; ++k) {
        const u32 i = tid + k * kSortBlock;
        const bool head = i == 0 || i >= valid || ((keys[i - (i ? 1 : 0)] ^ keys[i]) >> LOW) != 0;
        const u32 H = __ballot_sync(kFull, head);
        if (lane == 0) headMask[i >> 5] = H;
        someRun |= H != kFull;
    }
    if (tid < kHeadWords - kSortTile / 32) headMask[kSortTile / 32 + tid] = kFull;
    if (!__syncthreads_or(someRun)) {                        // every element is alone in its run (most tiles of most inputs):
        tileWriteOut<SHIFT, false>(sm, keysOut, valsOut, valid);   // the stable split has put it in place already
        return;
    }
    bool tooLong = false;
#pragma unroll 1
    for (int k = 0; k < kSortItems; ++k) {
        const u32 i = tid + k * kSortBlock;
        const u32 cb = i - lane;                             // first of the warp's 32 slots
        if (cb >= valid) break;                              // warp-uniform
        const u32 H = headMask[i >> 5];
        const bool act = i < valid;
        const u32 mine = low[2 * (act ? i : cb)];
        const u64 mineKey = keys[act ? i : cb];             // LOW > 32: the low word does not hold all the low bits
        const u32 dstBase = sm.globalBase[digitOf(keys[act ? i : cb], SHIFT)];
        u32 slot = i;
        if (H != kFull || !(headMask[(i >> 5) + 1] & 1u)) {  // not heads only, or the last slot's run goes on behind them
            // this lane's run [runStart, runEnd): the nearest head at or below it and the nearest head above it
            const u32 below = H & (kFull >> (31u - lane));
            const u32 above = (H >> 1) >> lane;              // bit 0 <-> lane + 1
            u32 runStart = cb + 31u - (u32)__clz((int)below), runEnd = i + (u32)__ffs((int)above);
            if (!below) {                                    // it began before these 32 slots (cb > 0: slot 0 is a head)
                u32 w = (cb - 1u) >> 5, bits = headMask[w], steps = 0;
                while (!bits && steps <= kFixupMaxRun / 32) { bits = headMask[--w]; ++steps; }
                runStart = (w << 5) + 31u - (u32)__clz((int)bits);
                if (!bits) runStart = 0, tooLong = act;
            }
            if (!above) {                                    // it goes on behind them (sentinel words end every run)
                u32 w = (cb >> 5) + 1u, bits = headMask[w], steps = 0;
                while (!bits && steps <= kFixupMaxRun / 32) { bits = headMask[++w]; ++steps; }
                runEnd = (w << 5) + (u32)__ffs((int)bits) - 1u;
                if (!bits) runEnd = runStart, tooLong = act;
            }
            if (runEnd - runStart > kFixupMaxRun + 1u) {     // beyond the limit: the redo sorts it all
                if (act) tooLong = true;
                runEnd = runStart;
            }
            u32 before = 0;                                  // members that precede: smaller low bits, or equal and earlier
            if (act) {
                if constexpr (LOW <= 32) {
                    for (u32 m = runStart; m < runEnd; ++m) {
                        const u32 v = low[2 * m];
                        before += (v < mine || (v == mine && m < i)) ? 1u : 0u;
                    }
                } else {                                     // the members of a run agree in the bits >= LOW: whole keys
                    for (u32 m = runStart; m < runEnd; ++m) {
                        const u64 v = keys[m];
                        before += (v < mineKey || (v == mineKey && m < i)) ? 1u : 0u;
                    }
                }
            }
            slot = runStart + before;
        }
        if (act && !tooLong) {
            const u32 dst = dstBase + slot;
            keysOut[dst] = keys[i];
            valsOut[dst] = sm.vals[i];
        }
    }
    if (tooLong) *reinterpret_cast<volatile u32*>(redo) = 1u;
}

template <int SHIFT, int LOW>
__global__ void __launch_bounds__(kSortBlock, kSortMinBlocks)
    onesweepLastKernel(const u64* __restrict__ keysIn, const u32* __restrict__ valsIn, u64* __restrict__ keysOut,
                       u32* __restrict__ valsOut, u32 n, const u32* __restrict__ digitBase, u32* ticket, u64* lookback,
                       u32 epoch, const u32* __restrict__ epochBase, u32* redo)
{
    chainEnter();
    epoch += *epochBase;
    extern __shared__ __align__(16) unsigned char smemRaw[];
    SortSmem& sm = *reinterpret_cast<SortSmem*>(smemRaw);
    __shared__ u32 sCut[2];
    __shared__ u32 sHeadMask[kHeadWords];
    const u32 tid = threadIdx.x;
    if (tid == 0) {
        const u32 t = atomicAdd(ticket, 1u);
        sm.tile = t;
#if CS_SORT_PREFETCH
        // as in the plain pass: the nominal range of the tile one generation of CTAs ahead (its cuts lie at most
        // kFixupMaxRun elements before the nominal ones), on its way into L2
        const u64 nom = ((u64)t + CS_SORT_PREFETCH) * kLastTile;
        if (nom < n) {
            const u64 pb = (nom - kFixupMaxRun) & ~3ull;            // 32-byte aligned for keys, 16-byte for values
            const u32 cnt = (u32)((n - pb) < (u64)kSortTile ? (n - pb) : (u64)kSortTile);
            bulkPrefetchL2(keysIn + pb, (cnt * 8u) & ~15u);
            bulkPrefetchL2(valsIn + pb, (cnt * 4u) & ~15u);
        }
#endif
    }
    u32* whWords = reinterpret_cast<u32*>(sm.warpHist);
    for (int i = tid; i < kHistWords; i += kSortBlock) whWords[i] = 0;
    __syncthreads();
    const u32 tile = sm.tile;
    if (tid < 64) {                                         // warps 0 and 1: where this tile starts and ends
        const u32 w = tid >> 5;
        const u64 nominal = (u64)(tile + w) * kLastTile;
        u32 cut = nominal < n ? (u32)nominal : n;
        bool tooLong = false;
        if (cut > 0 && cut < n) cut = groupStartBefore<LOW, SHIFT>(keysIn, cut, &tooLong);
        if ((tid & 31u) == 0) {
            sCut[w] = cut;
            if (tooLong) *reinterpret_cast<volatile u32*>(redo) = 1u;
        }
    }
    __syncthreads();
    const u32 base = sCut[0], valid = sCut[1] - sCut[0];
    u64 key[kSortItems];
    tileLoadKeys<false>(key, keysIn, base, valid);
    tileStage<SHIFT, false, false>(sm, key, valsIn, tile, base, valid, digitBase, lookback, epoch);
    tileWriteOutFixup<SHIFT, LOW>(sm, sHeadMask, keysOut, valsOut, valid, redo);
}

// The redo behind the fix-up: ONE cooperative launch of persistent CTAs that leaves at once unless *gate != 0
// (the default path pays a few microseconds for it).  Otherwise it sorts the (still complete) input of the fifth
// pass by all 7 digits, least significant first, with a grid barrier between the passes.  The key kernel only
// counts the digits the default path needs, so the histograms of the two lowest digits are made here first.
struct RedoArgs {
    u64* k[2];
    u32* v[2];
    u32 n;
    u32* hist;                  // [kSortPasses][kRadix]: scanned for the digits >= first, zero below
    u32 first;                  // first digit the key kernel / the histogram kernel counted (the plan's)
    u32* tickets;               // kSortPasses ticket counters
    u64* lookback;
    u32 epoch0;                 // pass p uses look-back epoch epoch0 + *epochBase + p
    const u32* epochBase;
    const u32* gate;
};

template <int SHIFT>
__device__ __forceinline__ void redoPass(SortSmem& sm, const RedoArgs& a, int in, u32 epoch0)
{
    const u32 tid = threadIdx.x;
    const u32 tiles = (a.n + kSortTile - 1) / kSortTile;
    u32* whWords = reinterpret_cast<u32*>(sm.warpHist);
    constexpr int pass = SHIFT / kRadixBits;
    for (;;) {
        __syncthreads();                                   // the previous tile is written out
        if (tid == 0) sm.tile = atomicAdd(a.tickets + pass, 1u);
        for (int i = tid; i < kHistWords; i += kSortBlock) whWords[i] = 0;
        __syncthreads();
        const u32 tile = sm.tile;
        if (tile >= tiles) break;
        const u64 base = (u64)tile * kSortTile;
        const u32 valid = (u32)((a.n - base) < (u64)kSortTile ? (a.n - base) : (u64)kSortTile);
        if (valid == kSortTile)
            onesweepTile<SHIFT, false, true, u64, true>(sm, a.k[in], a.v[in], a.k[in ^ 1], a.v[in ^ 1], tile, valid,
                                             a.hist + pass * kRadix, a.lookback, epoch0 + pass);
        else
            onesweepTile<SHIFT, false, false, u64, true>(sm, a.k[in], a.v[in], a.k[in ^ 1], a.v[in ^ 1], tile, valid,
                                              a.hist + pass * kRadix, a.lookback, epoch0 + pass);
    }
}

template <int P>
__device__ __forceinline__ void redoPasses(SortSmem& sm, const RedoArgs& a, cg::grid_group& grid, u32 epoch0)
{
    redoPass<P * kRadixBits>(sm, a, P & 1, epoch0);
    if constexpr (P + 1 < kSortPasses) {
        grid.sync();
        redoPasses<P + 1>(sm, a, grid, epoch0);
    }
}

__global__ void __launch_bounds__(kSortBlock, 1) onesweepRedoKernel(const RedoArgs a)
{
    extern __shared__ __align__(16) unsigned char smemRaw[];
    SortSmem& sm = *reinterpret_cast<SortSmem*>(smemRaw);
    if (*reinterpret_cast<const volatile u32*>(a.gate) == 0) return;
    cg::grid_group grid = cg::this_grid();
    const u32 epoch0 = a.epoch0 + *a.epochBase;
    const u32 tid = threadIdx.x;
    {   // digit counts of the passes the key kernel did not count (zero so far), then their exclusive scans
        u32* sh = reinterpret_cast<u32*>(smemRaw);
        const int first = (int)a.first;                       // at most kSortMaxFirst digits: 8 KB of counters
        for (int i = tid; i < first * kRadix; i += kSortBlock) sh[i] = 0;
        __syncthreads();
        for (u64 i = (u64)blockIdx.x * kSortBlock + tid; i < a.n; i += (u64)gridDim.x * kSortBlock) {
            const u64 k = a.k[0][i];
#pragma unroll
            for (int p = 0; p < kSortMaxFirst; ++p)
                if (p < first) atomicAdd(&sh[p * kRadix + digitOf(k, p * kRadixBits)], 1u);
        }
        __syncthreads();
        for (int i = tid; i < first * kRadix; i += kSortBlock)
            if (sh[i]) atomicAdd(&a.hist[i], sh[i]);
        grid.sync();
        for (u32 p = blockIdx.x; p < a.first; p += gridDim.x) {   // block-uniform trip count
            u32 total;
            u32* warpSums = reinterpret_cast<u32*>(smemRaw);
            const u32 idx = p * kRadix + tid;
            const u32 c = tid < kRadix ? *reinterpret_cast<volatile u32*>(&a.hist[idx]) : 0u;
            __syncthreads();
            const u32 ex = blockExclusiveScan<kSortBlock>(c, warpSums, &total);
            if (tid < kRadix) a.hist[idx] = ex;
            __syncthreads();
        }
        grid.sync();
    }
    redoPasses<0>(sm, a, grid, epoch0);
    if ((kSortPasses & 1) == 0) {                          // an even number of passes ends where it began: move it over
        grid.sync();
        for (u64 i = (u64)blockIdx.x * kSortBlock + tid; i < a.n; i += (u64)gridDim.x * kSortBlock) {
            a.k[1][i] = a.k[0][i];
            a.v[1][i] = a.v[0][i];
        }
    }
}

cs_status enqueueSortReset(cs_context* ctx, cudaStream_t s)
{
    CS_CUDA(ctx, cudaMemsetAsync(ctx->sortHist, 0, (kSortPasses * kRadix + 64) * sizeof(u32), s));
    return CS_OK;
}

// A plan with first digit F sorts by the digits F .. kSortPasses - 1, the last of them (the key's top digit) in the
// fused pass that also orders the bits below F * kRadixBits inside runs of equal leading digits; F = kSortMaxFirst
// (tiny plan), kSortShortFirst (short plan), kSortTopFirst (default plan).  The plain plan sorts by all kSortPasses digits.
constexpr int kLastShift = (kSortPasses - 1) * kRadixBits;
static_assert(kSortMaxFirst + 1 < kSortPasses && kSortMaxFirst == kSortShortFirst + 1 && kSortShortFirst == kSortTopFirst + 1,
              "plans of the sort: first digits 4, 3, 2");

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
    const u32 epoch = nextEpoch(ctx, s);
    const int in = pl.cur, out = in ^ 1;
    launchChained(onesweepKernel<SHIFT, FIRST, u64>, dim3(pl.tiles), dim3(kSortBlock), sizeof(SortSmem), s, 
        pl.k[in], FIRST ? nullptr : pl.v[in], pl.k[out], pl.v[out], pl.n, ctx->sortHist + (SHIFT / kRadixBits) * kRadix,
        ctx->sortTickets + pl.ticketSlot++, ctx->sortLookback, epoch, epochBase(ctx));
    CS_LAUNCH_CHECK(ctx, "onesweepKernel");
    pl.cur = out;
    return CS_OK;
}

// The radix kernels need more dynamic shared memory than the default limit: opt in on the context's device
// (function attributes are per device, so this runs once per cs_create, not once per process).
template <int P>
static cudaError_t sortInitPasses()
{
    const int bytes = (int)sizeof(SortSmem);
    cudaError_t e = cudaFuncSetAttribute(onesweepKernel<P * kRadixBits, false, u64>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if constexpr (P + 1 < kSortPasses) {
        if (e == cudaSuccess) e = sortInitPasses<P + 1>();
    }
    return e;
}
cs_status sortInit32(cs_context* ctx);
cs_status sortInit(cs_context* ctx)
{
    const int bytes = (int)sizeof(SortSmem);
    CS_CUDA(ctx, sortInitPasses<0>());
    CS_CUDA(ctx, cudaFuncSetAttribute(onesweepKernel<0, true, u64>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    CS_CUDA(ctx, cudaFuncSetAttribute(onesweepKernel<kSortTopFirst * kRadixBits, true, u64>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    CS_CUDA(ctx, cudaFuncSetAttribute(onesweepKernel<kSortShortFirst * kRadixBits, true, u64>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    CS_CUDA(ctx, cudaFuncSetAttribute(onesweepKernel<kSortMaxFirst * kRadixBits, true, u64>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    CS_CUDA(ctx, cudaFuncSetAttribute(onesweepLastKernel<kLastShift, kSortTopFirst * kRadixBits>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    CS_CUDA(ctx, cudaFuncSetAttribute(onesweepLastKernel<kLastShift, kSortShortFirst * kRadixBits>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    CS_CUDA(ctx, cudaFuncSetAttribute(onesweepLastKernel<kLastShift, kSortMaxFirst * kRadixBits>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    CS_CUDA(ctx, cudaFuncSetAttribute(onesweepRedoKernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    int perSM = 0;
    CS_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&perSM, onesweepRedoKernel, kSortBlock, bytes));
    if (perSM < 1) return fail(ctx, CS_ERR_CUDA, "onesweepRedoKernel does not fit on an SM");
    ctx->redoGrid = (u32)perSM * (u32)ctx->numSMs;
    return sortInit32(ctx);
}

// the plain passes of the digits P .. END - 1
template <int P, int END>
static cs_status launchPasses(cs_context* ctx, PassPlan& pl, cudaStream_t s)
{
    if constexpr (P < END) {
        CS_TRY((launchPass<P * kRadixBits, false>(ctx, pl, s)));
        return launchPasses<P + 1, END>(ctx, pl, s);
    } else {
        return CS_OK;
    }
}

// Where the first radix pass reads the unsorted keys.  The passes alternate between the workspace's arrays and the
// caller's and must end in the caller's: a plan with an odd number of passes starts in the workspace, one with an even
// number in the caller's arrays.
u64* sortSource(cs_context* ctx, u64* keys, int plan) { return (planPasses(plan) & 1) ? ctx->keysAlt : keys; }

// Which plan the next sort on this context runs (cs_setSortMode; include/cornerstone.h).  CS_SORT_AUTO climbs a
// ladder: the tiny plan; after a plan had to be redone, the next coarser one for planHold sorts (doubling with every
// failure, so that inputs that never fit a plan pay for ever fewer attempts at it); after the default plan had to be
// redone, the plain plan for kPlainHold sorts.
static bool planForced(const cs_context* ctx)
{
    return ctx->sortMode == CS_SORT_PLAIN || ctx->sortMode == CS_SORT_SHORT || ctx->sortMode == CS_SORT_TINY;
}

static int peekPlan(const cs_context* ctx)
{
    switch (ctx->sortMode) {
        case CS_SORT_PLAIN: return kPlanPlain;
        case CS_SORT_SHORT: return kPlanShort;
        case CS_SORT_TINY: return kPlanTiny;
        default: break;
    }
    if (ctx->autoPlainLeft > 0) return kPlanPlain;
    if (ctx->sortMode == CS_SORT_AUTO)
        for (int p = 0; p < kPlanDefault; ++p)
            if (ctx->planLeft[p] == 0) return p;
    return kPlanDefault;
}

void sortPlanOutcome(cs_context* ctx, int plan, bool redone)
{
    if (plan == kPlanPlain) return;
    if (!redone) {
        if (plan < kPlanDefault) ctx->planHold[plan] = kShortHold;     // it fits: forget the back-off
        return;
    }
    if (planForced(ctx)) return;                                        // forced plans do not adapt
    if (plan == kPlanDefault) {
        ctx->autoPlainLeft = kPlainHold;
    } else {
        ctx->planLeft[plan] = ctx->planHold[plan];
        ctx->planHold[plan] = ctx->planHold[plan] * 2 < kShortHoldMax ? ctx->planHold[plan] * 2 : kShortHoldMax;
    }
    // a run too long for this plan lies inside a run of every finer plan: they wait at least their full hold again
    for (int p = 0; p < plan && p < kPlanDefault; ++p)
        if (ctx->planLeft[p] < ctx->planHold[p]) ctx->planLeft[p] = ctx->planHold[p];
}

int sortDecidePlan(cs_context* ctx)
{
    if (ctx->hostCtrl->sortRedoHint) {                      // written by the stream behind an earlier cs_sortKeys
        ctx->hostCtrl->sortRedoHint = 0;
        sortPlanOutcome(ctx, ctx->lastPlan, true);
    }
    const int plan = peekPlan(ctx);
    if (plan == kPlanPlain) {
        if (ctx->autoPlainLeft > 0) --ctx->autoPlainLeft;
    } else if (ctx->sortMode == CS_SORT_AUTO) {             // a sort that does not try a finer plan counts towards its hold
        for (int p = 0; p < plan && p < kPlanDefault; ++p)
            if (ctx->planLeft[p] > 0) --ctx->planLeft[p];
    }
    ctx->lastPlan = plan;
    return plan;
}

int sortPeekPlainPasses(const cs_context* ctx)
{
    int plan = peekPlan(ctx);
    if (ctx->hostCtrl->sortRedoHint && !planForced(ctx) && ctx->lastPlan != kPlanPlain) {
        // the last sort was redone: the next one takes the next coarser plan that is not on hold
        plan = ctx->lastPlan + 1;
        while (plan < kPlanDefault && (ctx->sortMode != CS_SORT_AUTO || ctx->planLeft[plan] > 0)) ++plan;
    }
    return plan == kPlanPlain ? kSortPasses : planPasses(plan) - 1;
}

// the leading digits F + 1 .. and the fused last pass of a plan with first digit F, then the gated redo
template <int F>
static cs_status enqueueShortCut(cs_context* ctx, PassPlan& pl, bool fused, cudaStream_t s)
{
    constexpr int kLow = F * kRadixBits;
    u32* redo = ctx->sortTickets + kSortRedoSlot;
    {   // leading digits
        StageTimer tp(ctx, CS_STAGE_SORT_PASSES, s);
        CS_TRY((launchPass<kLow, true>(ctx, pl, s)));
        CS_TRY((launchPasses<F + 1, kSortPasses - 1>(ctx, pl, s)));
    }
    StageTimer tf(ctx, CS_STAGE_SORT_FIXUP, s);
    {   // top digit; this pass also orders the low bits inside the runs
        const u32 epoch = nextEpoch(ctx, s);
        const int in = pl.cur, out = in ^ 1;
        launchChained(onesweepLastKernel<kLastShift, kLow>, dim3(divUp(pl.n, kLastTile)), dim3(kSortBlock), sizeof(SortSmem), s, 
            pl.k[in], pl.v[in], pl.k[out], pl.v[out], pl.n, ctx->sortHist + (kSortPasses - 1) * kRadix,
            ctx->sortTickets + pl.ticketSlot++, ctx->sortLookback, epoch, epochBase(ctx), redo);
        CS_LAUNCH_CHECK(ctx, "onesweepLastKernel");
    }
    // gated redo from the input of the last pass (pl.cur still names it); its result ends in the other pair,
    // which is where the last pass wrote
    RedoArgs a;
    a.k[0] = pl.k[pl.cur]; a.k[1] = pl.k[pl.cur ^ 1];
    a.v[0] = pl.v[pl.cur]; a.v[1] = pl.v[pl.cur ^ 1];
    a.n = pl.n;
    a.hist = ctx->sortHist;
    a.first = (u32)F;
    a.tickets = ctx->sortTickets + pl.ticketSlot;
    a.lookback = ctx->sortLookback;
    a.epoch0 = reserveEpochs(ctx, kSortPasses, s);
    a.epochBase = epochBase(ctx);
    a.gate = redo;
    const u32 grid = pl.tiles < ctx->redoGrid ? pl.tiles : ctx->redoGrid;
    void* args[] = {(void*)&a};
    CS_CUDA(ctx, cudaLaunchCooperativeKernel((const void*)onesweepRedoKernel, dim3(grid), dim3(kSortBlock), args,
                                             sizeof(SortSmem), s));
    CS_LAUNCH_CHECK(ctx, "onesweepRedoKernel");
    // a hint for callers that never read the control block (cs_sortKeys): the outcome reaches the host with the
    // stream, and the next sort on this context looks at it (cs_buildOctree reads the flag with the control block)
    if (!fused) CS_CUDA(ctx, cudaMemcpyAsync(&ctx->hostCtrl->sortRedoHint, redo, sizeof(u32), cudaMemcpyDeviceToHost, s));
    return CS_OK;
}

// fused: the unsorted keys already lie in sortSource(ctx, keys, plan) and ctx->sortHist holds the counts of the plan's
// digits (cs_buildOctree: the key kernel wrote both); otherwise they are in `keys`.
cs_status enqueueSort(cs_context* ctx, u64* keys, u32* perm, u64 n, bool fused, int plan, cudaStream_t s)
{
    StageTimer t(ctx, CS_STAGE_SORT, s);
    if (n == 0) return CS_OK;
    u64* first = sortSource(ctx, keys, plan);
    {
        StageTimer th(ctx, CS_STAGE_SORT_HIST, s);
        if (!fused) {
            CS_TRY(enqueueSortReset(ctx, s));
            u32 grid = (u32)ctx->numSMs * 4;
            u32 need = divUp((n + 1) / 2, kHistBlock);
            if (need < grid) grid = need ? need : 1;
            sortHistKernel<<<grid, kHistBlock, 0, s>>>(keys, n, ctx->sortHist, first == keys ? nullptr : first,
                                                       planFirstDigit(plan));
            CS_LAUNCH_CHECK(ctx, "sortHistKernel");
        }
        launchChained(sortScanHistKernel, dim3(kSortPasses), dim3(kRadix), 0, s, ctx->sortHist);
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
    if (plan == kPlanPlain) {                               // all digits, least significant first
        StageTimer tp(ctx, CS_STAGE_SORT_PASSES, s);
        CS_TRY((launchPass<0, true>(ctx, pl, s)));
        return launchPasses<1, kSortPasses>(ctx, pl, s);
    }
    return plan == kPlanTiny    ? enqueueShortCut<kSortMaxFirst>(ctx, pl, fused, s)
           : plan == kPlanShort ? enqueueShortCut<kSortShortFirst>(ctx, pl, fused, s)
                                : enqueueShortCut<kSortTopFirst>(ctx, pl, fused, s);
}

// ---- 30-bit keys (L = 10) -----------------------------------------------------------------------
// (u32 key, u32 index): 8 B per element, 16 B per element and pass.  30 bits = 4 digits of 9 bits (the last one 3
// bits wide): 4 plain passes of the same kernel; with so few bits there is nothing left for a fix-up.  An even
// number of passes: they start and end in the caller's arrays.
constexpr int kSortPasses32 = (30 + kRadixBits - 1) / kRadixBits;
static_assert(kSortPasses32 % 2 == 0, "the 30-bit sort starts and ends in the caller's arrays");

__global__ void __launch_bounds__(kHistBlock) sortHist32Kernel(const u32* __restrict__ keys, u64 n, u32* gHist)
{
    __shared__ u32 sh[kSortPasses32 * kRadix];
    for (int i = threadIdx.x; i < kSortPasses32 * kRadix; i += kHistBlock) sh[i] = 0;
    __syncthreads();
    const u64 tid = (u64)blockIdx.x * kHistBlock + threadIdx.x;
    const u64 nthreads = (u64)gridDim.x * kHistBlock;
    auto add = [&](u32 k) {
#pragma unroll
        for (int p = 0; p < kSortPasses32; ++p) atomicAdd(&sh[p * kRadix + digitOf(k, p * kRadixBits)], 1u);
    };
    u64 i = tid;
    for (; i + 3 * nthreads < n; i += 4 * nthreads) {
        const u32 a = ldStreamU32(keys + i), b = ldStreamU32(keys + i + nthreads), c = ldStreamU32(keys + i + 2 * nthreads),
                  d = ldStreamU32(keys + i + 3 * nthreads);
        add(a); add(b); add(c); add(d);
    }
    for (; i < n; i += nthreads) add(ldStreamU32(keys + i));
    __syncthreads();
    for (int j = threadIdx.x; j < kSortPasses32 * kRadix; j += kHistBlock) {
        const u32 v = sh[j];
        if (v) atomicAdd(&gHist[j], v);
    }
}

template <int SHIFT, bool FIRST>
static cs_status launchPass32(cs_context* ctx, u32* const (&k)[2], u32* const (&v)[2], int in, u32 n, u32 tiles, int slot,
                              cudaStream_t s)
{
    const u32 epoch = nextEpoch(ctx, s);
    onesweepKernel<SHIFT, FIRST, u32><<<tiles, kSortBlock, sizeof(SortSmemT<u32>), s>>>(
        k[in], FIRST ? nullptr : v[in], k[in ^ 1], v[in ^ 1], n, ctx->sortHist + (SHIFT / kRadixBits) * kRadix,
        ctx->sortTickets + slot, ctx->sortLookback, epoch, epochBase(ctx));
    CS_LAUNCH_CHECK(ctx, "onesweepKernel<u32>");
    return CS_OK;
}

template <int P>
static cudaError_t sortInitPasses32()
{
    cudaError_t e = cudaFuncSetAttribute(onesweepKernel<P * kRadixBits, false, u32>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)sizeof(SortSmemT<u32>));
    if constexpr (P + 1 < kSortPasses32) {
        if (e == cudaSuccess) e = sortInitPasses32<P + 1>();
    }
    return e;
}

template <int P>
static cs_status launchPasses32(cs_context* ctx, u32* const (&k)[2], u32* const (&v)[2], u32 n, u32 tiles, cudaStream_t s)
{
    if constexpr (P < kSortPasses32) {
        CS_TRY((launchPass32<P * kRadixBits, P == 0>(ctx, k, v, P & 1, n, tiles, P, s)));
        return launchPasses32<P + 1>(ctx, k, v, n, tiles, s);
    } else {
        return CS_OK;
    }
}

cs_status sortInit32(cs_context* ctx)
{
    const int bytes = (int)sizeof(SortSmemT<u32>);
    CS_CUDA(ctx, cudaFuncSetAttribute(onesweepKernel<0, true, u32>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    CS_CUDA(ctx, sortInitPasses32<1>());
    return CS_OK;
}

cs_status enqueueSort32(cs_context* ctx, u32* keys, u32* perm, u64 n, cudaStream_t s)
{
    StageTimer t(ctx, CS_STAGE_SORT, s);
    if (n == 0) return CS_OK;
    {
        StageTimer th(ctx, CS_STAGE_SORT_HIST, s);
        CS_TRY(enqueueSortReset(ctx, s));
        u32 grid = (u32)ctx->numSMs * 4;
        const u32 need = divUp(n, kHistBlock);
        if (need < grid) grid = need ? need : 1;
        sortHist32Kernel<<<grid, kHistBlock, 0, s>>>(keys, n, ctx->sortHist);
        CS_LAUNCH_CHECK(ctx, "sortHist32Kernel");
        launchChained(sortScanHistKernel, dim3(kSortPasses32), dim3(kRadix), 0, s, ctx->sortHist);
        CS_LAUNCH_CHECK(ctx, "sortScanHistKernel");
    }
    u32* const k[2] = {keys, reinterpret_cast<u32*>(ctx->keysAlt)};
    u32* const v[2] = {perm, ctx->permAlt};
    const u32 tiles = divUp(n, kSortTile);
    StageTimer tp(ctx, CS_STAGE_SORT_PASSES, s);
    return launchPasses32<0>(ctx, k, v, (u32)n, tiles, s);
}

}  // namespace cs
