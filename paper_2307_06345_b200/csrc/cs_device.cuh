// Device-side primitives: warp scans, decoupled look-back words, binary search, cache-hinted
// vector loads/stores.  sm_100a only.
#pragma once

#include "cs_internal.cuh"

namespace cs {

constexpr u32 kFull = 0xFFFFFFFFu;

__device__ __forceinline__ u32 laneId()
{
    u32 r;
    asm volatile("mov.u32 %0, %%laneid;" : "=r"(r));
    return r;
}
__device__ __forceinline__ u32 laneMaskLt()
{
    u32 r;
    asm volatile("mov.u32 %0, %%lanemask_lt;" : "=r"(r));
    return r;
}

// ---- streaming 128-bit / 64-bit global accesses ----------------------------------------
// Inputs that are read exactly once bypass L1 allocation (blackwell guide, G13/G14).
__device__ __forceinline__ double2 ldStreamD2(const double* p)
{
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ double ldStreamD(const double* p)
{
    double v;
    asm volatile("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ ulonglong2 ldStreamU2(const u64* p)
{
    ulonglong2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.u64 {%0, %1}, [%2];" : "=l"(v.x), "=l"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ u64 ldStreamU64(const u64* p)
{
    u64 v;
    asm volatile("ld.global.nc.L1::no_allocate.u64 %0, [%1];" : "=l"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ u32 ldStreamU32(const u32* p)
{
    u32 v;
    asm volatile("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ void stStreamU2(u64* p, u64 a, u64 b)
{
    asm volatile("st.global.L1::no_allocate.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(a), "l"(b) : "memory");
}

// Ask the copy engine to bring [p, p + bytes) into L2 (bytes: a multiple of 16, p 16-byte aligned): issued by one thread
// for the tile that a CTA will pick up one generation of resident CTAs later, so that its first loads hit L2.
__device__ __forceinline__ void bulkPrefetchL2(const void* p, u32 bytes)
{
    if (bytes) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// Programmatic dependent launch.  A kernel launched with launchChained() (cs_internal.cuh) may be scheduled while the
// kernel before it on the stream still runs.  chainEnter() is the first statement of such a kernel: it lets the CTAs of
// the kernel BEHIND this one take the slots this grid leaves free (they then wait in their own chainEnter), and waits
// until the kernel before this one has finished and its writes are visible.  No global memory is touched before it.
// Launched without the attribute, both instructions do nothing.
__device__ __forceinline__ void chainEnter()
{
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

// ---- decoupled look-back words -----------------------------------------------------------
// One 64-bit word per (tile, counter): [63:34] epoch, [33:32] status, [31:0] value.  Value and
// flag travel in one 8-byte store, so no fence is needed between them.  The epoch makes
// stale words of earlier launches read as "not ready": the array is never cleared.
constexpr u32 kLbAggregate = 1u;   // value = this tile's own count
constexpr u32 kLbPrefix = 2u;      // value = inclusive prefix over tiles 0..t

__device__ __forceinline__ u64 lbPack(u32 epoch, u32 status, u32 value)
{
    return ((u64)((epoch << 2) | status) << 32) | value;
}
__device__ __forceinline__ void lbStore(u64* p, u64 w)
{
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(w) : "memory");
}
__device__ __forceinline__ u64 lbLoad(const u64* p)
{
    u64 w;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(w) : "l"(p) : "memory");
    return w;
}
// Spin until the word belongs to this epoch; returns it.
__device__ __forceinline__ u64 lbWait(const u64* p, u32 epoch)
{
    u64 w = lbLoad(p);
    while ((u32)(w >> 34) != (epoch & 0x3FFFFFFFu)) {
        __nanosleep(20);
        w = lbLoad(p);
    }
    return w;
}
// Exclusive prefix of counter `c` for tile `tile` (> 0): walk predecessors until a prefix word.
__device__ __forceinline__ u32 lbLookBack(const u64* state, u32 stride, u32 c, u32 tile, u32 epoch)
{
    u32 excl = 0;
    for (u32 p = tile; p-- > 0;) {
        u64 w = lbWait(state + (size_t)p * stride + c, epoch);
        excl += (u32)w;
        if (((u32)(w >> 32) & 3u) == kLbPrefix) break;
    }
    return excl;
}

// Warp-wide look-back for a single counter per tile: the 32 lanes inspect 32 predecessors per
// step, so the frontier of finished prefixes advances 32 tiles per memory round trip.  Must be
// called by all 32 lanes of one warp; returns the exclusive prefix of `tile` (> 0) in every lane.
__device__ __forceinline__ u32 lbLookBackWarp(const u64* state, u32 tile, u32 epoch)
{
    const u32 lane = laneId();
    u32 excl = 0;
    int top = (int)tile - 1;                          // nearest predecessor not yet summed
    while (true) {
        const int p = top - (int)lane;
        u64 w = 0;
        bool isPrefix = false;
        if (p >= 0) {
            w = lbWait(state + p, epoch);
            isPrefix = ((u32)(w >> 32) & 3u) == kLbPrefix;
        }
        const u32 prefMask = __ballot_sync(kFull, isPrefix);
        // lanes up to (and including) the nearest prefix contribute; lanes with p < 0 hold 0
        const u32 nearest = prefMask ? (u32)(__ffs(prefMask) - 1) : 31u;
        u32 v = lane <= nearest ? (u32)w : 0u;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
        excl += v;
        if (prefMask || top < 32) break;             // found a prefix, or reached tile 0 (always a prefix)
        top -= 32;
    }
    return excl;
}

// ---- warp / block scans --------------------------------------------------------------------
__device__ __forceinline__ u32 warpInclusiveScan(u32 v)
{
    const u32 lane = laneId();
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        u32 t = __shfl_up_sync(kFull, v, o);
        if (lane >= (u32)o) v += t;
    }
    return v;
}
__device__ __forceinline__ u32 warpReduceSum(u32 v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}

// Block-wide exclusive scan of one value per thread.  `warpSums` = smem scratch of BLOCK/32 + 1
// words.  Returns the exclusive prefix; *total receives the block sum.  Contains 2 barriers.
template <int BLOCK>
__device__ __forceinline__ u32 blockExclusiveScan(u32 v, u32* warpSums, u32* total)
{
    constexpr int WARPS = BLOCK / 32;
    const u32 lane = laneId();
    const u32 warp = threadIdx.x >> 5;
    u32 inc = warpInclusiveScan(v);
    if (lane == 31) warpSums[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        u32 s = lane < WARPS ? warpSums[lane] : 0;
        u32 si = warpInclusiveScan(s);
        if (lane < WARPS) warpSums[lane] = si - s;
        if (lane == WARPS - 1) warpSums[WARPS] = si;
    }
    __syncthreads();
    *total = warpSums[WARPS];
    return warpSums[warp] + inc - v;
}

// ---- binary search ---------------------------------------------------------------------------
// First index in [lo, hi) with P[idx] >= key (hi if none): Eq. 3's "locating K_i in P", A6.
__device__ __forceinline__ u32 lowerBound(const u64* __restrict__ P, u32 lo, u32 hi, u64 key)
{
    while (lo < hi) {
        u32 mid = lo + ((hi - lo) >> 1);
        if (__ldg(P + mid) < key) lo = mid + 1;
        else hi = mid;
    }
    return lo;
}

// division level of a cornerstone gap delta = 8^m: L - m; delta must be a power of 8
__device__ __forceinline__ int levelOfDelta(u64 delta) { return kL - (63 - __clzll((long long)delta)) / 3; }

// true iff delta is 8^m with 0 <= m <= L
__device__ __forceinline__ bool isPowerOf8(u64 delta)
{
    if (delta == 0 || (delta & (delta - 1))) return false;
    return ((63 - __clzll((long long)delta)) % 3) == 0;
}

}  // namespace cs
