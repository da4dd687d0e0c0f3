// cs_partitionLeavesStatic: the SFC domain decomposition of cs_partitionLeaves (A29) for
// callers that must not allocate: no context (cs_create calls cudaMalloc), no workspace.  The scratch of the kernel,
// one 64-bit sum per tile of kStatTile leaf counts plus a ticket, lives in a file-scope __device__ array of fixed size,
// so the entry point takes at most CS_STATIC_PARTITION_MAX_LEAVES leaves.  Every GPU that loads the library holds
// the array (kStatWords * 8 bytes = 64.25 KB) until the process exits.
//
// One kernel (the context path runs two: partTileSumKernel, partBoundsKernel in cs_global.cu): every CTA sums its
// tile into the scratch and draws a ticket; the CTA that draws the last one scans the sums and finds the boundaries.
// All calls share the array: calls that overlap on the GPU (two streams, two host threads) race, the caller
// serialises them.  The ticket must start at zero and is cleared by a memset node in front of every launch; the
// sums are overwritten before they are read, so what an earlier call left behind does not matter.
#include <mutex>

#include "cs_device.cuh"

namespace cs {

constexpr int kStatTile = 2048;                                            // leaf counts per CTA
constexpr u32 kStatMaxTiles = CS_STATIC_PARTITION_MAX_LEAVES / kStatTile;  // 8192
constexpr u32 kStatWords = kStatMaxTiles + 32;                             // + the ticket's own 256 bytes
constexpr int kStatBlock = 256;
static_assert(CS_STATIC_PARTITION_MAX_LEAVES % kStatTile == 0, "whole tiles");

// In host code this name is a host-side stand-in, not a device address: host code uses staticScratch() below.
static __device__ __align__(256) unsigned long long g_partScratch[kStatWords];

__device__ __forceinline__ bool statReached(u64 C, u32 R, u32 r, u64 total)   // C * R >= r * total, in 128 bits
{
    const u64 ah = __umul64hi(C, (u64)R), al = C * (u64)R;
    const u64 bh = __umul64hi(total, (u64)r), bl = total * (u64)r;
    return ah > bh || (ah == bh && al >= bl);
}

__device__ __forceinline__ u64 warpInclusiveScanU64(u64 v, u32 lane)
{
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const u64 u = __shfl_up_sync(kFull, v, o);
        if (lane >= (u32)o) v += u;
    }
    return v;
}

// scratch: [0, tiles) tile sums (then their exclusive prefix), [kStatMaxTiles] the ticket (zero at launch)
__global__ void __launch_bounds__(kStatBlock)
    partitionStaticKernel(const u32* __restrict__ N, u32 nl, u64* scratch, u32 tiles, u32 R, u32* __restrict__ bounds)
{
    __shared__ u64 red[kStatBlock / 32];
    __shared__ u64 sCarry;
    __shared__ bool sLast;
    const u32 tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    // ---- sum of this CTA's tile ---------------------------------------------------------------------------
    {
        const u32 t0 = blockIdx.x * kStatTile;
        u64 s = 0;
        for (u32 q = tid; q < (u32)kStatTile; q += kStatBlock) {
            const u32 i = t0 + q;
            if (i < nl) s += N[i];
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(kFull, s, o);
        if (lane == 0) red[warp] = s;
        __syncthreads();
        if (tid == 0) {
            u64 v = 0;
            for (int w = 0; w < kStatBlock / 32; ++w) v += red[w];
            scratch[blockIdx.x] = v;
            __threadfence();                                                 // the sum before the ticket
            u32* ticket = reinterpret_cast<u32*>(scratch + kStatMaxTiles);
            sLast = (atomicAdd(ticket, 1u) + 1u == tiles);
            sCarry = 0;
        }
        __syncthreads();
        if (!sLast) return;
        __threadfence();
    }
    // ---- last CTA: exclusive scan of the tile sums, in place, kStatBlock at a time ---------------------------
    for (u32 b = 0; b < tiles; b += kStatBlock) {
        const u32 t = b + tid;
        const u64 v = t < tiles ? __ldcg(scratch + t) : 0;
        const u64 inc = warpInclusiveScanU64(v, lane);
        if (lane == 31) red[warp] = inc;
        __syncthreads();
        u64 before = sCarry;
        for (u32 w = 0; w < warp; ++w) before += red[w];
        if (t < tiles) scratch[t] = before + inc - v;
        __syncthreads();
        if (tid == kStatBlock - 1) sCarry = before + inc;
        __syncthreads();
    }
    const u64 total = sCarry;
    if (tid == 0) {
        bounds[0] = 0;
        bounds[R] = nl;
    }
    // ---- one warp per boundary r: the tile by a binary search over the prefixes, then a walk over its counts ----
    for (u32 r = 1 + warp; r < R; r += kStatBlock / 32) {
        u32 result = 0;
        if (total != 0) {
            u32 lo = 0, hi = tiles;                                  // invariant: tile lo qualifies, tile hi does not
            while (hi - lo > 1) {
                const u32 mid = (lo + hi) >> 1;
                if (!statReached(scratch[mid], R, r, total)) lo = mid;
                else hi = mid;
            }
            u64 C = scratch[lo];
            const u32 t0 = lo * kStatTile;
            result = nl;
            for (u32 q = 0; q < (u32)kStatTile; q += 32) {           // first i > t0 with C_i * R >= r * total
                const u32 i = t0 + q + lane;
                const u64 inc = warpInclusiveScanU64(i < nl ? N[i] : 0, lane);
                const u32 m = __ballot_sync(kFull, statReached(C + inc, R, r, total));   // C_{i+1}
                if (m) {
                    result = t0 + q + (u32)__ffs((int)m);
                    break;
                }
                C += __shfl_sync(kFull, inc, 31);
            }
            if (result > nl) result = nl;
        }
        if (lane == 0) bounds[r] = result;
    }
}

// Device address of g_partScratch on the current device: looked up once per device (with that device current), no
// allocation.
constexpr int kStatMaxDevices = 64;
static std::mutex g_statMutex;
static u64* g_statPtr[kStatMaxDevices] = {};

static cs_status staticScratch(u64** out, const char* fn)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cudaFail(nullptr, e, fn);
    if (dev < 0 || dev >= kStatMaxDevices) return fail(nullptr, CS_ERR_INVALID_ARG, "%s: device %d out of range", fn, dev);
    std::lock_guard<std::mutex> lock(g_statMutex);
    if (!g_statPtr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_partScratch);
        if (e != cudaSuccess || !p) return cudaFail(nullptr, e, "cudaGetSymbolAddress (cs_partitionLeavesStatic)");
        g_statPtr[dev] = (u64*)p;
    }
    *out = g_statPtr[dev];
    return CS_OK;
}

}  // namespace cs

using namespace cs;

extern "C" {

uint32_t cs_partitionLeavesStaticMax(void) { return CS_STATIC_PARTITION_MAX_LEAVES; }

cs_status cs_partitionLeavesStaticSetup(void)
{
    u64* p = nullptr;
    return staticScratch(&p, "cs_partitionLeavesStaticSetup");
}

cs_status cs_partitionLeavesStatic(const uint32_t* counts, uint32_t numLeaves, uint32_t numRanks, uint32_t* bounds,
                                   void* stream)
{
    if (!counts || !bounds) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_partitionLeavesStatic: null pointer");
    if (numLeaves == 0 || numRanks == 0)
        return fail(nullptr, CS_ERR_INVALID_ARG, "cs_partitionLeavesStatic: numLeaves or numRanks is 0");
    if (numLeaves > CS_STATIC_PARTITION_MAX_LEAVES)
        return fail(nullptr, CS_ERR_CAPACITY,
                    "cs_partitionLeavesStatic: numLeaves = %u exceeds the static scratch (at most %u leaves); use "
                    "cs_partitionLeaves with a context",
                    numLeaves, (unsigned)CS_STATIC_PARTITION_MAX_LEAVES);
    u64* scratch = nullptr;
    CS_TRY(staticScratch(&scratch, "cs_partitionLeavesStatic"));
    cudaStream_t s = (cudaStream_t)stream;
    const u32 tiles = divUp(numLeaves, kStatTile);
    cudaError_t e = cudaMemsetAsync(scratch + kStatMaxTiles, 0, sizeof(u64), s);   // the ticket starts at zero
    if (e != cudaSuccess) return cudaFail(nullptr, e, "cs_partitionLeavesStatic (ticket reset)");
    partitionStaticKernel<<<tiles, kStatBlock, 0, s>>>(counts, numLeaves, scratch, tiles, numRanks, bounds);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cudaFail(nullptr, e, "partitionStaticKernel");
    return CS_OK;
}

}  // extern "C"
