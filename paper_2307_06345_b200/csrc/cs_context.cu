// Context, workspace, error plumbing, profiling, device-wide exclusive scan.
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

#include "cs_device.cuh"

namespace cs {

static thread_local char g_lastError[512] = "";

cs_status fail(cs_context* ctx, cs_status st, const char* fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof(buf), fmt, ap);
    va_end(ap);
    snprintf(g_lastError, sizeof(g_lastError), "%s", buf);
    if (ctx) ctx->lastError = buf;
    return st;
}

cs_status cudaFail(cs_context* ctx, cudaError_t e, const char* what)
{
    return fail(ctx, CS_ERR_CUDA, "CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
}

// ---- workspace layout --------------------------------------------------------------------
struct Layout {
    size_t keysAlt, permAlt, sortHist, sortLookback, boxPartials, boxCounter, leafK0, leafK1, leafOff0, leafOff1,
        leafOffFinal, leafTasks, leafOpk, leafTileInfo, divLevel, tileLookback, dirFlags, dirTotals, dirBases, dirListSize, dirListKeys, dirListMeta, linkTileHist, hilbertTable, epochWords, ctrl, total;
};

static size_t alignUp(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

static Layout makeLayout(uint64_t maxParticles, uint32_t maxLeaves, int boxGrid)
{
    Layout L{};
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o = alignUp(o + bytes); return at; };
    const size_t sortTiles = (maxParticles + kSortLastTile - 1) / kSortLastTile + 1;   // the smaller of the two tile sizes
    const size_t dirTiles = (maxParticles >> kDirectTileLog2) + 2;          // one-pass leaf build: positions 0 .. n
    size_t leafTiles = ((size_t)maxLeaves + 1 + 1023) / 1024 + 1;          // covers kLeafTile, kScanTile >= 1024
    if (leafTiles < dirTiles / 1024 + 2) leafTiles = dirTiles / 1024 + 2;  // the scan of the one-pass build's tile totals
    const size_t linkTiles = ((size_t)maxLeaves + kLinkTile - 1) / kLinkTile + 1;
    static_assert(kLeafTile >= 1024 && kScanTile >= 1024, "look-back array is sized for tiles of >= 1024");
    L.keysAlt = take(maxParticles * sizeof(u64));
    L.permAlt = take(maxParticles * sizeof(u32));
    L.sortHist = take((kSortPasses * kRadix + 64) * sizeof(u32));
    L.sortLookback = take(sortTiles * kRadix * sizeof(u64));
    L.boxPartials = take((size_t)boxGrid * 6 * sizeof(double));
    L.boxCounter = take(64);
    L.leafK0 = take(((size_t)maxLeaves + 2) * sizeof(u64));
    L.leafK1 = take(((size_t)maxLeaves + 2) * sizeof(u64));
    L.leafOff0 = take(((size_t)maxLeaves + 2) * sizeof(u32));
    L.leafOff1 = take(((size_t)maxLeaves + 2) * sizeof(u32));
    L.leafOffFinal = take(((size_t)maxLeaves + 2) * sizeof(u32));
    L.leafTasks = take(2 * ((size_t)maxLeaves / 8 + 8) * sizeof(uint4));   // linear list, search list
    const size_t roundTiles = ((size_t)maxLeaves + kLeafTile - 1) / kLeafTile + 1;
    L.leafOpk = take(roundTiles * kLeafBlock * sizeof(u32));
    L.leafTileInfo = take(roundTiles * sizeof(uint4));
    L.divLevel = take(dirTiles << kDirectTileLog2);                        // 1 byte per particle, whole tiles
    L.tileLookback = take(leafTiles * sizeof(u64));                        // one counter per tile (leaf rounds, scan)
    L.dirFlags = take(dirTiles << (kDirectTileLog2 - 3));                  // one-pass leaf build: 1 bit per position
    L.dirTotals = take((dirTiles + 2) * sizeof(u32));                      // K entries per tile
    L.dirBases = take((dirTiles + 2) * sizeof(u32));                       // exclusive prefix of dirTotals
    L.dirListSize = take(dirTiles * sizeof(u32));
    L.dirListKeys = take(dirTiles * kDirectCompact * sizeof(ulonglong2));   // 2 B per particle
    L.dirListMeta = take(dirTiles * kDirectCompact * sizeof(u32));          // 0.5 B per particle
    L.linkTileHist = take(linkTiles * kLinkBins * sizeof(u32));            // plain counts, never look-back words
    L.hilbertTable = take(24 * 512 * sizeof(unsigned short) + 24 * 8);      // + the one-level inverse table
    L.epochWords = take(64);
    L.ctrl = take(sizeof(DeviceCtrl));
    L.total = o;
    return L;
}

constexpr int kBoxGridMax = 148 * 8;

// Look-back words carry the epoch of the launch that wrote them, so the arrays are never cleared between
// launches; only when the 30-bit epoch counter would wrap are they zeroed once (epoch 0 is never handed out).
u32 reserveEpochs(cs_context* ctx, u32 count, cudaStream_t s)
{
    if (ctx->capturing) {                                   // relative to the base the replay supplies (cs_api.cu)
        const u32 first = ctx->captureEpochs + 1;
        ctx->captureEpochs += count;
        return first;
    }
    if (ctx->epoch + count >= (1u << 30)) {
        Layout L = makeLayout(ctx->maxParticles, ctx->maxLeaves, kBoxGridMax);
        cudaError_t e = cudaMemsetAsync(ctx->sortLookback, 0, L.boxPartials - L.sortLookback, s);
        if (e == cudaSuccess) e = cudaMemsetAsync(ctx->tileLookback, 0, L.dirFlags - L.tileLookback, s);
        if (e != cudaSuccess) cudaFail(ctx, e, "reserveEpochs (look-back reset)");   // the next launch check reports it
        ctx->epoch = 0;
    }
    const u32 first = ctx->epoch + 1;
    ctx->epoch += count;
    return first;
}

u32 nextEpoch(cs_context* ctx, cudaStream_t s) { return reserveEpochs(ctx, 1, s); }

cs_status enqueueReadCtrl(cs_context* ctx, cudaStream_t s)
{
    CS_CUDA(ctx, cudaMemcpyAsync(&ctx->hostCtrl->c, ctx->ctrl, sizeof(DeviceCtrl), cudaMemcpyDeviceToHost, s));
    CS_CUDA(ctx, cudaMemcpyAsync(&ctx->hostCtrl->sortRedo, ctx->sortTickets + kSortRedoSlot, sizeof(u32),
                                 cudaMemcpyDeviceToHost, s));
    return CS_OK;
}

cs_status readCtrl(cs_context* ctx, cudaStream_t s)
{
    CS_TRY(enqueueReadCtrl(ctx, s));
    CS_CUDA(ctx, cudaStreamSynchronize(s));
    return CS_OK;
}

// ---- device-wide exclusive scan (g2's building block; decoupled look-back) -----------------
__global__ void __launch_bounds__(kScanBlock) scanKernel(const u32* __restrict__ in, u32* __restrict__ out, u32 n,
                                                         u32* ticket, u64* lookback, u32 epoch,
                                                         const u32* __restrict__ epochBase)
{
    chainEnter();
    epoch += *epochBase;
    __shared__ u32 sTile, sPrefix;
    __shared__ u32 warpSums[kScanBlock / 32 + 1];
    const u32 tiles = (n + kScanTile - 1) / kScanTile;
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) sTile = atomicAdd(ticket, 1u);
        __syncthreads();
        const u32 tile = sTile;
        if (tile >= tiles) break;
        const u32 first = tile * kScanTile + threadIdx.x * kScanItems;
        u32 v[kScanItems];
        u32 sum = 0;
#pragma unroll
        for (int k = 0; k < kScanItems; ++k) {
            v[k] = (first + k < n) ? in[first + k] : 0u;
            sum += v[k];
        }
        u32 total;
        u32 excl = blockExclusiveScan<kScanBlock>(sum, warpSums, &total);
        if (threadIdx.x < 32) {                       // warp 0: publish, then warp-wide look-back
            u64* st = lookback + tile;
            u32 p = 0;
            if (tile == 0) {
                if (threadIdx.x == 0) lbStore(st, lbPack(epoch, kLbPrefix, total));
            } else {
                if (threadIdx.x == 0) lbStore(st, lbPack(epoch, kLbAggregate, total));
                p = lbLookBackWarp(lookback, tile, epoch);
                if (threadIdx.x == 0) lbStore(st, lbPack(epoch, kLbPrefix, p + total));
            }
            if (threadIdx.x == 0) {
                sPrefix = p;
                if (tile == tiles - 1) out[n] = p + total;
            }
        }
        __syncthreads();
        u32 run = sPrefix + excl;
#pragma unroll
        for (int k = 0; k < kScanItems; ++k) {
            if (first + k < n) out[first + k] = run;
            run += v[k];
        }
    }
}

__global__ void setU32Kernel(u32* p, u32 v) { *p = v; }

cs_status enqueueExclusiveScan(cs_context* ctx, const u32* in, u32* out, u32 n, cudaStream_t s)
{
    if (n == 0) {
        setU32Kernel<<<1, 1, 0, s>>>(out, 0u);
        CS_LAUNCH_CHECK(ctx, "setU32Kernel");
        return CS_OK;
    }
    CS_CUDA(ctx, cudaMemsetAsync(&ctx->ctrl->scanTicket, 0, sizeof(u32), s));
    u32 epoch = nextEpoch(ctx, s);
    u32 tiles = divUp(n, kScanTile);
    u32 grid = tiles < (u32)ctx->numSMs * 8 ? tiles : (u32)ctx->numSMs * 8;
    launchChained(scanKernel, dim3(grid), dim3(kScanBlock), 0, s, in, out, n, &ctx->ctrl->scanTicket, ctx->tileLookback, epoch, epochBase(ctx));
    CS_LAUNCH_CHECK(ctx, "scanKernel");
    return CS_OK;
}

}  // namespace cs

using namespace cs;

extern "C" {

const char* cs_version(void) { return "cornerstone-b200 0.1 (sm_100a)"; }

size_t cs_workspaceBytes(uint64_t maxParticles, uint32_t maxLeaves)
{
    return makeLayout(maxParticles, maxLeaves, kBoxGridMax).total;
}

const char* cs_lastError(const cs_context* ctx) { return ctx ? ctx->lastError.c_str() : g_lastError; }

cs_status cs_create(cs_context** out, int device, uint64_t maxParticles, uint32_t maxLeaves)
{
    if (!out) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_create: ctx is null");
    *out = nullptr;
    if (maxParticles >= (1ull << 32)) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_create: maxParticles >= 2^32");
    if (maxLeaves == 0 || maxLeaves > 0x7FFFFFF0u)
        return fail(nullptr, CS_ERR_INVALID_ARG, "cs_create: maxLeaves out of range");
    cs_context* ctx = new (std::nothrow) cs_context();
    if (!ctx) return fail(nullptr, CS_ERR_CUDA, "cs_create: out of host memory");
    ctx->device = device;
    ctx->maxParticles = maxParticles;
    ctx->maxLeaves = maxLeaves;
    ctx->maxNodes = maxLeaves + (maxLeaves - 1) / 7 + 1;
    DeviceGuard guard(device);                 // the caller's current device is restored on return
    cudaError_t e = guard.err;
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->numSMs, cudaDevAttrMultiProcessorCount, device);
    Layout L = makeLayout(maxParticles, maxLeaves, kBoxGridMax);
    if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->slab, L.total);
    if (e == cudaSuccess) e = cudaMemset(ctx->slab + L.sortHist, 0, L.total - L.sortHist);
    if (e == cudaSuccess) e = cudaMallocHost((void**)&ctx->hostCtrl, sizeof(HostCtrl));
    if (e == cudaSuccess) memset(ctx->hostCtrl, 0, sizeof(HostCtrl));
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&ctx->captureStream, cudaStreamNonBlocking);
    for (int i = 0; i < CS_NUM_STAGES && e == cudaSuccess; ++i) {
        e = cudaEventCreate(&ctx->evBegin[i]);
        if (e == cudaSuccess) e = cudaEventCreate(&ctx->evEnd[i]);
    }
    if (e != cudaSuccess) {
        cs_status st = cudaFail(nullptr, e, "cs_create");
        cs_destroy(ctx);
        return st;
    }
    ctx->slabBytes = L.total;
    ctx->keysAlt = (u64*)(ctx->slab + L.keysAlt);
    ctx->permAlt = (u32*)(ctx->slab + L.permAlt);
    ctx->sortHist = (u32*)(ctx->slab + L.sortHist);
    ctx->sortTickets = ctx->sortHist + kSortPasses * kRadix;
    ctx->sortLookback = (u64*)(ctx->slab + L.sortLookback);
    ctx->boxPartials = (double*)(ctx->slab + L.boxPartials);
    ctx->boxCounter = (u32*)(ctx->slab + L.boxCounter);
    ctx->leafK[0] = (u64*)(ctx->slab + L.leafK0);
    ctx->leafK[1] = (u64*)(ctx->slab + L.leafK1);
    ctx->leafOff[0] = (u32*)(ctx->slab + L.leafOff0);
    ctx->leafOff[1] = (u32*)(ctx->slab + L.leafOff1);
    ctx->leafOffFinal = (u32*)(ctx->slab + L.leafOffFinal);
    ctx->leafTasks = (uint4*)(ctx->slab + L.leafTasks);
    ctx->leafOpk = (u32*)(ctx->slab + L.leafOpk);
    ctx->leafTileInfo = (uint4*)(ctx->slab + L.leafTileInfo);
    ctx->divLevel = (unsigned char*)(ctx->slab + L.divLevel);
    ctx->maxTasks = maxLeaves / 8 + 8;
    ctx->tileLookback = (u64*)(ctx->slab + L.tileLookback);
    ctx->dirFlags = (unsigned char*)(ctx->slab + L.dirFlags);
    ctx->dirTotals = (u32*)(ctx->slab + L.dirTotals);
    ctx->dirBases = (u32*)(ctx->slab + L.dirBases);
    ctx->dirListSize = (u32*)(ctx->slab + L.dirListSize);
    ctx->dirListKeys = (ulonglong2*)(ctx->slab + L.dirListKeys);
    ctx->dirListMeta = (u32*)(ctx->slab + L.dirListMeta);
    ctx->linkTileHist = (u32*)(ctx->slab + L.linkTileHist);
    ctx->ctrl = (DeviceCtrl*)(ctx->slab + L.ctrl);
    ctx->epochWords = (u32*)(ctx->slab + L.epochWords);
    ctx->hilbertTable = (unsigned short*)(ctx->slab + L.hilbertTable);
    {
        unsigned short table[24 * 512];
        hilbertBuildTable(table);
        e = cudaMemcpy(ctx->hilbertTable, table, sizeof(table), cudaMemcpyHostToDevice);
        unsigned char inv[24 * 8];
        hilbertBuildInverse(inv);
        ctx->hilbertInverse = reinterpret_cast<unsigned char*>(ctx->hilbertTable + 24 * 512);
        if (e == cudaSuccess) e = cudaMemcpy(ctx->hilbertInverse, inv, sizeof(inv), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) {
            cs_status stc = cudaFail(nullptr, e, "cs_create (Hilbert table)");
            cs_destroy(ctx);
            return stc;
        }
    }
    cs_status st = sortInit(ctx);
    if (st == CS_OK) st = leavesDirectInit(ctx);
    if (st == CS_OK) st = leavesInit(ctx);
    if (st != CS_OK) {
        cs_destroy(ctx);
        return st;
    }
    *out = ctx;
    return CS_OK;
}

void cs_destroy(cs_context* ctx)
{
    if (!ctx) return;
    DeviceGuard guard(ctx->device);
    if (ctx->slab) cudaFree(ctx->slab);
    if (ctx->hostPathSlab) cudaFree(ctx->hostPathSlab);
    if (ctx->wideSlab) cudaFree(ctx->wideSlab);
    if (ctx->hostCtrl) cudaFreeHost(ctx->hostCtrl);
    if (ctx->buildGraph) cudaGraphExecDestroy(ctx->buildGraph);
    if (ctx->captureStream) cudaStreamDestroy(ctx->captureStream);
    if (ctx->copyStream) cudaStreamDestroy(ctx->copyStream);
    for (cudaEvent_t e : ctx->copyEvents)
        if (e) cudaEventDestroy(e);
    for (int i = 0; i < CS_NUM_STAGES; ++i) {
        if (ctx->evBegin[i]) cudaEventDestroy(ctx->evBegin[i]);
        if (ctx->evEnd[i]) cudaEventDestroy(ctx->evEnd[i]);
    }
    delete ctx;
}

cs_status cs_setProfiling(cs_context* ctx, int enabled)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_setProfiling: ctx is null");
    ctx->profiling = enabled != 0;
    for (int i = 0; i < CS_NUM_STAGES; ++i) ctx->evUsed[i] = false;
    return CS_OK;
}

cs_status cs_stageTimes(cs_context* ctx, float* ms, uint64_t* launches)
{
    if (!ctx || !ms) return fail(ctx, CS_ERR_INVALID_ARG, "cs_stageTimes: null argument");
    for (int i = 0; i < CS_NUM_STAGES; ++i) {
        ms[i] = 0.f;
        if (ctx->evUsed[i]) {
            CS_CUDA(ctx, cudaEventSynchronize(ctx->evEnd[i]));
            CS_CUDA(ctx, cudaEventElapsedTime(&ms[i], ctx->evBegin[i], ctx->evEnd[i]));
        }
    }
    if (launches) *launches = ctx->launches;
    return CS_OK;
}

}  // extern "C"
