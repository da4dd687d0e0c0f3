// extern "C" entry points of libcornerstone_b200.so (see include/cornerstone.h).
#include <cstring>
#include <new>

#include "cs_internal.cuh"

using namespace cs;

namespace {

cs_status statusFromCtrl(cs_context* ctx, const char* where)
{
    const u32 st = ctx->hostCtrl->c.status;
    switch (st) {
        case CS_OK: return CS_OK;
        case CS_ERR_CAPACITY: return fail(ctx, CS_ERR_CAPACITY, "%s: result exceeds the given capacity", where);
        case CS_ERR_NOT_CORNERSTONE:
            return fail(ctx, CS_ERR_NOT_CORNERSTONE, "%s: leaf array violates Eq. 2 (not a cornerstone array)", where);
        case CS_ERR_NOT_CONVERGED:
            return fail(ctx, CS_ERR_NOT_CONVERGED, "%s: maxRounds reached before convergence", where);
        default: return fail(ctx, CS_ERR_CUDA, "%s: unexpected device status %u", where, st);
    }
}

cs_status checkParticles(cs_context* ctx, const char* fn, uint64_t n)
{
    if (n >= (1ull << 32)) return fail(ctx, CS_ERR_INVALID_ARG, "%s: n >= 2^32", fn);
    if (n > ctx->maxParticles)
        return fail(ctx, CS_ERR_CAPACITY, "%s: n = %llu exceeds the context's maxParticles = %llu", fn,
                    (unsigned long long)n, (unsigned long long)ctx->maxParticles);
    return CS_OK;
}

// the stages of cs_buildOctree back to back on `s`, ending with the copy of the control block to the host
cs_status enqueueBuild(cs_context* ctx, const double* x, const double* y, const double* z, uint64_t n, uint32_t bucketSize,
                       const uint64_t* prevLeaves, uint32_t prevNumLeaves, uint32_t maxRounds, const cs_octree_buffers* b,
                       int plan, cudaStream_t s)
{
    const u32 leafCap = b->leafCapacity < ctx->maxLeaves ? b->leafCapacity : ctx->maxLeaves;
    if (!ctx->boxReady) CS_TRY(enqueueBox(ctx, x, y, z, n, b->box6, s));
    CS_TRY(enqueueSortReset(ctx, s));
    // the key kernel writes where the first radix pass reads, and accumulates the histograms of the plan's digits
    CS_TRY(enqueueKeys(ctx, x, y, z, n, b->box6, sortSource(ctx, (u64*)b->keys, plan), planFirstDigit(plan), ctx->curve, s));
    CS_TRY(enqueueSort(ctx, (u64*)b->keys, b->perm, n, /*fused=*/true, plan, s));
    CS_TRY(enqueueLeaves(ctx, (const u64*)b->keys, n, bucketSize, (const u64*)prevLeaves, prevNumLeaves, maxRounds,
                         (u64*)b->leaves, b->counts, leafCap, kL, s));
    // link and node counts in one pass: the leaves' particle offsets are still in the workspace
    CS_TRY(enqueueLink(ctx, (const u64*)b->leaves, &ctx->ctrl->numLeaves, 0, leafCap, (u64*)b->prefixes, b->levels,
                       b->childOffsets, b->parents, b->levelRange, b->leafToNode, b->nodeToLeaf, b->nodeCapacity,
                       ctx->leafOffFinal, b->nodeFirst, b->nodeCount, s));
    return enqueueReadCtrl(ctx, s);
}

// Capture enqueueBuild as a CUDA graph on the context's own stream (the caller's may be the legacy default stream,
// which cannot be captured) and instantiate it.  The look-back epochs of the captured kernels are relative to a device
// word that the graph's first node loads from the pinned control block, so that every replay runs in fresh epochs.
// If the driver refuses (capture or instantiation), graphs are switched off for this context and the caller enqueues
// the stages directly.
cs_status captureBuild(cs_context* ctx, const double* x, const double* y, const double* z, uint64_t n, uint32_t bucketSize,
                       const uint64_t* prevLeaves, uint32_t prevNumLeaves, uint32_t maxRounds, const cs_octree_buffers* b,
                       int plan)
{
    if (ctx->buildGraph) {
        cudaGraphExecDestroy(ctx->buildGraph);
        ctx->buildGraph = nullptr;
    }
    cudaStream_t cs_ = ctx->captureStream;
    if (cudaStreamBeginCapture(cs_, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
        cudaGetLastError();
        ctx->graphMaxParticles = 0;
        return CS_OK;
    }
    const uint64_t launches0 = ctx->launches;
    ctx->capturing = true;
    ctx->captureEpochs = 0;
    cudaError_t e = cudaMemcpyAsync(ctx->epochWords + 1, &ctx->hostCtrl->epochBase, sizeof(u32), cudaMemcpyHostToDevice, cs_);
    cs_status st = e == cudaSuccess
                       ? enqueueBuild(ctx, x, y, z, n, bucketSize, prevLeaves, prevNumLeaves, maxRounds, b, plan, cs_)
                       : CS_ERR_CUDA;
    ctx->capturing = false;
    cudaGraph_t graph = nullptr;
    e = cudaStreamEndCapture(cs_, &graph);
    ctx->buildGraphLaunches = ctx->launches - launches0;
    ctx->launches = launches0;
    ctx->buildGraphEpochs = ctx->captureEpochs;
    if (st == CS_OK && e == cudaSuccess && graph) e = cudaGraphInstantiate(&ctx->buildGraph, graph, 0);
    if (graph) cudaGraphDestroy(graph);
    if (st != CS_OK || e != cudaSuccess || !ctx->buildGraph) {     // not capturable here: enqueue directly from now on
        cudaGetLastError();
        ctx->buildGraph = nullptr;
        ctx->graphMaxParticles = 0;
    }
    return CS_OK;
}

}  // namespace

extern "C" {

cs_status cs_computeBox(cs_context* ctx, const double* x, const double* y, const double* z, uint64_t n,
                        double* box6, void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_computeBox: ctx is null");
    if (!x || !y || !z || !box6) return fail(ctx, CS_ERR_INVALID_ARG, "cs_computeBox: null pointer");
    if (n == 0) return fail(ctx, CS_ERR_INVALID_ARG, "cs_computeBox: n == 0 (an empty set has no box)");
    CS_TRY(checkParticles(ctx, "cs_computeBox", n));
    DeviceGuard g(ctx->device);
    return enqueueBox(ctx, x, y, z, n, box6, (cudaStream_t)stream);
}

cs_status cs_computeKeys(cs_context* ctx, const double* x, const double* y, const double* z, uint64_t n,
                         const double* box6, uint64_t* keys, void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_computeKeys: ctx is null");
    if (n == 0) return CS_OK;
    if (!x || !y || !z || !box6 || !keys) return fail(ctx, CS_ERR_INVALID_ARG, "cs_computeKeys: null pointer");
    CS_TRY(checkParticles(ctx, "cs_computeKeys", n));
    DeviceGuard g(ctx->device);
    return enqueueKeys(ctx, x, y, z, n, box6, (u64*)keys, -1, CS_CURVE_MORTON, (cudaStream_t)stream);
}

cs_status cs_computeKeysHilbert(cs_context* ctx, const double* x, const double* y, const double* z, uint64_t n,
                                const double* box6, uint64_t* keys, void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_computeKeysHilbert: ctx is null");
    if (n == 0) return CS_OK;
    if (!x || !y || !z || !box6 || !keys) return fail(ctx, CS_ERR_INVALID_ARG, "cs_computeKeysHilbert: null pointer");
    CS_TRY(checkParticles(ctx, "cs_computeKeysHilbert", n));
    DeviceGuard g(ctx->device);
    return enqueueKeys(ctx, x, y, z, n, box6, (u64*)keys, -1, CS_CURVE_HILBERT, (cudaStream_t)stream);
}

cs_status cs_setCurve(cs_context* ctx, int curve)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_setCurve: ctx is null");
    if (curve != CS_CURVE_MORTON && curve != CS_CURVE_HILBERT)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_setCurve: unknown curve %d", curve);
    ctx->curve = curve;
    return CS_OK;
}

cs_status cs_sortKeys(cs_context* ctx, uint64_t* keys, uint32_t* perm, uint64_t n, void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_sortKeys: ctx is null");
    if (n == 0) return CS_OK;
    if (!keys || !perm) return fail(ctx, CS_ERR_INVALID_ARG, "cs_sortKeys: null pointer");
    CS_TRY(checkParticles(ctx, "cs_sortKeys", n));
    DeviceGuard g(ctx->device);
    return enqueueSort(ctx, (u64*)keys, perm, n, false, sortDecidePlan(ctx), (cudaStream_t)stream);
}

cs_status cs_buildLeaves(cs_context* ctx, const uint64_t* sortedKeys, uint64_t n, uint32_t bucketSize,
                         const uint64_t* prevLeaves, uint32_t prevNumLeaves, uint32_t maxRounds, uint64_t* leaves,
                         uint32_t* counts, uint32_t leafCapacity, uint32_t* numLeaves, uint32_t* rounds, void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_buildLeaves: ctx is null");
    if ((!sortedKeys && n) || !leaves || !counts || !numLeaves || !rounds)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildLeaves: null pointer");
    if (bucketSize == 0) return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildLeaves: bucketSize == 0");
    if (leafCapacity == 0) return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildLeaves: leafCapacity == 0");
    if (prevLeaves && prevNumLeaves == 0)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildLeaves: prevLeaves given with prevNumLeaves == 0");
    CS_TRY(checkParticles(ctx, "cs_buildLeaves", n));
    if (((uintptr_t)sortedKeys) & 15u)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildLeaves: sortedKeys must be 16-byte aligned");
    if (prevLeaves && (prevNumLeaves > ctx->maxLeaves || prevNumLeaves > leafCapacity))
        return fail(ctx, CS_ERR_CAPACITY, "cs_buildLeaves: prevNumLeaves exceeds the leaf capacity");
    DeviceGuard g(ctx->device);
    cudaStream_t s = (cudaStream_t)stream;
    CS_TRY(enqueueLeaves(ctx, (const u64*)sortedKeys, n, bucketSize, (const u64*)prevLeaves, prevNumLeaves, maxRounds,
                         (u64*)leaves, counts, leafCapacity, kL, s));
    CS_TRY(readCtrl(ctx, s));
    const DeviceCtrl& c = ctx->hostCtrl->c;
    *rounds = c.rounds;
    *numLeaves = (c.status == CS_OK || c.status == CS_ERR_NOT_CONVERGED) ? c.nl[c.rounds] : 0;
    return statusFromCtrl(ctx, "cs_buildLeaves");
}

cs_status cs_setSortMode(cs_context* ctx, int mode)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_setSortMode: ctx is null");
    if (mode != CS_SORT_AUTO && mode != CS_SORT_PLAIN && mode != CS_SORT_DEFAULT && mode != CS_SORT_SHORT && mode != CS_SORT_TINY)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_setSortMode: unknown mode %d", mode);
    ctx->sortMode = mode;
    ctx->autoPlainLeft = 0;
    for (int p = 0; p < kPlanDefault; ++p) {
        ctx->planLeft[p] = 0;
        ctx->planHold[p] = kShortHold;
    }
    ctx->hostCtrl->sortRedoHint = 0;
    return CS_OK;
}

int cs_sortPasses(const cs_context* ctx)
{
    if (!ctx) return 0;
    return sortPeekPlainPasses(ctx);
}

cs_status cs_setLeafMode(cs_context* ctx, int mode)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_setLeafMode: ctx is null");
    if (mode != CS_LEAVES_AUTO && mode != CS_LEAVES_ITERATIVE)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_setLeafMode: unknown mode %d", mode);
    ctx->leafMode = mode;
    return CS_OK;
}

cs_status cs_linkOctree(cs_context* ctx, const uint64_t* leaves, uint32_t numLeaves, uint64_t* prefixes,
                        uint32_t* levels, uint32_t* childOffsets, uint32_t* parents, uint32_t* levelRange,
                        uint32_t* leafToNode, uint32_t* nodeToLeaf, uint32_t nodeCapacity, uint32_t* numNodes,
                        void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_linkOctree: ctx is null");
    if (!leaves || !prefixes || !childOffsets || !levelRange || !numNodes)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_linkOctree: null pointer");
    if (numLeaves == 0) return fail(ctx, CS_ERR_INVALID_ARG, "cs_linkOctree: numLeaves == 0");
    if ((numLeaves - 1) % 7 != 0)
        return fail(ctx, CS_ERR_NOT_CORNERSTONE, "cs_linkOctree: (numLeaves - 1) mod 7 != 0 (PAPER.md:146)");
    if (numLeaves > ctx->maxLeaves) return fail(ctx, CS_ERR_CAPACITY, "cs_linkOctree: numLeaves exceeds maxLeaves");
    if (numLeaves + (numLeaves - 1) / 7 > nodeCapacity)
        return fail(ctx, CS_ERR_CAPACITY, "cs_linkOctree: nodeCapacity too small");
    DeviceGuard g(ctx->device);
    cudaStream_t s = (cudaStream_t)stream;
    CS_CUDA(ctx, cudaMemsetAsync(&ctx->ctrl->status, 0, sizeof(u32), s));
    CS_TRY(enqueueLink(ctx, (const u64*)leaves, nullptr, numLeaves, numLeaves, (u64*)prefixes, levels, childOffsets,
                       parents, levelRange, leafToNode, nodeToLeaf, nodeCapacity, nullptr, nullptr, nullptr, s));
    CS_TRY(readCtrl(ctx, s));
    *numNodes = ctx->hostCtrl->c.status == CS_OK ? ctx->hostCtrl->c.numNodes : 0;
    return statusFromCtrl(ctx, "cs_linkOctree");
}

cs_status cs_nodeCounts(cs_context* ctx, const uint64_t* sortedKeys, uint64_t n, const uint64_t* prefixes,
                        uint32_t numNodes, const uint32_t* leafCounts, const uint32_t* nodeToLeaf, uint32_t numLeaves,
                        uint32_t* nodeFirst, uint32_t* nodeCount, void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_nodeCounts: ctx is null");
    if (numNodes == 0) return CS_OK;
    if ((!sortedKeys && n) || !prefixes || !nodeFirst || !nodeCount)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_nodeCounts: null pointer");
    if ((leafCounts == nullptr) != (nodeToLeaf == nullptr))
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_nodeCounts: leafCounts and nodeToLeaf must be given together");
    CS_TRY(checkParticles(ctx, "cs_nodeCounts", n));
    if (leafCounts && numLeaves > ctx->maxLeaves)
        return fail(ctx, CS_ERR_CAPACITY, "cs_nodeCounts: numLeaves exceeds maxLeaves");
    DeviceGuard g(ctx->device);
    cudaStream_t s = (cudaStream_t)stream;
    const u32* leafOffsets = nullptr;
    if (leafCounts) {
        CS_TRY(enqueueExclusiveScan(ctx, leafCounts, ctx->leafOffFinal, numLeaves, s));
        leafOffsets = ctx->leafOffFinal;
    }
    return enqueueNodeCounts(ctx, (const u64*)sortedKeys, n, (const u64*)prefixes, nullptr, numNodes, numNodes,
                             leafOffsets, nodeToLeaf, nodeFirst, nodeCount, s);
}

cs_status cs_setGraphLimit(cs_context* ctx, uint64_t maxParticles)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_setGraphLimit: ctx is null");
    ctx->graphMaxParticles = maxParticles;
    return CS_OK;
}

cs_status cs_buildOctree(cs_context* ctx, const double* x, const double* y, const double* z, uint64_t n,
                         uint32_t bucketSize, const uint64_t* prevLeaves, uint32_t prevNumLeaves, uint32_t maxRounds,
                         const cs_octree_buffers* b, cs_octree_sizes* sizes, void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_buildOctree: ctx is null");
    if (!x || !y || !z || !b || !sizes) return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildOctree: null pointer");
    if (!b->box6 || !b->keys || !b->perm || !b->leaves || !b->counts || !b->prefixes || !b->childOffsets ||
        !b->levelRange || !b->nodeToLeaf || !b->nodeFirst || !b->nodeCount)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildOctree: a required output buffer is null");
    if (n == 0) return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildOctree: n == 0");
    if (bucketSize == 0) return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildOctree: bucketSize == 0");
    if (b->leafCapacity == 0 || b->nodeCapacity == 0)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildOctree: zero capacity");
    if (prevLeaves && prevNumLeaves == 0)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildOctree: prevLeaves given with prevNumLeaves == 0");
    CS_TRY(checkParticles(ctx, "cs_buildOctree", n));
    if (((uintptr_t)b->keys) & 15u)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildOctree: buffers->keys must be 16-byte aligned");
    if (prevLeaves && (prevNumLeaves > ctx->maxLeaves || prevNumLeaves > b->leafCapacity))
        return fail(ctx, CS_ERR_CAPACITY, "cs_buildOctree: prevNumLeaves exceeds the leaf capacity");
    DeviceGuard g(ctx->device);
    cudaStream_t s = (cudaStream_t)stream;
    const int plan = sortDecidePlan(ctx);
    bool replayed = false;
    if (!ctx->profiling && n <= ctx->graphMaxParticles) {
        // small inputs are bound by launch overhead: the whole call is one CUDA graph, captured when first seen with
        // these arguments and replayed while they stay the same (a time-stepping caller passes the same buffers)
        BuildGraphKey key;
        memset(&key, 0, sizeof(key));
        key.x = x; key.y = y; key.z = z; key.n = n; key.bucket = bucketSize; key.prevNumLeaves = prevNumLeaves;
        key.maxRounds = maxRounds; key.prevLeaves = prevLeaves; key.buffers = *b; key.plain = plan;
        key.curve = ctx->curve; key.leafMode = ctx->leafMode; key.stream = s;
        const bool known = ctx->buildGraph && memcmp(&key, &ctx->buildGraphKey, sizeof(key)) == 0;
        if (!known) {
            // capture on the second call in a row with the same arguments: a one-off call is cheaper enqueued directly
            if (ctx->buildGraphSeen && memcmp(&key, &ctx->buildGraphCandidate, sizeof(key)) == 0) {
                CS_TRY(captureBuild(ctx, x, y, z, n, bucketSize, prevLeaves, prevNumLeaves, maxRounds, b, plan));
                if (ctx->buildGraph) memcpy(&ctx->buildGraphKey, &key, sizeof(key));
            } else {
                memcpy(&ctx->buildGraphCandidate, &key, sizeof(key));
                ctx->buildGraphSeen = true;
            }
        }
        if (ctx->buildGraph && memcmp(&key, &ctx->buildGraphKey, sizeof(key)) == 0) {
            const u32 first = reserveEpochs(ctx, ctx->buildGraphEpochs ? ctx->buildGraphEpochs : 1u, s);
            ctx->hostCtrl->epochBase = first - 1u;
            CS_CUDA(ctx, cudaGraphLaunch(ctx->buildGraph, s));
            ctx->launches += ctx->buildGraphLaunches;
            CS_CUDA(ctx, cudaStreamSynchronize(s));
            replayed = true;
        }
    }
    if (!replayed) {
        CS_TRY(enqueueBuild(ctx, x, y, z, n, bucketSize, prevLeaves, prevNumLeaves, maxRounds, b, plan, s));
        CS_CUDA(ctx, cudaStreamSynchronize(s));
    }
    sortPlanOutcome(ctx, plan, plan != kPlanPlain && ctx->hostCtrl->sortRedo != 0);   // deep clustering: the next plan for a while
    ctx->hostCtrl->sortRedoHint = 0;
    const DeviceCtrl& c = ctx->hostCtrl->c;
    sizes->rounds = c.rounds;
    sizes->converged = c.converged;
    const bool ok = (c.status == CS_OK || c.status == CS_ERR_NOT_CONVERGED);
    sizes->numLeaves = ok ? c.numLeaves : 0;
    sizes->numNodes = ok ? c.numNodes : 0;
    return statusFromCtrl(ctx, "cs_buildOctree");
}

cs_status cs_buildOctreeHost(cs_context* ctx, const double* x, const double* y, const double* z, uint64_t n,
                             uint32_t bucketSize, const cs_octree_buffers* h, cs_octree_sizes* sizes, void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_buildOctreeHost: ctx is null");
    if (!x || !y || !z || !h || !sizes) return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildOctreeHost: null pointer");
    if (n == 0) return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildOctreeHost: n == 0");
    CS_TRY(checkParticles(ctx, "cs_buildOctreeHost", n));
    DeviceGuard g(ctx->device);
    cudaStream_t s = (cudaStream_t)stream;
    // context-owned device staging: sized once for the context's capacities
    const size_t np = ctx->maxParticles, nlc = ctx->maxLeaves, nnc = ctx->maxNodes;
    auto up = [](size_t v) { return (v + 255) / 256 * 256; };
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o = up(o + bytes); return at; };
    const size_t oX = take(np * 8), oY = take(np * 8), oZ = take(np * 8), oBox = take(64 + 8 * 64), oKeys = take(np * 8),
                 oPerm = take(np * 4), oLeaves = take((nlc + 1) * 8), oCounts = take(nlc * 4), oPre = take(nnc * 8),
                 oLev = take(nnc * 4), oCO = take(nnc * 4), oPar = take(nnc * 4), oLR = take(256),
                 oL2N = take(nlc * 4), oN2L = take(nnc * 4), oNF = take(nnc * 4), oNC = take(nnc * 4);
    if (!ctx->hostPathSlab) {
        CS_CUDA(ctx, cudaMalloc((void**)&ctx->hostPathSlab, o));
        ctx->hostPathBytes = o;
        CS_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->copyStream, cudaStreamNonBlocking));
        for (cudaEvent_t& e : ctx->copyEvents) CS_CUDA(ctx, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    }
    char* d = ctx->hostPathSlab;
    double* dx = (double*)(d + oX); double* dy = (double*)(d + oY); double* dz = (double*)(d + oZ);
    double* chunkBoxes = (double*)(d + oBox) + 8;            // 8 doubles per chunk, behind box6
    // Large inputs: the upload runs on a second stream in kChunks pieces, and the box of every piece is reduced on
    // `stream` as soon as it has arrived (exact min / max: the fold of the pieces' boxes is the box of the set), so the
    // box stage hides under the upload.  Everything after it needs the whole box.
    constexpr int kChunks = 8;
    const bool chunked = n > ctx->graphMaxParticles && n >= (1u << 20);
    if (chunked) {
        const uint64_t per = ((n + kChunks - 1) / kChunks + 511) / 512 * 512;
        CS_CUDA(ctx, cudaEventRecord(ctx->copyEvents[kChunks], s));          // the staging buffers are free once `stream` got here
        CS_CUDA(ctx, cudaStreamWaitEvent(ctx->copyStream, ctx->copyEvents[kChunks], 0));
        int used = 0;
        for (int c = 0; c < kChunks; ++c) {
            const uint64_t a = (uint64_t)c * per;
            if (a >= n) break;
            const uint64_t cnt = n - a < per ? n - a : per;
            CS_CUDA(ctx, cudaMemcpyAsync(dx + a, x + a, cnt * 8, cudaMemcpyHostToDevice, ctx->copyStream));
            CS_CUDA(ctx, cudaMemcpyAsync(dy + a, y + a, cnt * 8, cudaMemcpyHostToDevice, ctx->copyStream));
            CS_CUDA(ctx, cudaMemcpyAsync(dz + a, z + a, cnt * 8, cudaMemcpyHostToDevice, ctx->copyStream));
            CS_CUDA(ctx, cudaEventRecord(ctx->copyEvents[c], ctx->copyStream));
            CS_CUDA(ctx, cudaStreamWaitEvent(s, ctx->copyEvents[c], 0));
            CS_TRY(enqueueBox(ctx, dx + a, dy + a, dz + a, cnt, chunkBoxes + 8 * c, s));
            ++used;
        }
        CS_TRY(enqueueBoxFold(ctx, chunkBoxes, used, (double*)(d + oBox), s));
    } else {
        CS_CUDA(ctx, cudaMemcpyAsync(dx, x, n * 8, cudaMemcpyHostToDevice, s));
        CS_CUDA(ctx, cudaMemcpyAsync(dy, y, n * 8, cudaMemcpyHostToDevice, s));
        CS_CUDA(ctx, cudaMemcpyAsync(dz, z, n * 8, cudaMemcpyHostToDevice, s));
    }
    cs_octree_buffers b{};
    b.box6 = (double*)(d + oBox); b.keys = (uint64_t*)(d + oKeys); b.perm = (uint32_t*)(d + oPerm);
    b.leaves = (uint64_t*)(d + oLeaves); b.counts = (uint32_t*)(d + oCounts); b.prefixes = (uint64_t*)(d + oPre);
    b.levels = (uint32_t*)(d + oLev); b.childOffsets = (uint32_t*)(d + oCO); b.parents = (uint32_t*)(d + oPar);
    b.levelRange = (uint32_t*)(d + oLR); b.leafToNode = (uint32_t*)(d + oL2N); b.nodeToLeaf = (uint32_t*)(d + oN2L);
    b.nodeFirst = (uint32_t*)(d + oNF); b.nodeCount = (uint32_t*)(d + oNC);
    b.leafCapacity = ctx->maxLeaves; b.nodeCapacity = ctx->maxNodes;
    ctx->boxReady = chunked;
    cs_status st = cs_buildOctree(ctx, dx, dy, dz, n, bucketSize, nullptr, 0, 0, &b, sizes, stream);
    ctx->boxReady = false;
    if (st != CS_OK) return st;
    const size_t nl = sizes->numLeaves, nn = sizes->numNodes;
    if ((h->leaves || h->counts || h->leafToNode) && nl > h->leafCapacity)
        return fail(ctx, CS_ERR_CAPACITY, "cs_buildOctreeHost: host leafCapacity too small");
    if ((h->prefixes || h->childOffsets) && nn > h->nodeCapacity)
        return fail(ctx, CS_ERR_CAPACITY, "cs_buildOctreeHost: host nodeCapacity too small");
    auto back = [&](void* dst, const void* src, size_t bytes) -> cudaError_t {
        if (!dst || bytes == 0) return cudaSuccess;
        return cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, s);
    };
    CS_CUDA(ctx, back(h->box6, b.box6, 48));
    CS_CUDA(ctx, back(h->keys, b.keys, n * 8));
    CS_CUDA(ctx, back(h->perm, b.perm, n * 4));
    CS_CUDA(ctx, back(h->leaves, b.leaves, (nl + 1) * 8));
    CS_CUDA(ctx, back(h->counts, b.counts, nl * 4));
    CS_CUDA(ctx, back(h->prefixes, b.prefixes, nn * 8));
    CS_CUDA(ctx, back(h->levels, b.levels, nn * 4));
    CS_CUDA(ctx, back(h->childOffsets, b.childOffsets, nn * 4));
    CS_CUDA(ctx, back(h->parents, b.parents, nn * 4));
    CS_CUDA(ctx, back(h->levelRange, b.levelRange, CS_NUM_LEVEL_OFFSETS * 4));
    CS_CUDA(ctx, back(h->leafToNode, b.leafToNode, nl * 4));
    CS_CUDA(ctx, back(h->nodeToLeaf, b.nodeToLeaf, nn * 4));
    CS_CUDA(ctx, back(h->nodeFirst, b.nodeFirst, nn * 4));
    CS_CUDA(ctx, back(h->nodeCount, b.nodeCount, nn * 4));
    CS_CUDA(ctx, cudaStreamSynchronize(s));
    return CS_OK;
}

// ---- the distributed build of Sec. 6, one rank's calls (cs_global.cu) ---------------------------------------------------

cs_status cs_countLeaves(cs_context* ctx, const uint64_t* sortedKeys, uint64_t n, const uint64_t* leaves, uint32_t numLeaves,
                         uint32_t* counts, void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_countLeaves: ctx is null");
    if ((!sortedKeys && n) || !leaves || !counts) return fail(ctx, CS_ERR_INVALID_ARG, "cs_countLeaves: null pointer");
    if (numLeaves == 0) return fail(ctx, CS_ERR_INVALID_ARG, "cs_countLeaves: numLeaves == 0");
    CS_TRY(checkParticles(ctx, "cs_countLeaves", n));
    if (numLeaves > ctx->maxLeaves) return fail(ctx, CS_ERR_CAPACITY, "cs_countLeaves: numLeaves exceeds maxLeaves");
    DeviceGuard g(ctx->device);
    return enqueueCountLeaves(ctx, (const u64*)sortedKeys, n, (const u64*)leaves, numLeaves, counts, (cudaStream_t)stream);
}

cs_status cs_rebalance(cs_context* ctx, const uint64_t* leaves, const uint32_t* counts, uint32_t numLeaves,
                       uint32_t bucketSize, uint64_t* newLeaves, uint32_t leafCapacity, uint32_t* newNumLeaves,
                       uint32_t* changed, void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_rebalance: ctx is null");
    if (!leaves || !counts || !newLeaves || !newNumLeaves || !changed)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_rebalance: null pointer");
    if (numLeaves == 0) return fail(ctx, CS_ERR_INVALID_ARG, "cs_rebalance: numLeaves == 0");
    if (bucketSize == 0) return fail(ctx, CS_ERR_INVALID_ARG, "cs_rebalance: bucketSize == 0");
    if (newLeaves == leaves) return fail(ctx, CS_ERR_INVALID_ARG, "cs_rebalance: in place is not supported");
    if (numLeaves > ctx->maxLeaves) return fail(ctx, CS_ERR_CAPACITY, "cs_rebalance: numLeaves exceeds maxLeaves");
    DeviceGuard g(ctx->device);
    cudaStream_t s = (cudaStream_t)stream;
    const u32 cap = leafCapacity < ctx->maxLeaves ? leafCapacity : ctx->maxLeaves;
    CS_TRY(enqueueRebalance(ctx, (const u64*)leaves, counts, numLeaves, bucketSize, kL, (u64*)newLeaves, cap, s));
    CS_TRY(readCtrl(ctx, s));
    const DeviceCtrl& c = ctx->hostCtrl->c;
    *newNumLeaves = c.status == CS_OK ? c.numLeaves : 0;
    *changed = c.status == CS_OK ? (c.converged ? 0u : 1u) : 0u;
    return statusFromCtrl(ctx, "cs_rebalance");
}

cs_status cs_partitionLeaves(cs_context* ctx, const uint32_t* counts, uint32_t numLeaves, uint32_t numRanks,
                             uint32_t* bounds, void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_partitionLeaves: ctx is null");
    if (!counts || !bounds) return fail(ctx, CS_ERR_INVALID_ARG, "cs_partitionLeaves: null pointer");
    if (numLeaves == 0 || numRanks == 0) return fail(ctx, CS_ERR_INVALID_ARG, "cs_partitionLeaves: numLeaves or numRanks is 0");
    if (numLeaves > ctx->maxLeaves) return fail(ctx, CS_ERR_CAPACITY, "cs_partitionLeaves: numLeaves exceeds maxLeaves");
    DeviceGuard g(ctx->device);
    return enqueuePartition(ctx, counts, numLeaves, numRanks, bounds, (cudaStream_t)stream);
}

cs_status cs_nodeCountsFromLeaves(cs_context* ctx, const uint64_t* leaves, const uint32_t* leafCounts, uint32_t numLeaves,
                                  const uint64_t* prefixes, uint32_t numNodes, uint32_t* nodeFirst, uint32_t* nodeCount,
                                  void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_nodeCountsFromLeaves: ctx is null");
    if (numNodes == 0) return CS_OK;
    if (!leaves || !leafCounts || !prefixes || !nodeFirst || !nodeCount)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_nodeCountsFromLeaves: null pointer");
    if (numLeaves == 0) return fail(ctx, CS_ERR_INVALID_ARG, "cs_nodeCountsFromLeaves: numLeaves == 0");
    if (numLeaves > ctx->maxLeaves) return fail(ctx, CS_ERR_CAPACITY, "cs_nodeCountsFromLeaves: numLeaves exceeds maxLeaves");
    DeviceGuard g(ctx->device);
    return enqueueNodeCountsFromLeaves(ctx, (const u64*)leaves, leafCounts, numLeaves, (const u64*)prefixes, numNodes,
                                       nodeFirst, nodeCount, (cudaStream_t)stream);
}

cs_status cs_gatherParticles(cs_context* ctx, const double* x, const double* y, const double* z, const uint32_t* perm,
                             uint64_t n, double* xs, double* ys, double* zs, void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_gatherParticles: ctx is null");
    if (n == 0) return CS_OK;
    if (!x || !y || !z || !perm || !xs || !ys || !zs) return fail(ctx, CS_ERR_INVALID_ARG, "cs_gatherParticles: null pointer");
    if (xs == x || ys == y || zs == z) return fail(ctx, CS_ERR_INVALID_ARG, "cs_gatherParticles: in place is not supported");
    if (n >= (1ull << 32)) return fail(ctx, CS_ERR_INVALID_ARG, "cs_gatherParticles: n >= 2^32");
    DeviceGuard g(ctx->device);
    return enqueueGather(ctx, x, y, z, perm, n, xs, ys, zs, (cudaStream_t)stream);
}

static cs_status nodeGeometryCall(cs_context* ctx, const char* fn, const uint64_t* prefixes, uint32_t numNodes,
                                  const double* box6, int curve, double* centers, double* halfSizes, void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "%s: ctx is null", fn);
    if (numNodes == 0) return CS_OK;
    if (!prefixes || !box6 || !centers || !halfSizes) return fail(ctx, CS_ERR_INVALID_ARG, "%s: null pointer", fn);
    DeviceGuard g(ctx->device);
    return enqueueNodeGeometry(ctx, (const u64*)prefixes, numNodes, box6, curve, centers, halfSizes, (cudaStream_t)stream);
}

cs_status cs_nodeGeometry(cs_context* ctx, const uint64_t* prefixes, uint32_t numNodes, const double* box6,
                          double* centers, double* halfSizes, void* stream)
{
    return nodeGeometryCall(ctx, "cs_nodeGeometry", prefixes, numNodes, box6, CS_CURVE_MORTON, centers, halfSizes, stream);
}

cs_status cs_nodeGeometryHilbert(cs_context* ctx, const uint64_t* prefixes, uint32_t numNodes, const double* box6,
                                 double* centers, double* halfSizes, void* stream)
{
    return nodeGeometryCall(ctx, "cs_nodeGeometryHilbert", prefixes, numNodes, box6, CS_CURVE_HILBERT, centers, halfSizes,
                            stream);
}

cs_status cs_nodeMassCenters(cs_context* ctx, const double* xs, const double* ys, const double* zs,
                             const uint32_t* nodeFirst, const uint32_t* nodeCount, const uint32_t* childOffsets,
                             const double* centers, const uint32_t* levelRange, uint32_t numNodes, double* com,
                             void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_nodeMassCenters: ctx is null");
    if (numNodes == 0) return CS_OK;
    if (!xs || !ys || !zs || !nodeFirst || !nodeCount || !childOffsets || !centers || !levelRange || !com)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_nodeMassCenters: null pointer");
    DeviceGuard g(ctx->device);
    return enqueueMassCenters(ctx, xs, ys, zs, nodeFirst, nodeCount, childOffsets, centers, levelRange, numNodes, com,
                              (cudaStream_t)stream);
}

cs_status cs_macMinDistance(cs_context* ctx, const double* centers, const double* halfSizes, uint32_t numNodes,
                            const double* focus6, double theta, uint8_t* pass, void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_macMinDistance: ctx is null");
    if (numNodes == 0) return CS_OK;
    if (!centers || !halfSizes || !focus6 || !pass) return fail(ctx, CS_ERR_INVALID_ARG, "cs_macMinDistance: null pointer");
    if (!(theta > 0.0)) return fail(ctx, CS_ERR_INVALID_ARG, "cs_macMinDistance: theta must be positive");
    DeviceGuard g(ctx->device);
    return enqueueMac(ctx, centers, halfSizes, numNodes, focus6, theta, pass, (cudaStream_t)stream);
}

}  // extern "C"
