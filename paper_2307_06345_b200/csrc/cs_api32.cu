// 30-bit keys, L = 10 ("reasonable choices for L are 10 or 21"): the entry points with the suffix 32.
//
// What is specific to the narrow keys is their generation (the key kernel writes the 63-bit key without its low
// 33 bits: the same quotient, scaled by 2^10 instead of 2^21) and the sort (cs_sort.cu: 8 bytes per element
// instead of 12, 4 passes).  The tree stages work on keys of 21 octal digits; a 30-bit key is the 10 leading
// digits of such a key, so the sorted keys and the leaf arrays are widened (key << 33, which also maps 8^10 to
// 8^21) into the workspace, the stages of cs_leaves*.cu / cs_link.cu run with the maximum depth set to 10, and
// their results are narrowed again.  A placeholder-bit prefix only holds a node's leading digits: it is the
// same number for the key and its widened form, and fits into 31 bits.
#include "cs_device.cuh"

using namespace cs;

namespace cs {

constexpr int kL32 = 10;
constexpr int kWiden = 3 * (kL - kL32);       // 33 bits

__global__ void __launch_bounds__(256) widenKernel(const u32* __restrict__ in, u64* __restrict__ out, u64 n)
{
    const u64 stride = (u64)gridDim.x * blockDim.x;
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) out[i] = (u64)in[i] << kWiden;
}

// count: host value, or read from the device (dCount, + extra entries) when the size is not known on the host yet
__global__ void __launch_bounds__(256) narrowKernel(const u64* __restrict__ in, u32* __restrict__ out, u32 hCount,
                                                    const u32* dCount, u32 extra, int shift, const DeviceCtrl* ctrl)
{
    if (ctrl) {
        const u32 st = ctrl->status;
        if (st == CS_ERR_CAPACITY || st == CS_ERR_NOT_CORNERSTONE) return;
    }
    const u32 count = dCount ? *dCount + extra : hCount;
    const u32 stride = gridDim.x * blockDim.x;
    for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i < count; i += stride) out[i] = (u32)(in[i] >> shift);
}

static u32 gridFor(const cs_context* ctx, u64 work)
{
    u32 g = divUp(work, 256);
    const u32 cap = (u32)ctx->numSMs * 8;
    if (g > cap) g = cap;
    return g ? g : 1;
}

// 64-bit staging of leaf arrays and prefixes, sized for the context's capacities (allocated on first use)
static cs_status wideBuffers(cs_context* ctx)
{
    if (ctx->wideSlab) return CS_OK;
    const size_t nl = (size_t)ctx->maxLeaves + 2, nn = (size_t)ctx->maxNodes + 2;
    CS_CUDA(ctx, cudaMalloc((void**)&ctx->wideSlab, (2 * nl + nn) * sizeof(u64)));
    ctx->wideLeaves = (u64*)ctx->wideSlab;
    ctx->widePrev = ctx->wideLeaves + nl;
    ctx->widePrefixes = ctx->widePrev + nl;
    return CS_OK;
}

static cs_status statusFromCtrl32(cs_context* ctx, const char* where)
{
    const u32 st = ctx->hostCtrl->c.status;
    switch (st) {
        case CS_OK: return CS_OK;
        case CS_ERR_CAPACITY: return fail(ctx, CS_ERR_CAPACITY, "%s: result exceeds the given capacity", where);
        case CS_ERR_NOT_CORNERSTONE:
            return fail(ctx, CS_ERR_NOT_CORNERSTONE, "%s: leaf array violates Eq. 2 (not a cornerstone array)", where);
        case CS_ERR_NOT_CONVERGED: return fail(ctx, CS_ERR_NOT_CONVERGED, "%s: maxRounds reached before convergence", where);
        default: return fail(ctx, CS_ERR_CUDA, "%s: unexpected device status %u", where, st);
    }
}

static cs_status checkN(cs_context* ctx, const char* fn, uint64_t n)
{
    if (n >= (1ull << 32)) return fail(ctx, CS_ERR_INVALID_ARG, "%s: n >= 2^32", fn);
    if (n > ctx->maxParticles) return fail(ctx, CS_ERR_CAPACITY, "%s: n exceeds the context's maxParticles", fn);
    return CS_OK;
}

}  // namespace cs

extern "C" {

cs_status cs_computeKeys32(cs_context* ctx, const double* x, const double* y, const double* z, uint64_t n,
                           const double* box6, int curve, uint32_t* keys, void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_computeKeys32: ctx is null");
    if (n == 0) return CS_OK;
    if (!x || !y || !z || !box6 || !keys) return fail(ctx, CS_ERR_INVALID_ARG, "cs_computeKeys32: null pointer");
    if (curve != CS_CURVE_MORTON && curve != CS_CURVE_HILBERT)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_computeKeys32: unknown curve %d", curve);
    CS_TRY(checkN(ctx, "cs_computeKeys32", n));
    DeviceGuard g(ctx->device);
    return enqueueKeys(ctx, x, y, z, n, box6, nullptr, -1, curve, (cudaStream_t)stream, keys);
}

cs_status cs_sortKeys32(cs_context* ctx, uint32_t* keys, uint32_t* perm, uint64_t n, void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_sortKeys32: ctx is null");
    if (n == 0) return CS_OK;
    if (!keys || !perm) return fail(ctx, CS_ERR_INVALID_ARG, "cs_sortKeys32: null pointer");
    CS_TRY(checkN(ctx, "cs_sortKeys32", n));
    DeviceGuard g(ctx->device);
    return enqueueSort32(ctx, keys, perm, n, (cudaStream_t)stream);
}

cs_status cs_buildLeaves32(cs_context* ctx, const uint32_t* sortedKeys, uint64_t n, uint32_t bucketSize,
                           const uint32_t* prevLeaves, uint32_t prevNumLeaves, uint32_t maxRounds, uint32_t* leaves,
                           uint32_t* counts, uint32_t leafCapacity, uint32_t* numLeaves, uint32_t* rounds, void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_buildLeaves32: ctx is null");
    if ((!sortedKeys && n) || !leaves || !counts || !numLeaves || !rounds)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildLeaves32: null pointer");
    if (bucketSize == 0 || leafCapacity == 0) return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildLeaves32: zero bucketSize / leafCapacity");
    if (prevLeaves && prevNumLeaves == 0)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildLeaves32: prevLeaves given with prevNumLeaves == 0");
    CS_TRY(checkN(ctx, "cs_buildLeaves32", n));
    if (prevLeaves && (prevNumLeaves > ctx->maxLeaves || prevNumLeaves > leafCapacity))
        return fail(ctx, CS_ERR_CAPACITY, "cs_buildLeaves32: prevNumLeaves exceeds the leaf capacity");
    DeviceGuard g(ctx->device);
    cudaStream_t s = (cudaStream_t)stream;
    CS_TRY(wideBuffers(ctx));
    const u32 cap = leafCapacity < ctx->maxLeaves ? leafCapacity : ctx->maxLeaves;
    if (n) {
        widenKernel<<<gridFor(ctx, n), 256, 0, s>>>(sortedKeys, ctx->keysAlt, n);
        CS_LAUNCH_CHECK(ctx, "widenKernel");
    }
    if (prevLeaves) {
        widenKernel<<<gridFor(ctx, (u64)prevNumLeaves + 1), 256, 0, s>>>(prevLeaves, ctx->widePrev, (u64)prevNumLeaves + 1);
        CS_LAUNCH_CHECK(ctx, "widenKernel");
    }
    CS_TRY(enqueueLeaves(ctx, ctx->keysAlt, n, bucketSize, prevLeaves ? ctx->widePrev : nullptr, prevNumLeaves, maxRounds,
                         ctx->wideLeaves, counts, cap, kL32, s));
    narrowKernel<<<gridFor(ctx, (u64)cap + 1), 256, 0, s>>>(ctx->wideLeaves, leaves, 0, &ctx->ctrl->numLeaves, 1, kWiden,
                                                            ctx->ctrl);
    CS_LAUNCH_CHECK(ctx, "narrowKernel");
    CS_TRY(readCtrl(ctx, s));
    const DeviceCtrl& c = ctx->hostCtrl->c;
    *rounds = c.rounds;
    *numLeaves = (c.status == CS_OK || c.status == CS_ERR_NOT_CONVERGED) ? c.nl[c.rounds] : 0;
    return statusFromCtrl32(ctx, "cs_buildLeaves32");
}

cs_status cs_linkOctree32(cs_context* ctx, const uint32_t* leaves, uint32_t numLeaves, uint32_t* prefixes,
                          uint32_t* levels, uint32_t* childOffsets, uint32_t* parents, uint32_t* levelRange,
                          uint32_t* leafToNode, uint32_t* nodeToLeaf, uint32_t nodeCapacity, uint32_t* numNodes,
                          void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_linkOctree32: ctx is null");
    if (!leaves || !prefixes || !childOffsets || !levelRange || !numNodes)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_linkOctree32: null pointer");
    if (numLeaves == 0) return fail(ctx, CS_ERR_INVALID_ARG, "cs_linkOctree32: numLeaves == 0");
    if ((numLeaves - 1) % 7 != 0)
        return fail(ctx, CS_ERR_NOT_CORNERSTONE, "cs_linkOctree32: (numLeaves - 1) mod 7 != 0 (PAPER.md:146)");
    if (numLeaves > ctx->maxLeaves) return fail(ctx, CS_ERR_CAPACITY, "cs_linkOctree32: numLeaves exceeds maxLeaves");
    const u32 nn = numLeaves + (numLeaves - 1) / 7;
    if (nn > nodeCapacity || nn > ctx->maxNodes) return fail(ctx, CS_ERR_CAPACITY, "cs_linkOctree32: nodeCapacity too small");
    DeviceGuard g(ctx->device);
    cudaStream_t s = (cudaStream_t)stream;
    CS_TRY(wideBuffers(ctx));
    CS_CUDA(ctx, cudaMemsetAsync(&ctx->ctrl->status, 0, sizeof(u32), s));
    widenKernel<<<gridFor(ctx, (u64)numLeaves + 1), 256, 0, s>>>(leaves, ctx->wideLeaves, (u64)numLeaves + 1);
    CS_LAUNCH_CHECK(ctx, "widenKernel");
    CS_TRY(enqueueLink(ctx, ctx->wideLeaves, nullptr, numLeaves, numLeaves, ctx->widePrefixes, levels, childOffsets, parents,
                       levelRange, leafToNode, nodeToLeaf, nodeCapacity < ctx->maxNodes ? nodeCapacity : ctx->maxNodes,
                       nullptr, nullptr, nullptr, s));
    narrowKernel<<<gridFor(ctx, nn), 256, 0, s>>>(ctx->widePrefixes, prefixes, nn, nullptr, 0, 0, ctx->ctrl);
    CS_LAUNCH_CHECK(ctx, "narrowKernel");
    CS_TRY(readCtrl(ctx, s));
    *numNodes = ctx->hostCtrl->c.status == CS_OK ? ctx->hostCtrl->c.numNodes : 0;
    return statusFromCtrl32(ctx, "cs_linkOctree32");
}

cs_status cs_buildOctree32(cs_context* ctx, const double* x, const double* y, const double* z, uint64_t n,
                           uint32_t bucketSize, const cs_octree_buffers32* b, cs_octree_sizes* sizes, void* stream)
{
    if (!ctx) return fail(nullptr, CS_ERR_INVALID_ARG, "cs_buildOctree32: ctx is null");
    if (!x || !y || !z || !b || !sizes) return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildOctree32: null pointer");
    if (!b->box6 || !b->keys || !b->perm || !b->leaves || !b->counts || !b->prefixes || !b->childOffsets ||
        !b->levelRange || !b->nodeToLeaf || !b->nodeFirst || !b->nodeCount)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildOctree32: a required output buffer is null");
    if (n == 0 || bucketSize == 0 || b->leafCapacity == 0 || b->nodeCapacity == 0)
        return fail(ctx, CS_ERR_INVALID_ARG, "cs_buildOctree32: n, bucketSize and the capacities must be positive");
    CS_TRY(checkN(ctx, "cs_buildOctree32", n));
    DeviceGuard g(ctx->device);
    cudaStream_t s = (cudaStream_t)stream;
    CS_TRY(wideBuffers(ctx));
    const u32 leafCap = b->leafCapacity < ctx->maxLeaves ? b->leafCapacity : ctx->maxLeaves;
    const u32 nodeCap = b->nodeCapacity < ctx->maxNodes ? b->nodeCapacity : ctx->maxNodes;

    CS_TRY(enqueueBox(ctx, x, y, z, n, b->box6, s));
    CS_TRY(enqueueKeys(ctx, x, y, z, n, b->box6, nullptr, -1, ctx->curve, s, b->keys));
    CS_TRY(enqueueSort32(ctx, b->keys, b->perm, n, s));
    widenKernel<<<gridFor(ctx, n), 256, 0, s>>>(b->keys, ctx->keysAlt, n);
    CS_LAUNCH_CHECK(ctx, "widenKernel");
    CS_TRY(enqueueLeaves(ctx, ctx->keysAlt, n, bucketSize, nullptr, 0, 0, ctx->wideLeaves, b->counts, leafCap, kL32, s));
    narrowKernel<<<gridFor(ctx, (u64)leafCap + 1), 256, 0, s>>>(ctx->wideLeaves, b->leaves, 0, &ctx->ctrl->numLeaves, 1,
                                                                kWiden, ctx->ctrl);
    CS_LAUNCH_CHECK(ctx, "narrowKernel");
    CS_TRY(enqueueLink(ctx, ctx->wideLeaves, &ctx->ctrl->numLeaves, 0, leafCap, ctx->widePrefixes, b->levels, b->childOffsets,
                       b->parents, b->levelRange, b->leafToNode, b->nodeToLeaf, nodeCap, ctx->leafOffFinal, b->nodeFirst,
                       b->nodeCount, s));
    narrowKernel<<<gridFor(ctx, nodeCap), 256, 0, s>>>(ctx->widePrefixes, b->prefixes, 0, &ctx->ctrl->numNodes, 0, 0, ctx->ctrl);
    CS_LAUNCH_CHECK(ctx, "narrowKernel");
    CS_TRY(readCtrl(ctx, s));
    const DeviceCtrl& c = ctx->hostCtrl->c;
    sizes->rounds = c.rounds;
    sizes->converged = c.converged;
    const bool ok = c.status == CS_OK;
    sizes->numLeaves = ok ? c.numLeaves : 0;
    sizes->numNodes = ok ? c.numNodes : 0;
    return statusFromCtrl32(ctx, "cs_buildOctree32");
}

}  // extern "C"
