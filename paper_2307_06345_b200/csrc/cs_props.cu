// Node properties on the linked octree: the particles in
// SFC order, the nodes' cells, centres of mass by an upward pass, the minimum-distance MAC of Eq. 12.
// Readings A25-A27 of DESIGN.md fix the operation order; every floating-point operation below is an
// explicitly rounded intrinsic (no FMA contraction), so the results equal the oracle's bit for bit.
#include <cooperative_groups.h>

#include "cs_device.cuh"

namespace cg = cooperative_groups;

namespace cs {

constexpr int kPropBlock = 256;

// ---- particles in SFC order: out[j] = in[perm[j]] for the three coordinate arrays --------------------------
// perm is read once, coalesced; the three gathers of a particle are issued together.
__global__ void __launch_bounds__(kPropBlock)
    gatherKernel(const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
                 const u32* __restrict__ perm, u64 n, double* __restrict__ xs, double* __restrict__ ys,
                 double* __restrict__ zs)
{
    const u64 stride = (u64)gridDim.x * kPropBlock;
    for (u64 j = (u64)blockIdx.x * kPropBlock + threadIdx.x; j < n; j += stride) {
        const u32 i = ldStreamU32(perm + j);
        const double a = __ldg(x + i), b = __ldg(y + i), c = __ldg(z + i);
        xs[j] = a;
        ys[j] = b;
        zs[j] = c;
    }
}

// ---- A25: cell of a node from its placeholder-bit key -------------------------------------------------------
// every third bit of v, starting at bit 0, packed into the low bits (inverse of the key interleave)
__device__ __forceinline__ u32 compact3(u64 v)
{
    v &= 0x1249249249249249ull;
    v = (v | (v >> 2)) & 0x10C30C30C30C30C3ull;
    v = (v | (v >> 4)) & 0x100F00F00F00F00Full;
    v = (v | (v >> 8)) & 0x001F0000FF0000FFull;
    v = (v | (v >> 16)) & 0x001F00000000FFFFull;
    v = (v | (v >> 32)) & 0x00000000001FFFFFull;
    return (u32)v;
}

// HILBERT (reading A28): the prefix holds Hilbert digits; the curve is walked backwards from the root, one table
// look-up per level: inv[state][w] = octant (4x + 2y + z) | next state << 3, start state (e = 0, d = 0) = 0.
template <bool HILBERT>
__global__ void __launch_bounds__(kPropBlock)
    nodeGeometryKernel(const u64* __restrict__ prefixes, u32 n, const double* __restrict__ box6,
                       const unsigned char* __restrict__ inv, double* __restrict__ centers, double* __restrict__ halfSizes)
{
    __shared__ unsigned char sInv[HILBERT ? 24 * 8 : 1];
    if (HILBERT) {
        for (int i = threadIdx.x; i < 24 * 8; i += kPropBlock) sInv[i] = inv[i];
        __syncthreads();
    }
    const u32 stride = gridDim.x * kPropBlock;
    for (u32 i = blockIdx.x * kPropBlock + threadIdx.x; i < n; i += stride) {
        const u64 p = prefixes[i];
        const int level = (63 - __clzll((long long)p)) / 3;
        const u64 digits = p ^ (1ull << (3 * level));
        u32 g[3];
        if (HILBERT) {
            u32 state = 0;
            g[0] = g[1] = g[2] = 0;
            for (int l = level - 1; l >= 0; --l) {
                const u32 ent = sInv[state * 8 + ((u32)(digits >> (3 * l)) & 7u)];
                state = ent >> 3;
                g[0] = (g[0] << 1) | ((ent >> 2) & 1u);
                g[1] = (g[1] << 1) | ((ent >> 1) & 1u);
                g[2] = (g[2] << 1) | (ent & 1u);
            }
        } else {
            g[0] = compact3(digits >> 2); g[1] = compact3(digits >> 1); g[2] = compact3(digits);   // digit = 4x + 2y + z (A3)
        }
        const double cells = (double)(1ull << level);
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const double lo = box6[2 * d], e = __dsub_rn(box6[2 * d + 1], box6[2 * d]);
            const double h = __ddiv_rn(e, cells);
            centers[(size_t)d * n + i] = __dadd_rn(lo, __dmul_rn(__dadd_rn((double)g[d], 0.5), h));
            halfSizes[(size_t)d * n + i] = __dmul_rn(0.5, h);
        }
    }
}

// ---- A26: centres of mass by an upward pass ------------------------------------------------------------------------
// Leaves sum their particles in sorted order, internal nodes their 8 children in order: the oracle's order.  Two
// launches: the leaves of ALL levels at once (they depend on the particles only: 7/8 of the nodes and all of the
// particle traffic), then the internal nodes level by level from the deepest to the root inside one cooperative
// launch with a grid barrier between levels (the level sizes stay on the device).
// four doubles of one 32-byte sector in one request (p 32-byte aligned; sm_100: 256-bit global loads)
__device__ __forceinline__ void ldSector(const double* p, double (&v)[4])
{
    asm volatile("ld.global.nc.L1::no_allocate.v4.f64 {%0, %1, %2, %3}, [%4];"
                 : "=d"(v[0]), "=d"(v[1]), "=d"(v[2]), "=d"(v[3])
                 : "l"(p));
}

__device__ __forceinline__ void leafCenter(const double* __restrict__ xs, const double* __restrict__ ys,
                                           const double* __restrict__ zs, const double* __restrict__ centers, u32 first,
                                           u32 count, u32 i, u32 n, bool sectors, double* __restrict__ com)
{
    if (count == 0) {
#pragma unroll
        for (int d = 0; d < 3; ++d) com[(size_t)d * n + i] = centers[(size_t)d * n + i];
        return;
    }
    // Neighbouring threads read ranges some 150 bytes apart, so every 8-byte load of a warp is its own L1 request; the
    // middle of the range is therefore read 32 bytes (one sector, 4 coordinates) per request.  The additions stay in
    // sorted order: three independent chains (x, y, z) that overlap.
    double sx = 0.0, sy = 0.0, sz = 0.0;
    u32 j = first;
    const u32 end = first + count;
    for (; j < end && (j & 3u); ++j) {
        sx = __dadd_rn(sx, xs[j]);
        sy = __dadd_rn(sy, ys[j]);
        sz = __dadd_rn(sz, zs[j]);
    }
    for (; sectors && j + 4 <= end; j += 4) {
        double a[4], b[4], c[4];
        ldSector(xs + j, a);
        ldSector(ys + j, b);
        ldSector(zs + j, c);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            sx = __dadd_rn(sx, a[k]);
            sy = __dadd_rn(sy, b[k]);
            sz = __dadd_rn(sz, c[k]);
        }
    }
    for (; j < end; ++j) {
        sx = __dadd_rn(sx, xs[j]);
        sy = __dadd_rn(sy, ys[j]);
        sz = __dadd_rn(sz, zs[j]);
    }
    const double c = (double)count;
    com[i] = __ddiv_rn(sx, c);
    com[(size_t)n + i] = __ddiv_rn(sy, c);
    com[2 * (size_t)n + i] = __ddiv_rn(sz, c);
}

__global__ void __launch_bounds__(kPropBlock)
    massCentersLeafKernel(const double* __restrict__ xs, const double* __restrict__ ys, const double* __restrict__ zs,
                          const u32* __restrict__ nodeFirst, const u32* __restrict__ nodeCount,
                          const u32* __restrict__ childOffsets, const double* __restrict__ centers, u32 n,
                          bool sectors /*xs, ys, zs are 32-byte aligned*/, double* __restrict__ com)
{
    const u32 stride = gridDim.x * kPropBlock;
    for (u32 i = blockIdx.x * kPropBlock + threadIdx.x; i < n; i += stride)
        if (childOffsets[i] == 0) leafCenter(xs, ys, zs, centers, nodeFirst[i], nodeCount[i], i, n, sectors, com);
}

__global__ void __launch_bounds__(kPropBlock)
    massCentersUpKernel(const u32* __restrict__ nodeCount, const u32* __restrict__ childOffsets,
                        const double* __restrict__ centers, const u32* __restrict__ levelRange, u32 n, double* com)
{
    cg::grid_group grid = cg::this_grid();
    const u32 stride = gridDim.x * kPropBlock;
    int deepest = kL;
    while (deepest > 0 && levelRange[deepest] >= n) --deepest;         // levels past the deepest start at n (A19)
    for (int level = deepest - 1; level >= 0; --level) {               // the deepest level holds leaves only
        const u32 begin = levelRange[level], end = levelRange[level + 1];
        for (u32 i = begin + blockIdx.x * kPropBlock + threadIdx.x; i < end; i += stride) {
            const u32 co = childOffsets[i];
            if (co == 0) continue;                                      // a leaf: done by the first launch
            const u32 count = nodeCount[i];
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                double r;
                if (count == 0) r = centers[(size_t)d * n + i];
                else {
                    double s = 0.0;
#pragma unroll
                    for (u32 k = 0; k < 8; ++k)
                        s = __dadd_rn(s, __dmul_rn((double)nodeCount[co + k], __ldcg(com + (size_t)d * n + co + k)));
                    r = __ddiv_rn(s, (double)count);
                }
                com[(size_t)d * n + i] = r;
            }
        }
        if (level > 0) grid.sync();
    }
}

// ---- A27: minimum-distance MAC against a focus box (Eq. 12) ------------------------------------------------------
__global__ void __launch_bounds__(kPropBlock)
    macKernel(const double* __restrict__ centers, const double* __restrict__ halfSizes, u32 n, double fx0, double fx1,
              double fy0, double fy1, double fz0, double fz1, double theta, unsigned char* __restrict__ pass)
{
    const double f0[3] = {fx0, fy0, fz0}, f1[3] = {fx1, fy1, fz1};
    const double t2 = __dmul_rn(theta, theta);
    const u32 stride = gridDim.x * kPropBlock;
    for (u32 i = blockIdx.x * kPropBlock + threadIdx.x; i < n; i += stride) {
        double r2 = 0.0, hmax = 0.0;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const double fc = __dmul_rn(0.5, __dadd_rn(f0[d], f1[d])), fh = __dmul_rn(0.5, __dsub_rn(f1[d], f0[d]));
            const double cc = centers[(size_t)d * n + i], h = halfSizes[(size_t)d * n + i];
            double gap = __dsub_rn(fabs(__dsub_rn(cc, fc)), __dadd_rn(h, fh));
            if (!(gap > 0.0)) gap = 0.0;
            r2 = __dadd_rn(r2, __dmul_rn(gap, gap));
            if (h > hmax) hmax = h;
        }
        const double l = __dmul_rn(2.0, hmax);
        pass[i] = __dmul_rn(r2, t2) > __dmul_rn(l, l) ? 1 : 0;
    }
}

static u32 gridFor(const cs_context* ctx, u64 work)
{
    u32 grid = divUp(work, kPropBlock);
    const u32 cap = (u32)ctx->numSMs * 16;
    if (grid > cap) grid = cap;
    return grid ? grid : 1;
}

cs_status enqueueGather(cs_context* ctx, const double* x, const double* y, const double* z, const u32* perm, u64 n,
                        double* xs, double* ys, double* zs, cudaStream_t s)
{
    if (n == 0) return CS_OK;
    gatherKernel<<<gridFor(ctx, n), kPropBlock, 0, s>>>(x, y, z, perm, n, xs, ys, zs);
    CS_LAUNCH_CHECK(ctx, "gatherKernel");
    return CS_OK;
}

cs_status enqueueNodeGeometry(cs_context* ctx, const u64* prefixes, u32 n, const double* box6, int curve, double* centers,
                              double* halfSizes, cudaStream_t s)
{
    if (n == 0) return CS_OK;
    if (curve == CS_CURVE_HILBERT)
        nodeGeometryKernel<true><<<gridFor(ctx, n), kPropBlock, 0, s>>>(prefixes, n, box6, ctx->hilbertInverse, centers, halfSizes);
    else
        nodeGeometryKernel<false><<<gridFor(ctx, n), kPropBlock, 0, s>>>(prefixes, n, box6, nullptr, centers, halfSizes);
    CS_LAUNCH_CHECK(ctx, "nodeGeometryKernel");
    return CS_OK;
}

cs_status enqueueMassCenters(cs_context* ctx, const double* xs, const double* ys, const double* zs, const u32* nodeFirst,
                             const u32* nodeCount, const u32* childOffsets, const double* centers, const u32* levelRange,
                             u32 n, double* com, cudaStream_t s)
{
    if (n == 0) return CS_OK;
    const bool sectors = ((((uintptr_t)xs) | ((uintptr_t)ys) | ((uintptr_t)zs)) & 31u) == 0;
    massCentersLeafKernel<<<gridFor(ctx, n), kPropBlock, 0, s>>>(xs, ys, zs, nodeFirst, nodeCount, childOffsets, centers, n,
                                                                 sectors, com);
    CS_LAUNCH_CHECK(ctx, "massCentersLeafKernel");
    if (n == 1) return CS_OK;
    int perSM = 0;
    CS_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&perSM, massCentersUpKernel, kPropBlock, 0));
    if (perSM < 1) return fail(ctx, CS_ERR_CUDA, "massCentersUpKernel does not fit on an SM");
    u32 grid = divUp(n / 8 + 1, kPropBlock);                   // the widest level of internal nodes has < n / 8 of them
    const u32 resident = (u32)perSM * (u32)ctx->numSMs;
    if (grid > resident) grid = resident;
    void* args[] = {(void*)&nodeCount, (void*)&childOffsets, (void*)&centers, (void*)&levelRange, (void*)&n, (void*)&com};
    CS_CUDA(ctx, cudaLaunchCooperativeKernel((const void*)massCentersUpKernel, dim3(grid), dim3(kPropBlock), args, 0, s));
    CS_LAUNCH_CHECK(ctx, "massCentersUpKernel");
    return CS_OK;
}

cs_status enqueueMac(cs_context* ctx, const double* centers, const double* halfSizes, u32 n, const double* focus6,
                     double theta, unsigned char* pass, cudaStream_t s)
{
    if (n == 0) return CS_OK;
    macKernel<<<gridFor(ctx, n), kPropBlock, 0, s>>>(centers, halfSizes, n, focus6[0], focus6[1], focus6[2], focus6[3],
                                                     focus6[4], focus6[5], theta, pass);
    CS_LAUNCH_CHECK(ctx, "macKernel");
    return CS_OK;
}

}  // namespace cs
