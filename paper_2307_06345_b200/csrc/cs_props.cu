// Node properties on the linked octree: the particles in
// SFC order, the nodes' cells, centres of mass by an upward pass, the minimum-distance MAC of Eq. 12.
// Readings A25-A27 of DESIGN.md fix the operation order; every floating-point operation below is an
// explicitly rounded intrinsic (no FMA contraction), so the results equal the oracle's bit for bit.
#include "cs_device.cuh"

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

__global__ void __launch_bounds__(kPropBlock)
    nodeGeometryKernel(const u64* __restrict__ prefixes, u32 n, const double* __restrict__ box6,
                       double* __restrict__ centers, double* __restrict__ halfSizes)
{
    const u32 stride = gridDim.x * kPropBlock;
    for (u32 i = blockIdx.x * kPropBlock + threadIdx.x; i < n; i += stride) {
        const u64 p = prefixes[i];
        const int level = (63 - __clzll((long long)p)) / 3;
        const u64 digits = p ^ (1ull << (3 * level));
        const u32 g[3] = {compact3(digits >> 2), compact3(digits >> 1), compact3(digits)};   // digit = 4x + 2y + z (A3)
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

// ---- A26: centres of mass, one level per launch from the deepest to the root -----------------------------------
// Leaves sum their particles in sorted order, internal nodes their 8 children in order: the oracle's order.
__global__ void __launch_bounds__(kPropBlock)
    massCentersLevelKernel(const double* __restrict__ xs, const double* __restrict__ ys, const double* __restrict__ zs,
                           const u32* __restrict__ nodeFirst, const u32* __restrict__ nodeCount,
                           const u32* __restrict__ childOffsets, const double* __restrict__ centers,
                           const u32* __restrict__ levelRange, int level, u32 n, double* __restrict__ com)
{
    const u32 begin = levelRange[level], end = levelRange[level + 1];
    const double* c[3] = {xs, ys, zs};
    const u32 stride = gridDim.x * kPropBlock;
    for (u32 i = begin + blockIdx.x * kPropBlock + threadIdx.x; i < end; i += stride) {
        const u32 count = nodeCount[i], first = nodeFirst[i], co = childOffsets[i];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            double r;
            if (count == 0) r = centers[(size_t)d * n + i];
            else {
                double s = 0.0;
                if (co == 0) {
                    for (u32 j = first; j < first + count; ++j) s = __dadd_rn(s, c[d][j]);
                } else {
                    for (u32 k = 0; k < 8; ++k)
                        s = __dadd_rn(s, __dmul_rn((double)nodeCount[co + k], com[(size_t)d * n + co + k]));
                }
                r = __ddiv_rn(s, (double)count);
            }
            com[(size_t)d * n + i] = r;
        }
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

cs_status enqueueNodeGeometry(cs_context* ctx, const u64* prefixes, u32 n, const double* box6, double* centers,
                              double* halfSizes, cudaStream_t s)
{
    if (n == 0) return CS_OK;
    nodeGeometryKernel<<<gridFor(ctx, n), kPropBlock, 0, s>>>(prefixes, n, box6, centers, halfSizes);
    CS_LAUNCH_CHECK(ctx, "nodeGeometryKernel");
    return CS_OK;
}

cs_status enqueueMassCenters(cs_context* ctx, const double* xs, const double* ys, const double* zs, const u32* nodeFirst,
                             const u32* nodeCount, const u32* childOffsets, const double* centers, const u32* levelRange,
                             u32 n, double* com, cudaStream_t s)
{
    if (n == 0) return CS_OK;
    // the level sizes stay on the device: every level gets a launch sized for the widest level possible
    const u32 grid = gridFor(ctx, n);
    for (int level = kL; level >= 0; --level) {
        massCentersLevelKernel<<<grid, kPropBlock, 0, s>>>(xs, ys, zs, nodeFirst, nodeCount, childOffsets, centers, levelRange,
                                                           level, n, com);
        CS_LAUNCH_CHECK(ctx, "massCentersLevelKernel");
    }
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
