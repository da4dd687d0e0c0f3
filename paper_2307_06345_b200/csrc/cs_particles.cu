// H1 bounding box and H2 Morton keys (readings A1-A3).
// Both are single streaming passes over the SoA coordinates: HBM-bound, 128-bit loads,
// persistent grid sized in multiples of the SM count.
#include "cs_device.cuh"

namespace cs {

constexpr int kBoxBlock = 512;
constexpr int kBoxBlocksPerSM = 4;
#ifndef CS_KEYS_MINBLOCKS
#define CS_KEYS_MINBLOCKS 4
#endif
constexpr int kKeysBlock = 256;
constexpr int kKeysBlocksPerSM = CS_KEYS_MINBLOCKS;

// ---------------------------------------------------------------------------------------------
// H1: per-dimension min / max.  Each CTA reduces a grid-strided slice, writes 6 partials, and
// the last CTA to finish (atomic counter) folds the partials into box6.  min/max of finite
// doubles is exact and order independent, so any reduction tree gives the oracle's bits
// (a zero extreme is canonicalised to +0.0 on both sides, A1).
// ---------------------------------------------------------------------------------------------
struct MinMax3 {
    double lo[3], hi[3];
};

__device__ __forceinline__ void mmInit(MinMax3& m)
{
    const double inf = __longlong_as_double(0x7FF0000000000000ll);
#pragma unroll
    for (int d = 0; d < 3; ++d) { m.lo[d] = inf; m.hi[d] = -inf; }
}
__device__ __forceinline__ void mmAdd(MinMax3& m, int d, double v)
{
    m.lo[d] = fmin(m.lo[d], v);
    m.hi[d] = fmax(m.hi[d], v);
}

template <bool VEC>
__global__ void __launch_bounds__(kBoxBlock) boxKernel(const double* __restrict__ x, const double* __restrict__ y,
                                                       const double* __restrict__ z, u64 n, double* partials,
                                                       u32* counter, double* box6)
{
    chainEnter();
    MinMax3 m;
    mmInit(m);
    const double* c[3] = {x, y, z};
    const u64 tid = (u64)blockIdx.x * kBoxBlock + threadIdx.x;
    const u64 nthreads = (u64)gridDim.x * kBoxBlock;
    if (VEC) {
        const u64 pairs = n >> 1;
        u64 i = tid;
        // 2 iterations x 3 dims x 16 B = 96 B in flight per thread
        for (; i + nthreads < pairs; i += 2 * nthreads) {
            double2 a[3], b[3];
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                a[d] = ldStreamD2(c[d] + 2 * i);
                b[d] = ldStreamD2(c[d] + 2 * (i + nthreads));
            }
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                mmAdd(m, d, a[d].x); mmAdd(m, d, a[d].y);
                mmAdd(m, d, b[d].x); mmAdd(m, d, b[d].y);
            }
        }
        for (; i < pairs; i += nthreads) {
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                double2 a = ldStreamD2(c[d] + 2 * i);
                mmAdd(m, d, a.x); mmAdd(m, d, a.y);
            }
        }
        if ((n & 1) && tid == 0) {
#pragma unroll
            for (int d = 0; d < 3; ++d) mmAdd(m, d, c[d][n - 1]);
        }
    } else {
        for (u64 i = tid; i < n; i += nthreads) {
#pragma unroll
            for (int d = 0; d < 3; ++d) mmAdd(m, d, ldStreamD(c[d] + i));
        }
    }
    // warp reduce
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            m.lo[d] = fmin(m.lo[d], __shfl_xor_sync(kFull, m.lo[d], o));
            m.hi[d] = fmax(m.hi[d], __shfl_xor_sync(kFull, m.hi[d], o));
        }
    }
    __shared__ double sRed[kBoxBlock / 32][6];
    __shared__ bool sLast;
    const u32 warp = threadIdx.x >> 5, lane = laneId();
    if (lane == 0) {
#pragma unroll
        for (int d = 0; d < 3; ++d) { sRed[warp][2 * d] = m.lo[d]; sRed[warp][2 * d + 1] = m.hi[d]; }
    }
    __syncthreads();
    if (threadIdx.x < 6) {
        double v = sRed[0][threadIdx.x];
        for (int w = 1; w < kBoxBlock / 32; ++w)
            v = (threadIdx.x & 1) ? fmax(v, sRed[w][threadIdx.x]) : fmin(v, sRed[w][threadIdx.x]);
        partials[(size_t)blockIdx.x * 6 + threadIdx.x] = v;
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) sLast = (atomicAdd(counter, 1u) + 1u == gridDim.x);
    __syncthreads();
    if (!sLast) return;
    __threadfence();
    // last CTA: fold gridDim.x partials
    const double inf = __longlong_as_double(0x7FF0000000000000ll);
    double acc[6];
#pragma unroll
    for (int q = 0; q < 6; ++q) acc[q] = (q & 1) ? -inf : inf;
    for (u32 b = threadIdx.x; b < gridDim.x; b += kBoxBlock) {
#pragma unroll
        for (int q = 0; q < 6; ++q) {
            double v = ((volatile double*)partials)[(size_t)b * 6 + q];
            acc[q] = (q & 1) ? fmax(acc[q], v) : fmin(acc[q], v);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int q = 0; q < 6; ++q) {
            double t = __shfl_xor_sync(kFull, acc[q], o);
            acc[q] = (q & 1) ? fmax(acc[q], t) : fmin(acc[q], t);
        }
    }
    __syncthreads();
    if (lane == 0) {
#pragma unroll
        for (int q = 0; q < 6; ++q) sRed[warp][q] = acc[q];
    }
    __syncthreads();
    if (threadIdx.x < 6) {
        double v = sRed[0][threadIdx.x];
        for (int w = 1; w < kBoxBlock / 32; ++w)
            v = (threadIdx.x & 1) ? fmax(v, sRed[w][threadIdx.x]) : fmin(v, sRed[w][threadIdx.x]);
        box6[threadIdx.x] = __dadd_rn(v, 0.0);   // -0.0 -> +0.0 (A1)
    }
    if (threadIdx.x == 0) *counter = 0;          // ready for the next call
}

cs_status enqueueBox(cs_context* ctx, const double* x, const double* y, const double* z, u64 n, double* box6,
                     cudaStream_t s)
{
    StageTimer t(ctx, CS_STAGE_BOX, s);
    const bool vec = ((((uintptr_t)x) | ((uintptr_t)y) | ((uintptr_t)z)) & 15u) == 0;
    u64 work = vec ? (n + 1) / 2 : n;
    u32 grid = (u32)ctx->numSMs * kBoxBlocksPerSM;
    u32 need = divUp(work, kBoxBlock);
    if (need < grid) grid = need ? need : 1;
    if (vec) launchChained(boxKernel<true>, dim3(grid), dim3(kBoxBlock), 0, s, x, y, z, n, ctx->boxPartials, ctx->boxCounter, box6);
    else launchChained(boxKernel<false>, dim3(grid), dim3(kBoxBlock), 0, s, x, y, z, n, ctx->boxPartials, ctx->boxCounter, box6);
    CS_LAUNCH_CHECK(ctx, "boxKernel");
    return CS_OK;
}

// box of the whole set from the boxes of its chunks (cs_buildOctreeHost reduces chunk by chunk under the upload)
__global__ void boxFoldKernel(const double* __restrict__ chunkBoxes, int chunks, double* __restrict__ box6)
{
    const int q = threadIdx.x;
    if (q >= 6) return;
    double v = chunkBoxes[q];
    for (int c = 1; c < chunks; ++c) v = (q & 1) ? fmax(v, chunkBoxes[8 * c + q]) : fmin(v, chunkBoxes[8 * c + q]);
    box6[q] = v;
}

cs_status enqueueBoxFold(cs_context* ctx, const double* chunkBoxes, int chunks, double* box6, cudaStream_t s)
{
    boxFoldKernel<<<1, 32, 0, s>>>(chunkBoxes, chunks, box6);
    CS_LAUNCH_CHECK(ctx, "boxFoldKernel");
    return CS_OK;
}

// ---------------------------------------------------------------------------------------------
// H2: Morton keys.  g = clamp(floor(((c - lo) / e) * 2^21), 0, 2^21 - 1) with explicitly
// rounded intrinsics (__dsub_rn, __ddiv_rn, __dmul_rn are never contracted into FMAs), then
// the 21 bits of each coordinate are spread to every third bit with shift-or-mask steps on
// 32-bit halves.  cvt.rmi.s32.f64 saturates and maps NaN (0/0 of a flat box) to 0: reading A1.
// Optionally (HIST) the 8 radix-digit histograms of the sort are accumulated on the fly,
// saving the sort a pass over the keys.
// ---------------------------------------------------------------------------------------------
// 11 bits -> every third bit of a 32-bit word (bit b -> bit 3b)
__device__ __forceinline__ u32 spread11(u32 v)
{
    v &= 0x7FFu;
    // v | (v << s) without overlapping bits == v * (2^s + 1): the multiplications issue on the FMA pipe, which
    // idles in this kernel, the shifts would compete with the rest for the half-rate ALU pipe
    v = (v * 0x00010001u) & 0x070000FFu;
    v = (v * 0x00000101u) & 0x0700F00Fu;
    v = (v * 0x00000011u) & 0x430C30C3u;
    v = (v * 0x00000005u) & 0x49249249u;
    return v;
}

// floor and clamp in 32-bit: cvt.rmi.s32.f64 saturates (+-inf, huge) and maps NaN to 0.
//
// The IEEE division of reading A2 costs ~25 instructions; its result is only needed to the integer
// below it.  With r21 = RN(1/e) * 2^21 (exact scaling), t' = RN(a * r21) differs from the reference
// t = RN(a / e) * 2^21 by at most 3 roundings, |t' - t| <= 3.01 * 2^-53 * 2^21 < 7.1e-10 for every
// |a / e| <= 1 (coordinates outside that range clamp to the same grid cell on both paths).  So if
// floor(t' - eps) == floor(t' + eps) with eps = 2^-27 = 7.45e-9 (the additions round by <= 2.4e-10),
// no integer lies between t and t' and floor(t) == floor(t').  Otherwise (about 1.5e-8 of the
// coordinates, or grid-aligned inputs) the reference expression itself is evaluated: exact on all inputs.
struct BoxParams {
    double lo[3], e[3], r21[3];   // r21 = 0 marks a dimension that always takes the reference expression
};

__device__ __forceinline__ u32 gridCoordinate(double c, double lo, double e, double r21)
{
    const double a = __dsub_rn(c, lo);
    int g;
    bool exact = true;
    if (r21 != 0.0) {
        const double t = __dmul_rn(a, r21);
        const int g0 = __double2int_rd(__dadd_rn(t, -0x1p-27));
        g = __double2int_rd(__dadd_rn(t, 0x1p-27));
        exact = g0 != g;
    }
    if (exact) g = __double2int_rd(__dmul_rn(__ddiv_rn(a, e), 2097152.0));
    g = max(g, 0);
    g = min(g, 2097151);
    return (u32)g;
}

__device__ __forceinline__ BoxParams loadBox(const double* __restrict__ box6)
{
    BoxParams b;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        b.lo[d] = box6[2 * d];
        b.e[d] = __dsub_rn(box6[2 * d + 1], box6[2 * d]);
        // the bound above needs a normal reciprocal that can be scaled by 2^21 exactly
        const bool ok = b.e[d] >= 0x1p-500 && b.e[d] <= 0x1p500;
        b.r21[d] = ok ? __dmul_rn(__drcp_rn(b.e[d]), 2097152.0) : 0.0;
    }
    return b;
}

// Interleave as two 32-bit words (all spreading in 32-bit arithmetic):
//   key bit 3b+2 = x bit b, 3b+1 = y bit b, 3b = z bit b   (digit = 4x + 2y + z, A3)
//   low word : x bits 0..9, y bits 0..10, z bits 0..10;  high word: x bits 10..20, y and z bits 11..20
__device__ __forceinline__ u64 mortonKey(double x, double y, double z, const BoxParams& b)
{
    const u32 gx = gridCoordinate(x, b.lo[0], b.e[0], b.r21[0]);
    const u32 gy = gridCoordinate(y, b.lo[1], b.e[1], b.r21[1]);
    const u32 gz = gridCoordinate(z, b.lo[2], b.e[2], b.r21[2]);
    const u32 lo = (spread11(gx & 0x3FFu) << 2) | (spread11(gy) << 1) | spread11(gz);
    const u32 hi = spread11(gx >> 10) | (spread11(gy >> 11) << 2) | (spread11(gz >> 11) << 1);
    return ((u64)hi << 32) | lo;
}

// ---------------------------------------------------------------------------------------------
// Hilbert keys (reading A28: the curve of the Butz algorithm in Hamilton's
// formulation).  The curve walks every cube octant by octant, so a Hilbert key is the Morton key
// re-labelled digit by digit: the octant taken at a level (the Morton digit, 4x + 2y + z) and the
// orientation of the curve in the current cube (its entry corner e and exit axis d: 8 x 3 = 24 states)
// give the Hilbert digit and the orientation in the sub-cube.  Three levels are resolved per table
// look-up: hilbertTable[state][9 Morton bits] = 9 Hilbert bits | next state << 9 (24 x 512 entries of 16
// bits, 24 KB, staged in shared memory): 21 levels = 7 look-ups from the curve's initial orientation
// (e = 0, d = 0).  (Two levels per look-up, 11 look-ups: the key kernel took 0.57 instead of 0.37 ms.)
// The table is generated on the host when a context is created, from the curve's definition:
//   gc(i) = i ^ (i >> 1);  e(w) = 0 (w = 0), gc(2 floor((w - 1) / 2));  d(w) = 0 (w = 0), tsb(w - 1) mod 3
//   (w even), tsb(w) mod 3 (w odd);  in state (e, d) octant l is the w-th of the cube, w = gc^-1(rotr3(l ^ e,
//   d + 1)), and its sub-cube has state (e ^ rotl3(e(w), d + 1), (d + d(w) + 1) mod 3).
// ---------------------------------------------------------------------------------------------
constexpr int kHilbertStates = 24;
constexpr int kHilbertEntries = 512;            // per state: three levels per look-up (state index = 3 e + d)

static void hilbertStep(u32 state, u32 l, u32& w, u32& next)
{
    auto rot = [](u32 b, u32 r, bool left) {
        r %= 3;
        return (left ? ((b << r) | (b >> (3 - r))) : ((b >> r) | (b << (3 - r)))) & 7u;
    };
    auto trailingOnes = [](u32 i) { u32 c = 0; for (; i & 1u; i >>= 1) ++c; return c; };
    const u32 e = state / 3, d = state % 3;
    const u32 t = rot(l ^ e, d + 1, false);
    w = t ^ (t >> 1) ^ (t >> 2);                                       // inverse Gray code on 3 bits
    const u32 ew = w == 0 ? 0u : (2 * ((w - 1) / 2)) ^ ((2 * ((w - 1) / 2)) >> 1);
    const u32 dw = w == 0 ? 0u : ((w & 1u) ? trailingOnes(w) % 3 : trailingOnes(w - 1) % 3);
    next = (e ^ rot(ew, d + 1, true)) * 3 + (d + dw + 1) % 3;
}

void hilbertBuildTable(unsigned short* table /*[24 * 512]*/)
{
    for (u32 s = 0; s < (u32)kHilbertStates; ++s)
        for (u32 o = 0; o < (u32)kHilbertEntries; ++o) {
            u32 w1, s1, w2, s2, w3, s3;
            hilbertStep(s, o >> 6, w1, s1);
            hilbertStep(s1, (o >> 3) & 7u, w2, s2);
            hilbertStep(s2, o & 7u, w3, s3);
            table[s * kHilbertEntries + o] = (unsigned short)((w1 << 6) | (w2 << 3) | w3 | (s3 << 9));
        }
}

// One-level inverse transitions for the node geometry (cs_props.cu): inv[state][Hilbert digit w] = octant l | next
// state << 3 (24 x 8 bytes), stored behind the two-level table.
void hilbertBuildInverse(unsigned char* inv /*[24 * 8]*/)
{
    for (u32 s = 0; s < (u32)kHilbertStates; ++s)
        for (u32 l = 0; l < 8; ++l) {
            u32 w, next;
            hilbertStep(s, l, w, next);
            inv[s * 8 + w] = (unsigned char)(l | (next << 3));
        }
}

__device__ __forceinline__ u64 hilbertFromMorton(u64 m, const unsigned short* __restrict__ tab)
{
    u32 ent = tab[(u32)(m >> 54)];                                    // state 0, digits 1..3
    u64 h = ent & 511u;
#pragma unroll
    for (int p = 1; p <= 6; ++p) {
        const u32 o = (u32)(m >> (54 - 9 * p)) & 511u;
        ent = tab[(ent >> 9) * kHilbertEntries + o];
        h = (h << 9) | (ent & 511u);
    }
    return h;
}

// HIST: first digit that is counted (the sort plan's first digit: the others are not sorted by), or -1 for none
template <int HIST>
__device__ __forceinline__ void histAdd(u32* sh, u64 key)
{
    if (HIST >= 0) {
#pragma unroll
        for (int p = HIST; p < kSortPasses; ++p)
            atomicAdd(&sh[(p - HIST) * kRadix + (u32)((key >> (p * kRadixBits)) & (kRadix - 1))], 1u);
    }
}

template <bool VEC, int HIST, bool HILBERT>
__global__ void __launch_bounds__(kKeysBlock, CS_KEYS_MINBLOCKS) keysKernel(const double* __restrict__ x, const double* __restrict__ y,
                                                         const double* __restrict__ z, u64 n,
                                                         const double* __restrict__ box6, u64* __restrict__ keys,
                                                         u32* gHist, const unsigned short* __restrict__ hilbertTable,
                                                         u32* __restrict__ keys32)
{
    chainEnter();
    constexpr int kHistWords = HIST >= 0 ? (kSortPasses - HIST) * kRadix : 1;
    __shared__ u32 sh[kHistWords];
    __shared__ unsigned short sTab[HILBERT ? kHilbertStates * kHilbertEntries : 1];
    if (HIST >= 0) {
        for (int i = threadIdx.x; i < kHistWords; i += kKeysBlock) sh[i] = 0;
    }
    if (HILBERT) {
        for (int i = threadIdx.x; i < kHilbertStates * kHilbertEntries / 2; i += kKeysBlock)
            reinterpret_cast<u32*>(sTab)[i] = reinterpret_cast<const u32*>(hilbertTable)[i];
    }
    if (HIST >= 0 || HILBERT) __syncthreads();
    const BoxParams b = loadBox(box6);
    auto sfcKey = [&](double px, double py, double pz) -> u64 {
        const u64 m = mortonKey(px, py, pz, b);
        return HILBERT ? hilbertFromMorton(m, sTab) : m;
    };
    // keys32 (L = 10): floor(t 2^10) = floor(t 2^21) >> 11 for the same quotient t (scaling by a power of
    // two is exact) and the clamps agree, so the 30-bit key is the 63-bit key without its low 33 bits
    auto put2 = [&](u64 i2, u64 k0, u64 k1) {
        if (HIST < 0 && keys32) *reinterpret_cast<uint2*>(keys32 + i2) = make_uint2((u32)(k0 >> 33), (u32)(k1 >> 33));
        else stStreamU2(keys + i2, k0, k1);
    };
    auto put1 = [&](u64 i1, u64 k) {
        if (HIST < 0 && keys32) keys32[i1] = (u32)(k >> 33);       // (never together with the 63-bit sort's histograms)
        else keys[i1] = k;
    };
    const u64 tid = (u64)blockIdx.x * kKeysBlock + threadIdx.x;
    const u64 nthreads = (u64)gridDim.x * kKeysBlock;
    if (VEC) {
        const u64 pairs = n >> 1;
        u64 i = tid;
        // two iterations of loads in flight per thread (96 B)
        for (; i + nthreads < pairs; i += 2 * nthreads) {
            const u64 i2 = i + nthreads;
            double2 ax = ldStreamD2(x + 2 * i), ay = ldStreamD2(y + 2 * i), az = ldStreamD2(z + 2 * i);
            double2 bx = ldStreamD2(x + 2 * i2), by = ldStreamD2(y + 2 * i2), bz = ldStreamD2(z + 2 * i2);
            u64 k0 = sfcKey(ax.x, ay.x, az.x);
            u64 k1 = sfcKey(ax.y, ay.y, az.y);
            put2(2 * i, k0, k1);
            histAdd<HIST>(sh, k0);
            histAdd<HIST>(sh, k1);
            k0 = sfcKey(bx.x, by.x, bz.x);
            k1 = sfcKey(bx.y, by.y, bz.y);
            put2(2 * i2, k0, k1);
            histAdd<HIST>(sh, k0);
            histAdd<HIST>(sh, k1);
        }
        for (; i < pairs; i += nthreads) {
            double2 vx = ldStreamD2(x + 2 * i);
            double2 vy = ldStreamD2(y + 2 * i);
            double2 vz = ldStreamD2(z + 2 * i);
            u64 k0 = sfcKey(vx.x, vy.x, vz.x);
            u64 k1 = sfcKey(vx.y, vy.y, vz.y);
            put2(2 * i, k0, k1);
            histAdd<HIST>(sh, k0);
            histAdd<HIST>(sh, k1);
        }
        if ((n & 1) && tid == 0) {
            u64 k = sfcKey(x[n - 1], y[n - 1], z[n - 1]);
            put1(n - 1, k);
            histAdd<HIST>(sh, k);
        }
    } else {
        for (u64 i = tid; i < n; i += nthreads) {
            u64 k = sfcKey(ldStreamD(x + i), ldStreamD(y + i), ldStreamD(z + i));
            put1(i, k);
            histAdd<HIST>(sh, k);
        }
    }
    if (HIST >= 0) {
        __syncthreads();
        for (int i = threadIdx.x; i < kHistWords; i += kKeysBlock) {
            u32 v = sh[i];
            if (v) atomicAdd(&gHist[HIST * kRadix + i], v);
        }
    }
}

cs_status enqueueKeys(cs_context* ctx, const double* x, const double* y, const double* z, u64 n, const double* box6,
                      u64* keys, int histFrom, int curve, cudaStream_t s, u32* keys32)
{
    StageTimer t(ctx, CS_STAGE_KEYS, s);
    if (n == 0) return CS_OK;
    const bool vec = ((((uintptr_t)x) | ((uintptr_t)y) | ((uintptr_t)z)) & 15u) == 0 &&
                     (keys32 ? (((uintptr_t)keys32) & 7u) == 0 : (((uintptr_t)keys) & 15u) == 0);
    u64 work = vec ? (n + 1) / 2 : n;
    u32 grid = (u32)ctx->numSMs * kKeysBlocksPerSM;
    u32 need = divUp(work, kKeysBlock);
    if (need < grid) grid = need ? need : 1;
    u32* h = ctx->sortHist;
    const unsigned short* tab = ctx->hilbertTable;
#define CS_KEYS_LAUNCH(V, H, C) launchChained(keysKernel<V, H, C>, dim3(grid), dim3(kKeysBlock), 0, s, x, y, z, n, box6, keys, h, tab, keys32)
#define CS_KEYS_HIST(V, C)                                        \
    do {                                                          \
        if (histFrom < 0) CS_KEYS_LAUNCH(V, -1, C);               \
        else if (histFrom == 0) CS_KEYS_LAUNCH(V, 0, C);          \
        else if (histFrom == kSortMaxFirst) CS_KEYS_LAUNCH(V, kSortMaxFirst, C); \
        else if (histFrom == kSortShortFirst) CS_KEYS_LAUNCH(V, kSortShortFirst, C); \
        else CS_KEYS_LAUNCH(V, kSortTopFirst, C);                 \
    } while (0)
    if (curve == CS_CURVE_HILBERT) {
        if (vec) CS_KEYS_HIST(true, true);
        else CS_KEYS_HIST(false, true);
    } else {
        if (vec) CS_KEYS_HIST(true, false);
        else CS_KEYS_HIST(false, false);
    }
#undef CS_KEYS_HIST
#undef CS_KEYS_LAUNCH
    CS_LAUNCH_CHECK(ctx, "keysKernel");
    return CS_OK;
}

}  // namespace cs
