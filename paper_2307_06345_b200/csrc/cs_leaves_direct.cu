// H4-H8, start {0, 8^21}, run to convergence: the fixpoint of f and g in ONE pass over P.
//
// The iteration of PAPER.md:62-128 from the root only ever splits (a node is split iff it holds
// more than N_crit particles and lies above depth L, and then its 8 children together hold more
// than N_crit, so they never merge back: DESIGN.md A8), hence its fixpoint is the top-down tree:
//   node (level l < L, prefix p) is internal  <=>  count(l, p) > N_crit                      (*)
// and the leaves are the children of internal nodes that are not internal (plus the root if it
// is not).  Because P is sorted, (*) can be decided from windows of b+1 = N_crit+1 consecutive
// keys: a node holds more than b particles iff it contains such a window, so with
//   w_i = min(#leading octal digits shared by P[i] and P[i+b], L-1)       (0 <= i < n-b)
// (L = 21; for the 30-bit keys of the L = 10 entry points, held in the top digits, the cap is 9: wcap below)
// the deepest internal node on the path of particle j has level
//   d_j = max{ w_i : j-b <= i <= j }                                       (sliding maximum)
// and the leaf that holds particle j has level D_j = d_j + 1 (D_j = 0, the root, if n <= b).
// Between two neighbours a = P[j-1] < c = P[j] that fall into different leaves (they share
// s < D_j digits) the leaf array K contains, in key order:
//   the empty siblings to the right of a's ancestors on levels D_{j-1} .. s+2,
//   the empty children of the common ancestor strictly between the two branches (level s+1),
//   the empty siblings to the left of c's ancestors on levels s+2 .. D_j,
//   the leaf of c.
// All of them have lower_bound position j in P (Eq. 3), so N_i follows from the off[] array
// like in the iterative path.  One kernel: per-tile counts, decoupled look-back across tiles,
// emission.  Per tile: window levels and the sliding maximum run on bytes, four per 32-bit SIMD
// operation; the positions where a leaf starts (one in ~18) are compacted with a block scan, so
// the digit arithmetic of the counts and the emission run on a dense list.
// rounds := (deepest leaf level) + 1 is what the iteration would have reported (one round per
// level, plus the confirming one: DESIGN.md A12).
#include "cs_device.cuh"

namespace cs {

#ifndef CS_DIR_MINBLOCKS
#define CS_DIR_MINBLOCKS 6
#endif
constexpr int kDirBlock = 256;
constexpr int kDirItems = 8;
constexpr int kDirTile = kDirBlock * kDirItems;          // 2048 particle boundaries per tile
static_assert(kDirTile == (1 << kDirectTileLog2), "look-back array of the context is sized for this tile");

constexpr u64 kOct1 = 0x1249249249249249ull;             // bit 0 of every octal digit (bits 0, 3, ..., 60)

// sum of the octal digits of key on levels lo..hi (1-based, digit l = bits [3(L-l), 3(L-l)+2]); 0 if lo > hi
__device__ __forceinline__ u32 digitSum(u64 key, int lo, int hi)
{
    if (lo > hi) return 0;
    const u64 upper = (lo <= 1) ? ~0ull >> 1 : ((1ull << (3 * (kL + 1 - lo))) - 1);
    const u64 lower = (1ull << (3 * (kL - hi))) - 1;
    const u64 m = key & upper & ~lower;
    return __popcll(m & kOct1) + 2 * __popcll(m & (kOct1 << 1)) + 4 * __popcll(m & (kOct1 << 2));
}
__device__ __forceinline__ u32 digitAt(u64 key, int l) { return (u32)(key >> (3 * (kL - l))) & 7u; }
__device__ __forceinline__ int sharedDigits(u64 a, u64 c) { return (__clzll((long long)(a ^ c)) - 1) / 3; }   // 21 if equal
// the same from x = a ^ c (bit 63 clear), without the 64-bit count of leading zeros: converted to float with
// rounding toward zero, x keeps its binary exponent e = floor(log2 x), and (clz - 1) / 3 = (62 - e) / 3, the
// division by multiplication (exact for 0 .. 189).  x = 0 converts to 0.0f (e = -127): 63, capped by the callers.
__device__ __forceinline__ u32 sharedDigitsX(u64 x)
{
    const u32 e = (__float_as_uint(__ull2float_rz(x)) >> 23);   // e + 127
    return ((62u + 127u) - e) * 43u >> 7;
}

// number of K entries owned by position j.  Da = D_{j-1}, Dc = D_j.
__device__ __forceinline__ u32 dirCount(u64 a, u64 c, int Da, int Dc, u32 j, u32 n)
{
    if (j > n) return 0;
    if (j == n) return (n ? 7u * Da - digitSum(a, 1, Da) : 1u) + 1u;      // right flank of the last particle, 8^21
    if (j == 0) return digitSum(c, 1, Dc) + 1u;                            // left flank of the first particle, its leaf
    const int s = sharedDigits(a, c);
    if (s >= Dc) return 0;                                                 // same leaf
    const u32 up = 7u * (u32)(Da - s - 1) - digitSum(a, s + 2, Da);
    const u32 mid = digitAt(c, s + 1) - digitAt(a, s + 1) - 1u;
    return up + mid + digitSum(c, s + 2, Dc) + 1u;
}

// write the K entries owned by position j to K[pos ..], off[pos ..] = j
__device__ __noinline__ void dirEmit(u64 a, u64 c, int Da, int Dc, u32 j, u32 n, u32 pos, u64* __restrict__ K,
                                        u32* __restrict__ off, u32 cap)
{
    auto put = [&](u64 key) {
        if (pos <= cap) {
            K[pos] = key;
            off[pos] = j;
        }
        ++pos;
    };
    int s = -1;
    if (j != 0 && j != n) s = sharedDigits(a, c);
    if (j != 0) {                                          // siblings to the right of a's ancestors, deepest first
        for (int l = Da; l >= s + 2; --l) {
            const u64 step = 1ull << (3 * (kL - l));
            const u64 parent = a & ~((step << 3) - 1);     // (step << 3) = 2^63 at l = 1: still a valid mask
            for (u32 q = digitAt(a, l) + 1; q < 8; ++q) put(parent + q * step);
        }
    }
    if (j == n) {
        put(kKeyEnd);                                      // A11: terminal element
        return;
    }
    if (j != 0) {                                          // empty children of the common ancestor between the branches
        const int l = s + 1;
        const u64 step = 1ull << (3 * (kL - l));
        const u64 parent = a & ~((step << 3) - 1);
        for (u32 q = digitAt(a, l) + 1; q < digitAt(c, l); ++q) put(parent + q * step);
    }
    for (int l = s + 2; l <= Dc; ++l) {                    // siblings to the left of c's ancestors, shallowest first
        const u64 step = 1ull << (3 * (kL - l));
        const u64 parent = c & ~((step << 3) - 1);
        for (u32 q = 0; q < digitAt(c, l); ++q) put(parent + q * step);
    }
    put(Dc == 0 ? 0ull : c & ~((1ull << (3 * (kL - Dc))) - 1));   // the leaf of c
}

// ---- kernel 1: levels ---------------------------------------------------------------------------
// dynamic shared memory: keys of [T0 - b - 1, T0 + T + b), window levels (two word arrays for the
// steps of the sliding maximum), neighbour levels s[p], list of leaf-start positions
struct DirLayout {
    u32 nKeys, words, wWords, offW0, offW1, offS, offList, total;
};
__host__ __device__ inline DirLayout dirLayout(u32 b)
{
    DirLayout L;
    const u32 W = b + 1;
    L.nKeys = kDirTile + 2 * b + 1;
    L.words = (kDirTile + 1 + W + 3) / 4 + 1;              // covers every byte a later step or the result needs
    L.wWords = L.words + W / 4 + 4;                        // + read-ahead of a step (at most 3/4 W bytes) + slack
    L.offW0 = L.nKeys * 8;
    L.offW1 = L.offW0 + L.wWords * 4;
    L.offS = (L.offW1 + L.wWords * 4 + 15u) & ~15u;
    L.offList = L.offS + kDirTile + 16;
    L.total = L.offList + kDirTile * 2;
    return L;
}

struct DirSmem {
    u64* K;                   // K[q] <-> particle G0 + q, G0 = T0 - b - 1
    u32* W0;                  // byte i <-> window start G0 + i
    u32* W1;
    unsigned char* S;         // S[p] = digits shared by the neighbours left and right of position T0 + p
    unsigned short* list;     // positions p (tile-local) that own K entries, ascending
};

// byte-wise maximum of two words whose bytes are all below 128 (levels are at most 21): the SIMD video
// instruction behind __vmaxu4 is emulated on this architecture (9 SASS), this takes 6
__device__ __forceinline__ u32 maxBytes(u32 a, u32 b)
{
    const u32 ge = ((a | 0x80808080u) - b) & 0x80808080u;   // bit 7 of a byte set <=> a's byte >= b's (no borrow crosses bytes)
    const u32 m = (ge >> 7) * 0xFFu;                        // 0xFF in those bytes
    return (a & m) | (b & ~m);
}

// bytes [4q + o, 4q + o + 4) of the word array a
__device__ __forceinline__ u32 dirShifted(const u32* a, u32 q, u32 o)
{
    const u32 w = q + (o >> 2);
    return __funnelshift_r(a[w], a[w + 1], 8 * (o & 3u));
}

// Keys -> window levels -> sliding maximum for one tile.  Returns the byte array dmax with
// dmax[q'] = d of particle T0 - 1 + q'.  EDGE: the tile touches the ends of P.
template <bool EDGE>
__device__ __forceinline__ const unsigned char* dirTileLevels(const DirSmem& sm, const DirLayout& L,
                                                              const u64* __restrict__ P, u32 n, u32 b, long long T0,
                                                              u32 wcap)
{
    const u32 tid = threadIdx.x;
    const long long G0 = T0 - (long long)b - 1;
    const u64* Pt = P + G0;                                // only dereferenced where G0 + q is inside P
    auto valid = [&](u32 q) { const long long g = G0 + q; return g >= 0 && g < (long long)n; };
    // ---- keys of the tile and its halo: all loads of a thread are in flight together -------------
    {
        u64 kr[kDirItems];
#pragma unroll
        for (int k = 0; k < kDirItems; ++k) {
            const u32 q = k * kDirBlock + tid;
            kr[k] = (!EDGE || valid(q)) ? ldStreamU64(Pt + q) : 0ull;
        }
        for (u32 q = kDirTile + tid; q < L.nKeys; q += kDirBlock) sm.K[q] = (!EDGE || valid(q)) ? ldStreamU64(Pt + q) : 0ull;
#pragma unroll
        for (int k = 0; k < kDirItems; ++k) sm.K[k * kDirBlock + tid] = kr[k];
        // the parts of the level arrays that no thread computes read as level 0
        for (u32 q = (kDirTile + b + 1) / 4 + tid; q < L.wWords; q += kDirBlock) sm.W0[q] = 0;
        for (u32 q = L.words + tid; q < L.wWords; q += kDirBlock) sm.W1[q] = 0;
    }
    __syncthreads();
    // ---- window levels w[i] = min(digits shared by P[g], P[g + b], L - 1), g = G0 + i (0 where the
    // window does not fit into P), and neighbour levels: a leaf starts at position p iff
    // S[p] <= d of particle T0 + p.  One pass, the key K[i + b] serves both ------------------------
    unsigned char* w0 = reinterpret_cast<unsigned char*>(sm.W0);
#pragma unroll
    for (int k = 0; k < kDirItems; ++k) {
        const u32 i = k * kDirBlock + tid;
        const u64 kb = sm.K[i + b];
        u32 w = sharedDigitsX(sm.K[i] ^ kb);
        w = w < wcap ? w : wcap;
        u32 sv = sharedDigitsX(kb ^ sm.K[i + b + 1]);
        if (EDGE) {
            if (!(G0 + i >= 0 && G0 + i + b < (long long)n)) w = 0;
            const u64 j = (u64)T0 + i;
            if (j == 0 || j == n) sv = 0;                  // first particle / tail of the array: always owns entries
            else if (j > n) sv = 255;                      // beyond the tail: never
        }
        w0[i] = (unsigned char)w;
        sm.S[i] = (unsigned char)sv;
    }
    for (u32 i = kDirTile + tid; i <= kDirTile + b; i += kDirBlock) {
        u32 w = sharedDigitsX(sm.K[i] ^ sm.K[i + b]);
        w = w < wcap ? w : wcap;
        if (EDGE && !(G0 + i >= 0 && G0 + i + b < (long long)n)) w = 0;
        w0[i] = (unsigned char)w;
    }
    __syncthreads();
    // ---- sliding maximum over b+1 consecutive windows, 4 bytes per operation: the window length
    // covered by a byte grows 4-fold per step (then 2-fold, then the two overlapping windows) --------
    u32* src = sm.W0;
    u32* dst = sm.W1;
    const u32 W = b + 1;
    u32 len = 1;                                           // byte i = max of w over [i, i + len)
    while (len * 4 <= W) {
        if ((len & 3u) == 0) {                             // whole-word offsets: no funnel shifts
            const u32 o = len >> 2;
            for (u32 q = tid; q < L.words; q += kDirBlock)
                dst[q] = maxBytes(maxBytes(src[q], src[q + o]), maxBytes(src[q + 2 * o], src[q + 3 * o]));
        } else {
            for (u32 q = tid; q < L.words; q += kDirBlock) {
                const u32 a = maxBytes(src[q], dirShifted(src, q, len));
                const u32 c = maxBytes(dirShifted(src, q, 2 * len), dirShifted(src, q, 3 * len));
                dst[q] = maxBytes(a, c);
            }
        }
        __syncthreads();
        u32* t = src; src = dst; dst = t;
        len *= 4;
    }
    if (len * 2 <= W) {
        for (u32 q = tid; q < L.words; q += kDirBlock) dst[q] = maxBytes(src[q], dirShifted(src, q, len));
        __syncthreads();
        u32* t = src; src = dst; dst = t;
        len *= 2;
    }
    if (len < W) {                                         // two overlapping windows of length len cover b+1
        for (u32 q = tid; q < (kDirTile + 1 + 3) / 4 + 1; q += kDirBlock) dst[q] = maxBytes(src[q], dirShifted(src, q, W - len));
        __syncthreads();
        src = dst;
    }
    return reinterpret_cast<const unsigned char*>(src);
}

// One tile of kDirTile positions per CTA: d of every particle (dArr), which positions own K entries
// (flags, one bit per position) and how many entries the tile owns (totals).  No CTA waits for another.
// BFIX: bucket size known at compile time (the layout, loop counts and offsets of the sliding maximum become
// constants), or 0 for any bucket size.
template <u32 BFIX>
__global__ void __launch_bounds__(kDirBlock, CS_DIR_MINBLOCKS)
    leavesLevelsKernel(DeviceCtrl* ctrl, const u64* __restrict__ P, u32 n, u32 bAny, u32 wcap, unsigned char* __restrict__ dArr,
                       unsigned char* __restrict__ flags, u32* __restrict__ totals, u32* __restrict__ listSize,
                       ulonglong2* __restrict__ listKeys, u32* __restrict__ listMeta)
{
    chainEnter();
    extern __shared__ __align__(16) unsigned char dsm[];
    __shared__ u32 sTotal, sMaxLevel;
    __shared__ u32 warpSums[kDirBlock / 32 + 1];
    const u32 b = BFIX ? BFIX : bAny;
    const DirLayout L = dirLayout(b);
    DirSmem sm;
    sm.K = reinterpret_cast<u64*>(dsm);
    sm.W0 = reinterpret_cast<u32*>(dsm + L.offW0);
    sm.W1 = reinterpret_cast<u32*>(dsm + L.offW1);
    sm.S = dsm + L.offS;
    sm.list = reinterpret_cast<unsigned short*>(dsm + L.offList);
    const u32 tid = threadIdx.x;
    const u32 tile = blockIdx.x;
    if (tid == 0) {
        sTotal = 0;
        sMaxLevel = 0;
    }
    const long long T0 = (long long)tile * kDirTile;
    const long long G0 = T0 - (long long)b - 1;
    const bool edge = G0 < 0 || G0 + (long long)L.nKeys > (long long)n;
    const unsigned char* dmax = edge ? dirTileLevels<true>(sm, L, P, n, b, T0, wcap) : dirTileLevels<false>(sm, L, P, n, b, T0, wcap);
    const u32* dm = reinterpret_cast<const u32*>(dmax);

    // ---- which positions own K entries: S[p] <= d_{T0+p}, 8 consecutive positions per thread ----
    const u32* s32 = reinterpret_cast<const u32*>(sm.S);
    const u32 sA = s32[2 * tid], sB = s32[2 * tid + 1];
    const u32 d0 = dm[2 * tid], d1 = dm[2 * tid + 1], d2 = dm[2 * tid + 2];
    const u32 dA = __funnelshift_r(d0, d1, 8), dB = __funnelshift_r(d1, d2, 8);   // d of particles T0 + 8 tid .. + 7
    const u32 fA = __vcmpleu4(sA, dA), fB = __vcmpleu4(sB, dB);                   // 0xFF per owning position
    // one bit per position: bit k of the byte <-> position 8 tid + k
    const u32 bitsA = ((fA & 0x01010101u) * 0x10204080u) >> 28, bitsB = ((fB & 0x01010101u) * 0x10204080u) >> 28;
    const u32 fbyte = bitsA | (bitsB << 4);
    const u32 mine = __popc(fbyte);
    u32 mx = __vmaxu4(dA, dB);
    mx = __vmaxu4(mx, mx >> 16);
    mx = __vmaxu4(mx, mx >> 8) & 0xFFu;                     // deepest internal level d on this thread's particles (0 past the tail)
    u32 nb;
    u32 slot = blockExclusiveScan<kDirBlock>(mine, warpSums, &nb);
    for (u32 f = fbyte; f; f &= f - 1) sm.list[slot++] = (unsigned short)(8 * tid + __ffs((int)f) - 1);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(kFull, mx, o));
    if ((tid & 31u) == 0 && mx + 1 > sMaxLevel) atomicMax(&sMaxLevel, mx + 1);   // leaf level D = d + 1
    __syncthreads();

    // ---- K entries owned by the tile; the leaf starts go to the emission kernel as a compact list (the two
    // keys, position, levels and entry count of each), or, if there are too many, as flags + level bytes -------
    const bool compact = nb <= (u32)kDirectCompact;
    if (!compact) flags[(size_t)tile * kDirBlock + tid] = (unsigned char)fbyte;
    // level bytes: the whole tile for the gather path, and always its last particles (position T0 + 2048 of the
    // next tile reads the level of particle T0 + 2047)
    if (!compact || tid == kDirBlock - 1) *reinterpret_cast<uint2*>(dArr + (size_t)T0 + 8 * tid) = make_uint2(dA, dB);
    u32 cnt = 0;
    for (u32 m = tid; m < nb; m += kDirBlock) {
        const u32 p = sm.list[m];
        const u64 a = sm.K[p + b], c = sm.K[p + b + 1];
        const u32 Da = dmax[p] + 1u, Dc = dmax[p + 1] + 1u;
        const u32 e = dirCount(a, c, (int)Da, (int)Dc, (u32)(T0 + p), n);
        cnt += e;
        if (compact) {                                       // p < 2^11, levels <= 22, e <= 7 * 21 + 7 + 1
            listKeys[(size_t)tile * kDirectCompact + m] = make_ulonglong2(a, c);
            listMeta[(size_t)tile * kDirectCompact + m] = p | (Da << 11) | (Dc << 16) | (e << 21);
        }
    }
    cnt = warpReduceSum(cnt);
    if ((tid & 31u) == 0 && cnt) atomicAdd(&sTotal, cnt);
    __syncthreads();
    if (tid == 0) {
        totals[tile] = sTotal;
        listSize[tile] = compact ? nb : 0xFFFFFFFFu;
        atomicMax(&ctrl->changed[0], sMaxLevel);           // changed[0] doubles as the deepest leaf level
    }
}

// ---- kernel 2: emission ---------------------------------------------------------------------------
// The same tiles; bases = exclusive prefix of totals over tiles (bases[tiles] = all K entries).  The
// listed positions fetch their two keys and levels from global memory; everything else is a bit scan.
constexpr int kEmitBlock = kDirBlock / 2;                 // 16 positions per thread: most threads hold a listed position
__global__ void __launch_bounds__(kEmitBlock)
    leavesEmitDirectKernel(DeviceCtrl* ctrl, const u64* __restrict__ P, u32 n, const unsigned char* __restrict__ dArr,
                           const unsigned char* __restrict__ flags, const u32* __restrict__ bases, u32 tiles,
                           const u32* __restrict__ listSize, const ulonglong2* __restrict__ listKeys,
                           const u32* __restrict__ listMeta, u64* __restrict__ K, u32* __restrict__ off, u32 cap)
{
    chainEnter();
    __shared__ unsigned short list[kDirTile];
    __shared__ u32 warpSums[kEmitBlock / 32 + 1];
    const u32 tid = threadIdx.x;
    const u32 tile = blockIdx.x;
    const u64 T0 = (u64)tile * kDirTile;
    u32 carry = bases[tile];
    const u32 listed = listSize[tile];
    if (listed != 0xFFFFFFFFu) {
        // ---- compact list from the levels kernel: nothing to gather, nothing to recount ------------------------
        for (u32 base = 0; base < listed; base += kEmitBlock) {
            const u32 m = base + tid;
            ulonglong2 ac = make_ulonglong2(0, 0);
            u32 meta = 0;
            if (m < listed) {
                ac = listKeys[(size_t)tile * kDirectCompact + m];
                meta = listMeta[(size_t)tile * kDirectCompact + m];
            }
            const u32 cnt = meta >> 21;
            u32 t;
            const u32 e = blockExclusiveScan<kEmitBlock>(cnt, warpSums, &t);
            if (cnt)
                dirEmit(ac.x, ac.y, (int)((meta >> 11) & 31u), (int)((meta >> 16) & 31u), (u32)(T0 + (meta & 2047u)), n,
                        carry + e, K, off, cap);
            carry += t;
            __syncthreads();                                // warpSums is reused by the next chunk
        }
    } else {
        const u32 fbits = reinterpret_cast<const unsigned short*>(flags)[(size_t)tile * kEmitBlock + tid];
        u32 nb;
        u32 slot = blockExclusiveScan<kEmitBlock>(__popc(fbits), warpSums, &nb);
        for (u32 f = fbits; f; f &= f - 1) list[slot++] = (unsigned short)(16 * tid + __ffs((int)f) - 1);
        __syncthreads();
        for (u32 base = 0; base < nb; base += kEmitBlock) {
            const u32 m = base + tid;
            u64 a = 0, c = 0;
            int Da = 0, Dc = 0;
            u32 j = 0, cnt = 0;
            if (m < nb) {
                j = (u32)(T0 + list[m]);
                if (j > 0) {
                    a = __ldg(P + j - 1);
                    Da = dArr[j - 1] + 1;
                }
                if (j < n) {
                    c = __ldg(P + j);
                    Dc = dArr[j] + 1;
                }
                cnt = dirCount(a, c, Da, Dc, j, n);
            }
            u32 t;
            const u32 e = blockExclusiveScan<kEmitBlock>(cnt, warpSums, &t);
            if (cnt) dirEmit(a, c, Da, Dc, j, n, carry + e, K, off, cap);
            carry += t;
            __syncthreads();                                // warpSums is reused by the next chunk
        }
    }
    if (tile == 0 && tid == 0) {                            // close the build
        const u32 nl = bases[tiles] - 1;                    // K entries minus the terminal 8^21
        const u32 rounds = ctrl->changed[0] + 1;            // one round per level + the confirming one (A12)
        ctrl->nl[0] = nl;
        ctrl->rounds = rounds;
        ctrl->nl[rounds] = nl;
        ctrl->directBuild = 1;
        if (nl > cap) ctrl->status = CS_ERR_CAPACITY;
        else {
            ctrl->numLeaves = nl;
            ctrl->converged = 1;
        }
        ctrl->done = 1;
    }
}

// n <= bucketSize (A15 for n == 0): the root is the only leaf, K = {0, 8^21}, one (confirming) round
__global__ void leavesDirectRootKernel(DeviceCtrl* ctrl, u64* K, u32* off, u32 n)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        K[0] = 0;
        K[1] = kKeyEnd;
        off[0] = 0;
        off[1] = n;
        ctrl->nl[0] = 1;
        ctrl->nl[1] = 1;
        ctrl->rounds = 1;
        ctrl->numLeaves = 1;
        ctrl->converged = 1;
        ctrl->directBuild = 1;
        ctrl->done = 1;
    }
}

// dynamic shared memory of the levels kernel up to the largest bucket size it takes (per device: once per cs_create)
cs_status leavesDirectInit(cs_context* ctx)
{
    CS_CUDA(ctx, cudaFuncSetAttribute(leavesLevelsKernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (int)dirLayout(kDirectMaxBucket).total));
    return CS_OK;
}

bool leavesDirectSupported(const cs_context* ctx, u32 bucket)
{
    return bucket <= (u32)kDirectMaxBucket && dirLayout(bucket).total <= 200u * 1024u && ctx->dirFlags != nullptr;
}

// enqueue the one-pass build into the workspace arrays leafK[0] / leafOff[0]; ctrl must be zeroed
cs_status enqueueLeavesDirect(cs_context* ctx, const u64* P, u64 n, u32 bucket, u32 cap, u32 maxLevel, cudaStream_t s)
{
    DeviceCtrl* ctrl = ctx->ctrl;
    if (n <= bucket) {                                     // no window of bucket+1 keys: the root is not split
        leavesDirectRootKernel<<<1, 32, 0, s>>>(ctrl, ctx->leafK[0], ctx->leafOff[0], (u32)n);
        CS_LAUNCH_CHECK(ctx, "leavesDirectRootKernel");
        return CS_OK;
    }
    const DirLayout L = dirLayout(bucket);
    const u32 tiles = (u32)(n / kDirTile) + 1;            // positions 0 .. n inclusive
    // the bucket sizes of BASELINE.json's configurations get kernels with the bucket size folded in
    auto* kernel = bucket == 64 ? leavesLevelsKernel<64> : bucket == 16 ? leavesLevelsKernel<16> : leavesLevelsKernel<0>;
    launchChained(kernel, dim3(tiles), dim3(kDirBlock), L.total, s, ctrl, P, (u32)n, bucket, maxLevel - 1, ctx->divLevel, ctx->dirFlags, ctx->dirTotals,
                                             ctx->dirListSize, ctx->dirListKeys, ctx->dirListMeta);
    CS_LAUNCH_CHECK(ctx, "leavesLevelsKernel");
    CS_TRY(enqueueExclusiveScan(ctx, ctx->dirTotals, ctx->dirBases, tiles, s));
    launchChained(leavesEmitDirectKernel, dim3(tiles), dim3(kEmitBlock), 0, s, ctrl, P, (u32)n, ctx->divLevel, ctx->dirFlags, ctx->dirBases, tiles,
                                                       ctx->dirListSize, ctx->dirListKeys, ctx->dirListMeta,
                                                       ctx->leafK[0], ctx->leafOff[0], cap);
    CS_LAUNCH_CHECK(ctx, "leavesEmitDirectKernel");
    return CS_OK;
}

}  // namespace cs
