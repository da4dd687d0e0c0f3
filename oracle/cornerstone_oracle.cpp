// =====================================================================================
// cornerstone_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, single-threaded CPU restatement of what the hot path of
// arXiv 2307.06345 ("Cornerstone", PAPER.md) computes.  It exists only so that the
// CUDA library can be checked against it bit for bit.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// load it.  It shares no code, header, table or helper with
// paper_2307_06345_b200/csrc/ and neither side includes the other.
//
// Build: g++ -std=c++17 -O2 -ffp-contract=off -fno-fast-math -shared -fPIC
//        (see oracle/build.py).  -ffp-contract=off keeps (c-lo)/e*2^21 as three
//        separately rounded IEEE-754 binary64 operations (reading A2).
//
// Every function cites the PAPER.md passage it follows; readings of silent or garbled
// passages are the "A<n>" items of DESIGN.md ("Readings of the paper").
// Parity pins: tests/test_oracle_*.py (every function here is pinned).  O8-O10 (node properties, the
// first row past the hot path) are pinned in tests/test_oracle_props.py; O2h (Hilbert keys), the
// O8h (node cells on the Hilbert curve), L = 10, O11 (one round of the distributed build) and O12 (SFC decomposition) in
// tests/test_oracle_next.py.  PARITY UNPINNED: which 3D Hilbert curve the paper's own code walks --
// the paper names none (its reference [11] lists millions); O2h's pins fix the properties the paper
// relies on (bijection, face-continuity, octant by octant), not that choice (reading A28).
// =====================================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <utility>
#include <vector>

namespace {

// Octree depth a key resolves: "reasonable choices for L are 10 or 21" (32- or 64-bit keys).
// 21 unless orc_set_L changes it; keys are held in uint64_t either way (a key of L octal digits is < 8^L).
int L = 21;
#define KEY_END (1ull << (3 * L))           /* 8^L, PAPER.md:66 (Eq. 2) */

// length of the key range of a node at division level l: 8^(L-l)
inline uint64_t nodeRange(int level) { return 1ull << (3 * (L - level)); }

}  // namespace

extern "C" {

// L = 10 (30-bit keys) or 21 (63-bit keys); returns the previous value, or -1 if refused.
int orc_set_L(int newL)
{
    if (newL < 1 || newL > 21) return -1;
    const int old = L;
    L = newL;
    return old;
}

// -------------------------------------------------------------------------------------
// O1  bounding box.  The paper is silent (it starts from grid coordinates,
// PAPER.md:54); north_star defines the key through (xmin, xmax).  Reading A1: closed
// per-dimension [min, max] over the particles; a zero result is returned as +0.0.
// box6 = {xmin, xmax, ymin, ymax, zmin, zmax}.  Returns 0, or 1 if n == 0.
// -------------------------------------------------------------------------------------
int orc_box(const double* x, const double* y, const double* z, uint64_t n, double* box6)
{
    if (n == 0) return 1;
    const double* c[3] = {x, y, z};
    for (int d = 0; d < 3; ++d) {
        double mn = c[d][0], mx = c[d][0];
        for (uint64_t i = 1; i < n; ++i) {
            if (c[d][i] < mn) mn = c[d][i];
            if (c[d][i] > mx) mx = c[d][i];
        }
        box6[2 * d]     = mn + 0.0;   // -0.0 -> +0.0 (round-to-nearest), A1
        box6[2 * d + 1] = mx + 0.0;
    }
    return 0;
}

// -------------------------------------------------------------------------------------
// O2  Morton keys, L bits per dimension (L = 21: 63-bit keys; L = 10: 30-bit keys).
// (Sec. 3, Eq. 1): the key is L octal digits, digit i selecting the octant at division level i.
// Grid coordinate (north_star; readings A2, A3):
//     g = clamp(floor(((c - lo) / (hi - lo)) * 2^L), 0, 2^L - 1)
// evaluated in binary64, one rounding per operation, in exactly this order.
// Octal digit = 4*xbit + 2*ybit + zbit; key bit 3L-1 is x bit L-1; higher bits are 0.
// -------------------------------------------------------------------------------------
static uint32_t gridCoordinate(double c, double lo, double e)
{
    const double cells = (double)(1u << L);   // 2^L, exact
    double t = (c - lo) / e;
    t = t * cells;
    double g = std::floor(t);
    if (!(g >= 0.0)) g = 0.0;            // negatives and NaN (0/0 for a flat box, A1)
    if (g > cells - 1.0) g = cells - 1.0;   // c == hi gives exactly 2^L
    return (uint32_t)g;
}

void orc_keys(const double* x, const double* y, const double* z, uint64_t n, const double* box6,
              uint64_t* keys)
{
    const double ex = box6[1] - box6[0];
    const double ey = box6[3] - box6[2];
    const double ez = box6[5] - box6[4];
    for (uint64_t i = 0; i < n; ++i) {
        uint32_t gx = gridCoordinate(x[i], box6[0], ex);
        uint32_t gy = gridCoordinate(y[i], box6[2], ey);
        uint32_t gz = gridCoordinate(z[i], box6[4], ez);
        uint64_t k = 0;
        for (int b = 0; b < L; ++b) {     // literal bit interleave, one octal digit per bit plane
            uint64_t digit = 4ull * ((gx >> b) & 1u) + 2ull * ((gy >> b) & 1u) + ((gz >> b) & 1u);
            k |= digit << (3 * b);
        }
        keys[i] = k;
    }
}

// -------------------------------------------------------------------------------------
// O2h  Hilbert keys ("a 3D version of the Hilbert curve [11, 13]", "any type of SFC that
// traverses a cube octant by octant"; Table 1 has rows for it).  The paper gives no encoding and its
// reference [11] is an inventory of millions of 3D Hilbert curves, so the curve is a choice: reading A28
// takes the curve of the Butz algorithm in Hamilton's formulation ("compact Hilbert indices"), n = 3:
//   gc(i) = i xor (i >> 1)                         the reflected Gray code: order of the octants in a cube
//   e(w)  = 0 if w = 0, else gc(2 floor((w-1)/2))  entry corner of the w-th sub-cube
//   d(w)  = 0 if w = 0, else tsb(w-1) mod 3 (w even), tsb(w) mod 3 (w odd), tsb = number of trailing 1 bits:
//           axis along which the curve leaves the w-th sub-cube
//   T_(e,d)(b) = (b xor e) rotated right by d+1 bits (within 3 bits)
// and, level by level from the most significant bit, with l = 4 xbit + 2 ybit + zbit (as A3):
//   l' = T_(e,d)(l);  w = gc^-1(l');  key = 8 key + w;  e = e xor rotl(e(w), d+1);  d = (d + d(w) + 1) mod 3.
// The grid coordinates are those of O2.  orc_hilbert_from_grid encodes integer grid points of an m-level
// grid (pins on small grids); orc_hilbert_keys takes coordinates and the box, m = L.
// -------------------------------------------------------------------------------------
namespace {
inline unsigned gc3(unsigned i) { return i ^ (i >> 1); }
inline unsigned gc3inv(unsigned g) { unsigned i = g; i ^= i >> 1; i ^= i >> 2; return i & 7u; }
inline unsigned tsb(unsigned i) { unsigned c = 0; while (i & 1u) { ++c; i >>= 1; } return c; }
inline unsigned rotr3(unsigned b, unsigned r) { r %= 3; return ((b >> r) | (b << (3 - r))) & 7u; }
inline unsigned rotl3(unsigned b, unsigned r) { r %= 3; return ((b << r) | (b >> (3 - r))) & 7u; }
inline unsigned entry3(unsigned w) { return w == 0 ? 0u : gc3(2 * ((w - 1) / 2)); }
inline unsigned dir3(unsigned w) { return w == 0 ? 0u : ((w % 2 == 0) ? tsb(w - 1) % 3 : tsb(w) % 3); }

uint64_t hilbertOfGrid(uint32_t gx, uint32_t gy, uint32_t gz, int m)
{
    uint64_t key = 0;
    unsigned e = 0, d = 0;
    for (int i = m - 1; i >= 0; --i) {
        unsigned l = 4u * ((gx >> i) & 1u) + 2u * ((gy >> i) & 1u) + ((gz >> i) & 1u);
        l = rotr3(l ^ e, d + 1);
        const unsigned w = gc3inv(l);
        key = 8 * key + w;
        e = e ^ rotl3(entry3(w), d + 1);
        d = (d + dir3(w) + 1) % 3;
    }
    return key;
}
}  // namespace

void orc_hilbert_from_grid(const uint32_t* gx, const uint32_t* gy, const uint32_t* gz, uint64_t n, int m, uint64_t* keys)
{
    for (uint64_t i = 0; i < n; ++i) keys[i] = hilbertOfGrid(gx[i], gy[i], gz[i], m);
}

void orc_hilbert_keys(const double* x, const double* y, const double* z, uint64_t n, const double* box6, uint64_t* keys)
{
    const double ex = box6[1] - box6[0];
    const double ey = box6[3] - box6[2];
    const double ez = box6[5] - box6[4];
    for (uint64_t i = 0; i < n; ++i)
        keys[i] = hilbertOfGrid(gridCoordinate(x[i], box6[0], ex), gridCoordinate(y[i], box6[2], ey),
                                gridCoordinate(z[i], box6[4], ez), L);
}

// -------------------------------------------------------------------------------------
// O3  sort.  PAPER.md:70 ("encoding ... followed by a radix-sort"), PAPER.md:168 ("the
// particle SFC keys provided as keys and the identity permutation as values").
// Reading A5: stable; perm[j] = original index of the particle at sorted slot j.
// -------------------------------------------------------------------------------------
void orc_sort(const uint64_t* keysIn, uint64_t n, uint64_t* keysOut, uint32_t* perm)
{
    std::vector<std::pair<uint64_t, uint32_t>> kv(n);
    for (uint64_t i = 0; i < n; ++i) kv[i] = {keysIn[i], (uint32_t)i};
    std::stable_sort(kv.begin(), kv.end(),
                     [](const std::pair<uint64_t, uint32_t>& a, const std::pair<uint64_t, uint32_t>& b) {
                         return a.first < b.first;
                     });
    for (uint64_t i = 0; i < n; ++i) {
        keysOut[i] = kv[i].first;
        perm[i]    = kv[i].second;
    }
}

// -------------------------------------------------------------------------------------
// O5  one f + g round, a literal sequential transcription of Sec. 4.
//   f  (Eq. 3): N_i = number of keys of P in [K_i, K_{i+1}); counted
//      here literally with a moving cursor over the sorted P (reading A6: lower bound).
//   g1 (Eq. 5): O_i = 8 (split), 0 (merged away) or 1 (keep).
//      Readings: A7 (no split at depth L), A8 (merge iff combined count <= Ncrit),
//      A9 (the root never merges; 8*delta is formed only below the root).
//   g2 (Eq. 6): exclusive prefix sum O'.
//   g3 (Eqs. 7-9; reading A10): K'[O'_i] = K_i if O_i = 1;
//      K'[O'_i + j] = K_i + j*delta_i/8, j = 0..7, if O_i = 8; A11: K'[O'_{n_l}] = 8^L.
// K has nl+1 entries.  N (nl), O (nl), Oprime (nl+1) are outputs (may be null).
// Kout must hold capOut+1 entries.  Returns the new leaf count, or -1 if > capOut.
// -------------------------------------------------------------------------------------
namespace {
// f (Eq. 3): literal per-leaf counting with a moving cursor over the sorted keys P
void countF(const uint64_t* P, uint64_t n, const uint64_t* K, uint32_t nl, std::vector<uint32_t>& Nv)
{
    uint64_t cur = 0;
    for (uint32_t i = 0; i < nl; ++i) {
        while (cur < n && P[cur] < K[i]) ++cur;    // keys below K_0 = 0 do not exist
        uint64_t c = 0;
        while (cur < n && P[cur] < K[i + 1]) { ++cur; ++c; }
        Nv[i] = (uint32_t)c;
    }
}

// g = g3 o g2 o g1 (Eqs. 4-9) from the counts Nv.  Returns the new leaf count, or -1 if > capOut.
int64_t rebalanceG(const uint64_t* K, uint32_t nl, uint32_t bucketSize, const std::vector<uint32_t>& Nv,
                   uint32_t* O, uint32_t* Oprime, uint64_t* Kout, uint32_t capOut)
{
    std::vector<uint32_t> Ov(nl), Op(nl + 1);
    // g1
    for (uint32_t i = 0; i < nl; ++i) {
        uint64_t delta = K[i + 1] - K[i];
        if (Nv[i] > bucketSize && delta > 1) { Ov[i] = 8; continue; }
        Ov[i] = 1;
        if (delta == KEY_END) continue;             // root leaf: nothing to merge into (A9)
        uint64_t pd = 8 * delta;
        uint32_t j  = (uint32_t)((K[i] % pd) / delta);
        if (j == 0) continue;                       // "K_i is not the first octant"
        if (i < j || (uint64_t)i - j + 8 > nl) continue;
        if (K[i - j] + pd != K[i - j + 8]) continue;   // all 8 siblings are leaves
        uint64_t sum = 0;
        for (uint32_t s = 0; s < 8; ++s) sum += Nv[i - j + s];
        if (sum <= bucketSize) Ov[i] = 0;           // A8
    }
    // g2
    uint64_t run = 0;
    for (uint32_t i = 0; i < nl; ++i) { Op[i] = (uint32_t)run; run += Ov[i]; }
    Op[nl] = (uint32_t)run;
    if (O) std::copy(Ov.begin(), Ov.end(), O);
    if (Oprime) std::copy(Op.begin(), Op.end(), Oprime);
    if (run > capOut) return -1;
    // g3
    for (uint32_t i = 0; i < nl; ++i) {
        if (Ov[i] == 1) Kout[Op[i]] = K[i];
        else if (Ov[i] == 8) {
            uint64_t delta = K[i + 1] - K[i];
            for (uint32_t j = 0; j < 8; ++j) Kout[Op[i] + j] = K[i] + j * (delta / 8);
        }
    }
    Kout[run] = KEY_END;
    return (int64_t)run;
}
}  // namespace

int64_t orc_round(const uint64_t* P, uint64_t n, const uint64_t* K, uint32_t nl, uint32_t bucketSize,
                  uint32_t* N, uint32_t* O, uint32_t* Oprime, uint64_t* Kout, uint32_t capOut)
{
    std::vector<uint32_t> Nv(nl);
    countF(P, n, K, nl, Nv);
    if (N) std::copy(Nv.begin(), Nv.end(), N);
    return rebalanceG(K, nl, bucketSize, Nv, O, Oprime, Kout, capOut);
}

// -------------------------------------------------------------------------------------
// O11  one round of the distributed build, Sec. 6 (Eq. 11): the particles'
// sorted keys are spread over R ranks, shard r = Pall[shardStart[r] .. shardStart[r+1]) (each shard
// sorted on its own).  f_glob = f_r o f: every rank counts its own shard (f, Eq. 3), f_r is the
// element-wise sum of the R count arrays ("a single call to MPI_Allreduce"), then g is applied to
// the summed counts, identically on every rank.  Nglob (nl) receives the summed counts.
// -------------------------------------------------------------------------------------
int64_t orc_global_round(const uint64_t* Pall, const uint64_t* shardStart, uint32_t R, const uint64_t* K, uint32_t nl,
                         uint32_t bucketSize, uint32_t* Nglob, uint32_t* O, uint32_t* Oprime, uint64_t* Kout,
                         uint32_t capOut)
{
    std::vector<uint32_t> sum(nl, 0), Nr(nl);
    for (uint32_t r = 0; r < R; ++r) {
        countF(Pall + shardStart[r], shardStart[r + 1] - shardStart[r], K, nl, Nr);   // f on rank r
        for (uint32_t i = 0; i < nl; ++i) sum[i] += Nr[i];                            // f_r
    }
    if (Nglob) std::copy(sum.begin(), sum.end(), Nglob);
    return rebalanceG(K, nl, bucketSize, sum, O, Oprime, Kout, capOut);
}

// -------------------------------------------------------------------------------------
// O12  SFC domain decomposition: "The global domain can then be partitioned into
// n_ranks subdomains by grouping K into n_ranks bins of consecutive leaves such that each bin contains
// approximately N_tot / n_ranks of the total particle count."  The paper gives no rule for
// "approximately"; reading A29: with C_i = N_0 + ... + N_{i-1}, bin r = leaves [b_r, b_{r+1}), b_0 = 0,
// b_{n_ranks} = n_l, and for 0 < r < n_ranks b_r is the first leaf boundary i with
// C_i * n_ranks >= r * N_tot (the first boundary at or past the ideal split r N_tot / n_ranks, compared
// in exact integer arithmetic).  bounds has nRanks + 1 entries; rank r owns keys [K[b_r], K[b_{r+1}]).
// -------------------------------------------------------------------------------------
void orc_partition(const uint32_t* N, uint32_t nl, uint32_t nRanks, uint32_t* bounds)
{
    uint64_t total = 0;
    for (uint32_t i = 0; i < nl; ++i) total += N[i];
    bounds[0] = 0;
    uint64_t C = 0;          // C_i
    uint32_t i = 0;
    for (uint32_t r = 1; r < nRanks; ++r) {
        while (i < nl && (unsigned __int128)C * nRanks < (unsigned __int128)r * total) { C += N[i]; ++i; }
        bounds[r] = i;
    }
    bounds[nRanks] = nl;
}

// -------------------------------------------------------------------------------------
// O5b  iterate f, g (reading A12): start from Kstart (nlStart leaves),
// repeat rounds until a round has O_i = 1 for all i, or maxRounds rounds were done
// (maxRounds = 0: until converged).  The returned K is the output of the last round
// performed (identical to its input when that round was all ones); *rounds counts the
// rounds including the confirming one; *converged says whether the last round was all
// ones.  counts (cap entries) receives N of the returned K.
// Returns the leaf count or -1 on capacity overflow.
// -------------------------------------------------------------------------------------
int64_t orc_leaves_iterative(const uint64_t* P, uint64_t n, uint32_t bucketSize, const uint64_t* Kstart,
                             uint32_t nlStart, uint32_t maxRounds, uint64_t* Kout, uint32_t* counts,
                             uint32_t cap, uint32_t* rounds, int* converged)
{
    std::vector<uint64_t> K(Kstart, Kstart + nlStart + 1), Kn(cap + 1);
    std::vector<uint32_t> O;
    uint32_t r = 0;
    int conv = 0;
    for (;;) {
        uint32_t nl = (uint32_t)K.size() - 1;
        O.assign(nl, 0);
        int64_t nn = orc_round(P, n, K.data(), nl, bucketSize, nullptr, O.data(), nullptr, Kn.data(), cap);
        ++r;
        if (nn < 0) return -1;
        conv = 1;
        for (uint32_t i = 0; i < nl; ++i) if (O[i] != 1) { conv = 0; break; }
        K.assign(Kn.begin(), Kn.begin() + nn + 1);
        if (conv || (maxRounds && r >= maxRounds)) break;
    }
    uint32_t nl = (uint32_t)K.size() - 1;
    std::copy(K.begin(), K.end(), Kout);
    uint64_t cur = 0;                               // f on the returned array
    for (uint32_t i = 0; i < nl; ++i) {
        uint64_t c = 0;
        while (cur < n && P[cur] < K[i + 1]) { ++cur; ++c; }
        counts[i] = (uint32_t)c;
    }
    *rounds = r;
    *converged = conv;
    return nl;
}

// -------------------------------------------------------------------------------------
// O4  converged leaves by the plain definition: PAPER.md:68 and :120 define "balanced"
// (leaf counts <= Ncrit, internal-node counts > Ncrit), which is the result of a
// conventional top-down construction: node [s, s+8^(L-l)) is split iff
// it holds more than bucketSize particles and l < L (A7).  Counting is literal: every
// node walks its own particles with a cursor.
// -------------------------------------------------------------------------------------
namespace {
struct TopDown {
    const uint64_t* P; uint64_t n; uint32_t bucket;
    std::vector<uint64_t>* K; std::vector<uint32_t>* cnt;
    // a = index of the first key >= s; returns the index of the first key >= s + range
    uint64_t node(uint64_t s, int level, uint64_t a)
    {
        const uint64_t len = nodeRange(level);
        const uint64_t e = s + len;                 // level 0: 2^63, fits
        uint64_t b = a;
        while (b < n && P[b] < e) ++b;              // literal count of [s, e)
        if (b - a > bucket && level < L) {
            uint64_t cur = a;
            for (int c = 0; c < 8; ++c) cur = node(s + c * (len / 8), level + 1, cur);
            return cur;
        }
        K->push_back(s);
        cnt->push_back((uint32_t)(b - a));
        return b;
    }
};
}  // namespace

int64_t orc_leaves_topdown(const uint64_t* P, uint64_t n, uint32_t bucketSize, uint64_t* Kout,
                           uint32_t* counts, uint32_t cap)
{
    std::vector<uint64_t> K;
    std::vector<uint32_t> cnt;
    TopDown td{P, n, bucketSize, &K, &cnt};
    td.node(0, 0, 0);
    if (K.size() > cap) return -(int64_t)K.size();   // tells the caller the capacity it needs
    std::copy(K.begin(), K.end(), Kout);
    Kout[K.size()] = KEY_END;
    std::copy(cnt.begin(), cnt.end(), counts);
    return (int64_t)K.size();
}

// -------------------------------------------------------------------------------------
// O6  fully linked octree in the format of Sec. 5: node keys NK in
// Warren-Salmon placeholder-bit format (a 1 bit followed by l octal digits, PAPER.md:
// 146,152), connectivity CO = index of the first child (0 => leaf), level offsets
// LO[L+2].  The node order is the one PAPER.md:158 produces ("radix sort NK to yield a
// breadth-first node ordering", reading A16): by level, SFC order inside a level.
// Built here the plain way: explicit node objects by recursive descent over K (every
// internal node has exactly 8 children), then numbered breadth-first.
// parents[] is reading A20 (parent[0] = 0); leafToNode / nodeToLeaf are reading A23
// (nodeToLeaf = 0xFFFFFFFF for internal nodes); levelRange is reading A19.
// Arrays must hold nl + (nl-1)/7 entries.  Returns the node count or -1 if K is not a
// cornerstone array whose leaves close into an octree.
// -------------------------------------------------------------------------------------
namespace {
struct BuildNode { uint64_t start; int level; int64_t child[8]; int64_t leaf; };
struct Linker {
    const uint64_t* K = nullptr; uint32_t nl = 0; uint32_t cursor = 0; bool bad = false;
    std::vector<BuildNode> nodes;
    int64_t build(uint64_t start, int level)
    {
        int64_t id = (int64_t)nodes.size();
        nodes.push_back(BuildNode{start, level, {-1, -1, -1, -1, -1, -1, -1, -1}, -1});
        if (bad || cursor >= nl) { bad = true; return id; }
        const uint64_t len = nodeRange(level);
        if (K[cursor] == start && K[cursor + 1] == start + len) {
            nodes[id].leaf = cursor++;
            return id;
        }
        if (level == L || K[cursor] != start || K[cursor + 1] > start + len) { bad = true; return id; }
        for (int c = 0; c < 8; ++c) {
            int64_t ch = build(start + c * (len / 8), level + 1);
            nodes[id].child[c] = ch;
        }
        return id;
    }
};
}  // namespace

int64_t orc_link(const uint64_t* K, uint32_t nl, uint64_t* prefixes, uint32_t* levels, uint32_t* childOffsets,
                 uint32_t* parents, uint32_t* levelRange, uint32_t* leafToNode, uint32_t* nodeToLeaf)
{
    if (nl == 0 || K[0] != 0 || K[nl] != KEY_END) return -1;
    Linker lk;
    lk.K = K;
    lk.nl = nl;
    lk.build(0, 0);
    if (lk.bad || lk.cursor != nl) return -1;
    const std::vector<BuildNode>& nd = lk.nodes;
    const uint32_t n = (uint32_t)nd.size();
    // breadth-first numbering: queue order = level by level, key order inside a level
    std::vector<int64_t> order;  order.reserve(n);
    std::vector<uint32_t> number(n);
    order.push_back(0);
    for (size_t h = 0; h < order.size(); ++h) {
        const BuildNode& b = nd[order[h]];
        if (b.leaf < 0) for (int c = 0; c < 8; ++c) order.push_back(b.child[c]);
    }
    for (uint32_t i = 0; i < n; ++i) number[order[i]] = i;
    for (int l = 0; l <= L + 1; ++l) levelRange[l] = n;
    parents[0] = 0;
    for (uint32_t i = 0; i < n; ++i) {
        const BuildNode& b = nd[order[i]];
        prefixes[i] = (1ull << (3 * b.level)) | (b.level == 0 ? 0 : (b.start >> (3 * (L - b.level))));
        levels[i] = (uint32_t)b.level;
        if (i < levelRange[b.level]) levelRange[b.level] = i;
        if (b.leaf >= 0) {
            childOffsets[i] = 0;
            nodeToLeaf[i] = (uint32_t)b.leaf;
            leafToNode[b.leaf] = i;
        } else {
            childOffsets[i] = number[b.child[0]];
            nodeToLeaf[i] = 0xFFFFFFFFu;
            for (int c = 0; c < 8; ++c) parents[number[b.child[c]]] = i;
        }
    }
    // levels deeper than the deepest one start at n (A19); already initialised to n.
    // a level that is empty but followed by no deeper level keeps n as well.
    return n;
}

// -------------------------------------------------------------------------------------
// O7  per-node particle ranges and counts ("additional octree node
// properties, such as particle counts"; PAPER.md:258 upward pass: leaves from the
// particles, internal nodes from their children; reading A21).
// leafCounts = N of the cornerstone array (from f).  nodeFirst = index into the sorted
// particle array of the node's first particle, nodeCount = its particle count.
// Recursive over the links starting at the root.
// -------------------------------------------------------------------------------------
namespace {
struct Upsweep {
    const uint32_t* childOffsets; const uint32_t* nodeToLeaf; const std::vector<uint64_t>* leafFirst;
    const uint32_t* leafCounts; uint32_t* nodeFirst; uint32_t* nodeCount;
    void visit(uint32_t i)
    {
        if (childOffsets[i] == 0) {
            uint32_t lf = nodeToLeaf[i];
            nodeFirst[i] = (uint32_t)(*leafFirst)[lf];
            nodeCount[i] = leafCounts[lf];
            return;
        }
        uint64_t sum = 0;
        for (uint32_t c = 0; c < 8; ++c) {
            visit(childOffsets[i] + c);
            sum += nodeCount[childOffsets[i] + c];
        }
        nodeFirst[i] = nodeFirst[childOffsets[i]];
        nodeCount[i] = (uint32_t)sum;
    }
};
}  // namespace

void orc_node_counts(const uint32_t* leafCounts, uint32_t nl, const uint32_t* childOffsets,
                     const uint32_t* nodeToLeaf, uint32_t numNodes, uint32_t* nodeFirst, uint32_t* nodeCount)
{
    (void)numNodes;
    std::vector<uint64_t> leafFirst(nl + 1, 0);
    for (uint32_t i = 0; i < nl; ++i) leafFirst[i + 1] = leafFirst[i] + leafCounts[i];
    Upsweep up{childOffsets, nodeToLeaf, &leafFirst, leafCounts, nodeFirst, nodeCount};
    up.visit(0);
}


// -------------------------------------------------------------------------------------
// O8  node geometry (NEXT-1 of SURVEY 8f; "additional node properties ...
// stored in separate arrays of length n").  A node with placeholder-bit key NK (a 1 followed
// by `level` octal digits) is the cell (ix, iy, iz) of the 2^level grid over
// the bounding box; digit = 4*xbit + 2*ybit + zbit (A3).  Reading A25: cell edge
// h_d = (hi_d - lo_d) / 2^level, centre c_d = lo_d + (i_d + 0.5) * h_d, half size 0.5 * h_d,
// each operation rounded once in binary64 (no contraction).  SoA outputs: centers[3][n],
// halfSizes[3][n].
// -------------------------------------------------------------------------------------
void orc_node_geometry(const uint64_t* prefixes, uint32_t n, const double* box6, double* centers, double* halfSizes)
{
    for (uint32_t i = 0; i < n; ++i) {
        const uint64_t p = prefixes[i];
        int bits = 0;
        while ((p >> bits) > 1) ++bits;                  // position of the placeholder bit
        const int level = bits / 3;
        uint64_t g[3] = {0, 0, 0};
        for (int l = 1; l <= level; ++l) {               // octal digits, most significant first
            const unsigned digit = (unsigned)((p >> (3 * (level - l))) & 7u);
            g[0] = (g[0] << 1) | ((digit >> 2) & 1u);
            g[1] = (g[1] << 1) | ((digit >> 1) & 1u);
            g[2] = (g[2] << 1) | (digit & 1u);
        }
        const double cells = (double)(1ull << level);
        for (int d = 0; d < 3; ++d) {
            const double lo = box6[2 * d], e = box6[2 * d + 1] - box6[2 * d];
            const double h = e / cells;
            centers[(size_t)d * n + i] = lo + ((double)g[d] + 0.5) * h;
            halfSizes[(size_t)d * n + i] = 0.5 * h;
        }
    }
}

// -------------------------------------------------------------------------------------
// O8h  node geometry for Hilbert keys (reading A28): the node's cell is found by walking the curve of O2h
// backwards, digit by digit from the most significant: in orientation (e, d) the w-th sub-cube of the
// curve is the octant l = T_(e,d)^-1(gc(w)) = rotl(gc(w), d+1) xor e (the inverse of l' = T_(e,d)(l),
// w = gc^-1(l')), with l = 4 xbit + 2 ybit + zbit; (e, d) are updated as in O2h.  The arithmetic on the
// cell is O8's (A25).
// -------------------------------------------------------------------------------------
void orc_node_geometry_hilbert(const uint64_t* prefixes, uint32_t n, const double* box6, double* centers,
                               double* halfSizes)
{
    for (uint32_t i = 0; i < n; ++i) {
        const uint64_t p = prefixes[i];
        int bits = 0;
        while ((p >> bits) > 1) ++bits;
        const int level = bits / 3;
        uint64_t g[3] = {0, 0, 0};
        unsigned e = 0, d = 0;
        for (int l = 1; l <= level; ++l) {
            const unsigned w = (unsigned)((p >> (3 * (level - l))) & 7u);
            const unsigned oct = rotl3(gc3(w), d + 1) ^ e;
            g[0] = (g[0] << 1) | ((oct >> 2) & 1u);
            g[1] = (g[1] << 1) | ((oct >> 1) & 1u);
            g[2] = (g[2] << 1) | (oct & 1u);
            e = e ^ rotl3(entry3(w), d + 1);
            d = (d + dir3(w) + 1) % 3;
        }
        const double cells = (double)(1ull << level);
        for (int k = 0; k < 3; ++k) {
            const double lo = box6[2 * k], ext = box6[2 * k + 1] - box6[2 * k];
            const double h = ext / cells;
            centers[(size_t)k * n + i] = lo + ((double)g[k] + 0.5) * h;
            halfSizes[(size_t)k * n + i] = 0.5 * h;
        }
    }
}

// -------------------------------------------------------------------------------------
// O9  centres of mass by an upward pass ("properties where the leaves depend
// on the contained particles and internal nodes on their children ... center-of-mass for
// gravity").  Unit masses (the path carries coordinates only).  Reading A26: a leaf's centre
// is the sum of its particles' coordinates, taken in sorted order (xs = x[perm], first ..
// first + count - 1), divided by count; an internal node's is sum_c count_c * com_c over its 8
// children in order, divided by its count; a node without particles takes its geometric
// centre.  Nodes are visited from the last index to the first: children have larger indices
// than their parent in the breadth-first layout.
// -------------------------------------------------------------------------------------
void orc_centers_of_mass(const double* xs, const double* ys, const double* zs, const uint32_t* nodeFirst,
                         const uint32_t* nodeCount, const uint32_t* childOffsets, const double* centers, uint32_t n,
                         double* com)
{
    const double* c[3] = {xs, ys, zs};
    for (uint32_t ii = n; ii-- > 0;) {
        for (int d = 0; d < 3; ++d) {
            double s = 0.0;
            if (nodeCount[ii] == 0) {
                com[(size_t)d * n + ii] = centers[(size_t)d * n + ii];
                continue;
            }
            if (childOffsets[ii] == 0) {
                for (uint32_t j = nodeFirst[ii]; j < nodeFirst[ii] + nodeCount[ii]; ++j) s = s + c[d][j];
            } else {
                for (uint32_t k = 0; k < 8; ++k) {
                    const uint32_t ch = childOffsets[ii] + k;
                    s = s + (double)nodeCount[ch] * com[(size_t)d * n + ch];
                }
            }
            com[(size_t)d * n + ii] = s / (double)nodeCount[ii];
        }
    }
}

// -------------------------------------------------------------------------------------
// O10  minimum-distance MAC, Eq. 12: fulfilled if r_min > l / theta, with
// r_min the minimum distance between source node and target, l the source node's edge
// length.  Target = an axis-aligned focus box F ("with respect to any point in
// F").  Reading A27: per dimension the gap between the two boxes is
// max(|c - fc| - (h + fh), 0) with fc, fh centre and half size of F; r_min^2 is the sum of the
// squared gaps (x, y, z in that order); l = 2 * max(hx, hy, hz) (the boxes need not be cubes);
// the decision is taken without the square root, as (r_min^2 * (theta * theta)) > (l * l),
// every operation rounded once in binary64.  pass[i] = 1 if fulfilled.
// -------------------------------------------------------------------------------------
void orc_mac_min_distance(const double* centers, const double* halfSizes, uint32_t n, const double* focus6, double theta,
                          uint8_t* pass)
{
    const double t2 = theta * theta;
    for (uint32_t i = 0; i < n; ++i) {
        double r2 = 0.0, hmax = 0.0;
        for (int d = 0; d < 3; ++d) {
            const double fc = 0.5 * (focus6[2 * d] + focus6[2 * d + 1]), fh = 0.5 * (focus6[2 * d + 1] - focus6[2 * d]);
            const double cc = centers[(size_t)d * n + i], h = halfSizes[(size_t)d * n + i];
            double gap = std::fabs(cc - fc) - (h + fh);
            if (!(gap > 0.0)) gap = 0.0;
            r2 = r2 + gap * gap;
            if (h > hmax) hmax = h;
        }
        const double l = 2.0 * hmax;
        pass[i] = (r2 * t2 > l * l) ? 1 : 0;
    }
}

}  // extern "C"
