/* =====================================================================================
 * cornerstone.h -- C ABI of the B200-native Cornerstone octree builder.
 *
 * One data-parallel hot path of arXiv 2307.06345: single-GPU construction of
 * the cornerstone octree from particle coordinates,
 *
 *   coordinates -> bounding box -> 64-bit Morton keys -> stable radix sort (+ permutation)
 *               -> cornerstone leaf array K by iterating f, g -> linked octree -> node counts
 *
 * Every entry point is extern "C", takes plain pointers and sizes, and never throws or
 * aborts: the return code is the only error channel (cs_lastError gives the text).
 *
 * Conventions
 *   - "dev" pointers are CUDA device pointers owned by the caller (e.g. a torch tensor's
 *     data_ptr()); the library never frees them and keeps no reference after the call.
 *     "host" pointers are ordinary host memory.  Scratch memory lives in the context.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *     Calls enqueue work on `stream`.  A call with a *host out* argument synchronises
 *     `stream` before returning; calls without one return as soon as the work is enqueued.
 *   - L = 21: keys are 63-bit Morton codes in a uint64_t, 8^21 = 2^63 is the
 *     terminal element of a cornerstone array (Eq. 2).
 *   - Arrays are structure-of-arrays, densely packed, naturally aligned; x, y, z, keys and
 *     leaves must be 16-byte aligned (any cudaMalloc / torch allocation is).
 *   - n < 2^32 particles (indices are uint32_t).
 *   - One stream at a time per context: all calls on a context share its workspace, and calls without a host
 *     out argument return before their work is done, so a context must not be used from two streams or host
 *     threads at once (calls are ordered only within the stream they are given).  Use one context per stream.
 * ===================================================================================== */
#ifndef CORNERSTONE_B200_H
#define CORNERSTONE_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CS_MAX_LEVEL 21u               /* L */
#define CS_KEY_END (1ull << 63)        /* 8^L */
#define CS_NUM_LEVEL_OFFSETS 23u       /* L + 2 entries of the level-offset array LO */
#define CS_NO_LEAF 0xFFFFFFFFu         /* nodeToLeaf[] of an internal node */

typedef struct cs_context cs_context;  /* opaque; owns the workspace; bound to one device */

typedef enum cs_status {
    CS_OK = 0,
    CS_ERR_INVALID_ARG = 1,      /* null pointer, n == 0 where a box is needed, n >= 2^32, bucketSize == 0 */
    CS_ERR_CAPACITY = 2,         /* result exceeds leafCapacity / the context's maxLeaves / maxParticles */
    CS_ERR_NOT_CORNERSTONE = 3,  /* prevLeaves / leaves violates Eq. 2 */
    CS_ERR_NOT_CONVERGED = 4,    /* maxRounds reached before a round with O_i = 1 for all i */
    CS_ERR_CUDA = 5              /* a CUDA runtime call failed; see cs_lastError */
} cs_status;

/* Stage identifiers for cs_stageTimes (milliseconds of device time, CUDA events). */
enum {
    CS_STAGE_BOX = 0, CS_STAGE_KEYS = 1, CS_STAGE_SORT = 2, CS_STAGE_LEAVES = 3, CS_STAGE_LINK = 4,
    CS_STAGE_COUNTS = 5, CS_STAGE_SORT_HIST = 6,
    CS_STAGE_SORT_PASSES = 7,    /* the plain radix passes: 2, 3 or 4 (tiny / short / default plan) or 7 (plain plan) */
    CS_STAGE_SORT_FIXUP = 8,     /* tiny / short / default plan: the last pass, which also orders the low bits, + the gated redo launch */
    CS_NUM_STAGES = 9
};

/* ---- context ------------------------------------------------------------------------ */

/* Bytes of device workspace cs_create will allocate for these capacities. */
size_t cs_workspaceBytes(uint64_t maxParticles, uint32_t maxLeaves);

/* Create a context on CUDA device `device` able to process up to maxParticles particles and
 * trees of up to maxLeaves leaves.  Allocates the workspace (cudaMalloc) once. */
cs_status cs_create(cs_context** ctx, int device, uint64_t maxParticles, uint32_t maxLeaves);
void cs_destroy(cs_context* ctx);

/* Text of the last error on this context ("" if none).  ctx may be NULL (global text). */
const char* cs_lastError(const cs_context* ctx);
const char* cs_version(void);

/* Enable (1) / disable (0) per-stage CUDA-event timing; read it back after the stream is
 * idle.  ms[CS_NUM_STAGES], host.  Stages not run since the last reset read 0.
 * launches (host, nullable) receives the number of kernels the library has launched on
 * this context since cs_create. */
cs_status cs_setProfiling(cs_context* ctx, int enabled);
cs_status cs_stageTimes(cs_context* ctx, float* ms, uint64_t* launches);

/* ---- stages of the path ----------------------------------------------------------------
 *
 * cs_computeBox -- per-dimension closed bounding box [min, max] of the particles.
 *   The paper starts from grid coordinates and is silent on the box; the key
 *   definition of BASELINE.json:north_star needs (xmin, xmax) per dimension (A1).
 *   x, y, z: dev, n doubles each, finite.  box6: dev, 6 doubles out
 *   {xmin, xmax, ymin, ymax, zmin, zmax}; a zero extreme is returned as +0.0.
 *   Errors: INVALID_ARG (null, n == 0, n >= 2^32), CAPACITY (n > maxParticles), CUDA.
 */
cs_status cs_computeBox(cs_context* ctx, const double* x, const double* y, const double* z, uint64_t n,
                        double* box6, void* stream);

/* cs_computeKeys -- 64-bit Morton keys, 21 bits per dimension (Eq. 1).
 *   g_d = clamp(floor(((c_d - lo_d) / (hi_d - lo_d)) * 2^21), 0, 2^21 - 1) in IEEE binary64,
 *   one rounding per operation in that order, no FMA contraction (A2);
 *   octal digit = 4*xbit + 2*ybit + zbit, key bit 62 = x bit 20, bit 63 = 0 (A3).
 *   A flat dimension (hi == lo) maps to grid coordinate 0 (A1).
 *   box6: dev (as written by cs_computeBox, or any user box).  keys: dev, n uint64 out.
 */
cs_status cs_computeKeys(cs_context* ctx, const double* x, const double* y, const double* z, uint64_t n,
                         const double* box6, uint64_t* keys, void* stream);

/* cs_computeKeysHilbert -- keys on a 3D Hilbert curve instead of the Morton Z-curve (Table 1
 *   has rows for both).  Same grid coordinates g_d as cs_computeKeys; the key is again 21 octal digits and its
 *   first i digits name the level-i cell that holds the particle ("any type of SFC that traverses a cube octant
 *   by octant"), so cs_sortKeys, cs_buildLeaves, cs_linkOctree and cs_nodeCounts apply unchanged.
 *   The paper gives no encoding; reading A28 takes the curve of the Butz algorithm in Hamilton's
 *   formulation: octants of a cube in reflected-Gray-code order, sub-cube w entered at corner e(w) and left
 *   along axis d(w).  Cells of consecutive keys share a face.  Arguments and errors as cs_computeKeys.
 *   (Node cells of such a tree: cs_nodeGeometryHilbert.) */
cs_status cs_computeKeysHilbert(cs_context* ctx, const double* x, const double* y, const double* z, uint64_t n,
                                const double* box6, uint64_t* keys, void* stream);

/* cs_setCurve -- the curve cs_buildOctree / cs_buildOctreeHost compute their keys on (default CS_CURVE_MORTON). */
enum { CS_CURVE_MORTON = 0, CS_CURVE_HILBERT = 1 };
cs_status cs_setCurve(cs_context* ctx, int curve);

/* cs_sortKeys -- stable ascending radix sort of the keys, carrying the particle index
 *   ("keys ... and the identity permutation as values"; A5).
 *   keys: dev, in: n keys < 2^63 in any order, out: sorted.  perm: dev, n uint32 out,
 *   perm[j] = original index of the particle now at sorted slot j (equal keys keep their
 *   original relative order).  n == 0 is a no-op.
 */
cs_status cs_sortKeys(cs_context* ctx, uint64_t* keys, uint32_t* perm, uint64_t n, void* stream);

/* cs_setSortMode -- how cs_sortKeys / cs_buildOctree reach the (unique) stable order.  The keys are 7 digits of 9
 *   bits.  A plan with first digit F runs radix passes over the digits F .. 6 only; the last of them also orders the
 *   bits below 9 F inside every run of equal leading digits.  If some run is longer than 257 elements, one more launch
 *   behind it redoes the sort with the 7 plain passes, decided on the device with no host round trip; the context
 *   learns of it (cs_buildOctree reads it with its sizes; after cs_sortKeys it follows the stream to the host).
 *   CS_SORT_AUTO (default): a ladder over the plans, finest first: the tiny plan (F = 4: 3 passes; fits while no cell
 *   of octree level 9 holds more than 257 particles: uniform particles, up to billions of them), the short plan
 *   (F = 3: 4 passes; level 12), the default plan (F = 2: 5 passes; level 15).  After a plan had to be redone the
 *   context uses the next one for the next 256 sorts, then tries the finer one again (512, 1024, ... sorts after every
 *   further failure, at most 16384; a plan is not retried while a coarser one still fails); after the default plan had
 *   to be redone, the 7 plain passes for 16 sorts.
 *   CS_SORT_DEFAULT: as CS_SORT_AUTO without the tiny and the short plan.  CS_SORT_SHORT, CS_SORT_TINY: always that plan
 *   (redone when it does not fit).  CS_SORT_PLAIN: always the 7 plain LSD passes.
 *   Setting a mode also forgets earlier redos.  The sorted keys and perm are identical in all modes.
 *   Errors: INVALID_ARG. */
enum { CS_SORT_AUTO = 0, CS_SORT_PLAIN = 1, CS_SORT_DEFAULT = 2, CS_SORT_SHORT = 3, CS_SORT_TINY = 4 };
cs_status cs_setSortMode(cs_context* ctx, int mode);
/* Plain radix passes of the next sort on this context (the ones CS_STAGE_SORT_PASSES times): 2, 3 or 4 (followed by
 * the fused last pass) or 7 (0 if ctx is NULL). */
int cs_sortPasses(const cs_context* ctx);

/* cs_buildLeaves -- cornerstone leaf array by alternating f (Eq. 3) and g = g3 o g2 o g1
 *   (Eqs. 4-9), until a round reports O_i = 1 for all i.
 *   sortedKeys: dev, n ascending keys < 2^63 (the array P).  bucketSize = N_crit >= 1.
 *   prevLeaves: dev, nullable.  NULL: start from the root {0, 8^21}.  Otherwise a valid
 *   cornerstone array with prevNumLeaves leaves (prevNumLeaves+1 keys), e.g. the previous
 *   time step's; it is validated against Eq. 2.
 *   maxRounds: 0 = iterate until converged (at most L+1 = 22 rounds are ever needed);
 *   k > 0 = at most k rounds; maxRounds = 1 is the paper's "single histogram count and
 *   rebalance update".  If the last round performed was not all-ones the
 *   outputs hold that round's result and the status is CS_ERR_NOT_CONVERGED.
 *   Readings: split only below depth L (A7); merge iff the 8 siblings hold <= bucketSize
 *   particles together (A8); the root never merges (A9); K'[O'_i + j] = K_i + j*delta_i/8 (A10).
 *   leaves: dev out, numLeaves+1 keys (capacity leafCapacity+1).  counts: dev out, N_i for
 *   the returned leaves (capacity leafCapacity).  numLeaves, rounds: host out (rounds counts
 *   f evaluations including the confirming one).  Synchronises `stream`.
 *   Errors: CAPACITY if a round would exceed leafCapacity or the context's maxLeaves
 *   (leaves / counts are then left untouched when the build started from the root; with prevLeaves
 *   they may hold the array of an earlier round), NOT_CORNERSTONE, INVALID_ARG, CUDA.
 *   Cost: from the root (default mode) one pass over sortedKeys.  With prevLeaves: one merge pass over
 *   sortedKeys and prevLeaves that locates every previous K_i (Eq. 3), then the rounds, all in one
 *   cooperative launch that ends with the first round that changes nothing: a small time step costs
 *   one update and the confirming round.
 */
cs_status cs_buildLeaves(cs_context* ctx, const uint64_t* sortedKeys, uint64_t n, uint32_t bucketSize,
                         const uint64_t* prevLeaves, uint32_t prevNumLeaves, uint32_t maxRounds,
                         uint64_t* leaves, uint32_t* counts, uint32_t leafCapacity,
                         uint32_t* numLeaves, uint32_t* rounds, void* stream);

/* cs_setLeafMode -- how cs_buildLeaves / cs_buildOctree reach the converged array when they
 *   start from the root (prevLeaves == NULL, maxRounds == 0).  From {0, 8^21} the rounds of
 *   PAPER.md:120-126 only ever split, so their fixpoint is the top-down tree "a node above
 *   depth L is internal iff it holds more than bucketSize particles".
 *   CS_LEAVES_AUTO (default): that fixpoint is computed in ONE pass over the sorted keys (a
 *   node holds more than b particles iff it contains b+1 consecutive keys of P); leaves,
 *   counts and `rounds` (deepest leaf level + 1) are identical to what the rounds return.
 *   bucketSize > 1024 falls back to the rounds.
 *   CS_LEAVES_ITERATIVE: always run the rounds f, g1, g2, g3 (Eqs. 3-9) literally.
 *   Incremental starts (prevLeaves) and bounded round counts (maxRounds > 0) always use the
 *   rounds.  Errors: INVALID_ARG. */
enum { CS_LEAVES_AUTO = 0, CS_LEAVES_ITERATIVE = 1 };
cs_status cs_setLeafMode(cs_context* ctx, int mode);

/* cs_linkOctree -- the fully linked octree of Sec. 5, all levels in
 *   parallel, in the paper's format: node keys NK in Warren-Salmon placeholder-bit form
 *   (a 1 bit followed by `level` octal digits), connectivity CO (index of
 *   the first of 8 children, 0 = leaf), level offsets LO[L+2].
 *   Node order = ascending placeholder key = breadth-first, SFC order within a level
 *   (A16).  numNodes = numLeaves + (numLeaves-1)/7.
 *   leaves: dev, numLeaves+1 keys forming a closed octree.  All outputs dev, sized numNodes
 *   unless noted: prefixes (NK), levels, childOffsets (CO), parents (parent[0] = 0; A20),
 *   levelRange[23] (LO; entries past the deepest level = numNodes; A19),
 *   leafToNode[numLeaves], nodeToLeaf[numNodes] (CS_NO_LEAF for internal nodes; A23).
 *   levels, parents, leafToNode, nodeToLeaf may be NULL (not produced).
 *   numNodes: host out.  nodeCapacity: capacity of the per-node arrays.  Synchronises.
 *   Errors: NOT_CORNERSTONE ((numLeaves-1) mod 7 != 0 or the leaves do not close into an
 *   octree), CAPACITY, INVALID_ARG, CUDA.
 */
cs_status cs_linkOctree(cs_context* ctx, const uint64_t* leaves, uint32_t numLeaves,
                        uint64_t* prefixes, uint32_t* levels, uint32_t* childOffsets, uint32_t* parents,
                        uint32_t* levelRange, uint32_t* leafToNode, uint32_t* nodeToLeaf,
                        uint32_t nodeCapacity, uint32_t* numNodes, void* stream);

/* cs_nodeCounts -- per-node particle range in the sorted particle array (PAPER.md:80, 192,
 *   258; A21): nodeFirst[i] = lower_bound(P, start_i), nodeCount[i] = lower_bound(P, end_i)
 *   - nodeFirst[i], where [start_i, end_i) is the key range encoded by prefixes[i].
 *   sortedKeys: dev, n.  prefixes: dev, numNodes placeholder-bit keys (from cs_linkOctree).
 *   Optional accelerator (both or neither): leafCounts[numLeaves] as returned by
 *   cs_buildLeaves for the same leaves, and nodeToLeaf[numNodes] from cs_linkOctree; leaf
 *   nodes then take their range from the prefix sum of leafCounts instead of searching P
 *   (the two definitions coincide).  Does not synchronise.
 */
cs_status cs_nodeCounts(cs_context* ctx, const uint64_t* sortedKeys, uint64_t n,
                        const uint64_t* prefixes, uint32_t numNodes,
                        const uint32_t* leafCounts, const uint32_t* nodeToLeaf, uint32_t numLeaves,
                        uint32_t* nodeFirst, uint32_t* nodeCount, void* stream);

/* ---- the whole path in one call ---------------------------------------------------------
 *
 * Output buffers of a full build.  All dev, caller-owned.  Per-leaf arrays hold leafCapacity
 * (+1 for leaves) entries, per-node arrays nodeCapacity entries. */
typedef struct cs_octree_buffers {
    double*   box6;          /* [6]   out */
    uint64_t* keys;          /* [n]   out: sorted keys P */
    uint32_t* perm;          /* [n]   out: permutation */
    uint64_t* leaves;        /* [leafCapacity + 1] out: K */
    uint32_t* counts;        /* [leafCapacity]     out: N */
    uint64_t* prefixes;      /* [nodeCapacity] out: NK */
    uint32_t* levels;        /* [nodeCapacity] out (nullable) */
    uint32_t* childOffsets;  /* [nodeCapacity] out: CO */
    uint32_t* parents;       /* [nodeCapacity] out (nullable) */
    uint32_t* levelRange;    /* [23] out: LO */
    uint32_t* leafToNode;    /* [leafCapacity] out (nullable) */
    uint32_t* nodeToLeaf;    /* [nodeCapacity] out */
    uint32_t* nodeFirst;     /* [nodeCapacity] out */
    uint32_t* nodeCount;     /* [nodeCapacity] out */
    uint32_t  leafCapacity;
    uint32_t  nodeCapacity;
} cs_octree_buffers;

typedef struct cs_octree_sizes {
    uint32_t numLeaves;
    uint32_t numNodes;
    uint32_t rounds;
    uint32_t converged;
} cs_octree_sizes;

/* cs_buildOctree -- box, keys, sort, leaves, link and node counts back to back on `stream`
 *   with every intermediate size kept on the device: no host round trip until the single
 *   synchronisation at the end that fills *sizes (host out).  Semantics of each stage are
 *   exactly those of the stage calls above (prevLeaves / prevNumLeaves / maxRounds as in
 *   cs_buildLeaves; prevLeaves may alias buffers->leaves).
 *   x, y, z: dev.  Errors: as the stages; on error the buffers hold unspecified data.
 */
cs_status cs_buildOctree(cs_context* ctx, const double* x, const double* y, const double* z, uint64_t n,
                         uint32_t bucketSize, const uint64_t* prevLeaves, uint32_t prevNumLeaves,
                         uint32_t maxRounds, const cs_octree_buffers* buffers, cs_octree_sizes* sizes,
                         void* stream);

/* cs_setGraphLimit -- cs_buildOctree calls with at most maxParticles particles (default 2^32: every call) are captured
 *   as ONE CUDA graph when the same arguments (pointers, sizes, modes, stream) are seen twice in a row, and replayed
 *   while they stay the same: small builds are bound by the cost of launching some 20 kernels, not by the device (a
 *   build of 2^16 particles takes 0.16 ms enqueued kernel by kernel, 0.13 ms replayed), and large ones still gain the
 *   gaps between their kernels (2^24: 0.976 -> 0.961 ms, 2^26: 3.76 -> 3.75 ms).  Results are identical.  0 switches
 *   graphs off.
 *   Calls with cs_setProfiling enabled are never replayed (the stage timers need the separate launches). */
cs_status cs_setGraphLimit(cs_context* ctx, uint64_t maxParticles);

/* cs_buildOctreeHost -- the same path for HOST coordinate buffers (end-to-end form):
 *   copies x, y, z host -> device, runs cs_buildOctree into context-owned device buffers
 *   (the context must have been created with capacities covering n and the tree), and
 *   copies the tree back into the caller's HOST arrays.  `host` has the layout of
 *   cs_octree_buffers but every pointer is host memory; NULL members are not copied back.
 *   Pinned (page-locked) host memory gives the full PCIe rate; pageable memory works.  Inputs above the graph limit
 *   (cs_setGraphLimit) are uploaded in 8 pieces on a second stream and the bounding box is reduced piece by piece under
 *   the upload; everything after the box needs all of it, so the rest of the build follows the upload.
 */
cs_status cs_buildOctreeHost(cs_context* ctx, const double* x, const double* y, const double* z, uint64_t n,
                             uint32_t bucketSize, const cs_octree_buffers* host, cs_octree_sizes* sizes,
                             void* stream);

/* ---- 32-bit keys: L = 10 ("reasonable choices for L are 10 or 21") --------------------------------
 *
 * The same path with keys of 10 octal digits (30 bits, in a uint32_t): the tree resolves 10 levels, 8^10 = 2^30
 * terminates a cornerstone array, leaves at level 10 may hold more than bucketSize particles (A7), prefixes are
 * placeholder-bit keys of at most 31 bits.  The grid coordinate is clamp(floor(((c - lo) / (hi - lo)) * 2^10), 0,
 * 2^10 - 1) with the same quotient as for L = 21, so a 30-bit key equals the 63-bit key of the same particle
 * shifted right by 33 bits.  The sort moves 8 instead of 12 bytes per element and needs 4 passes of 9-bit digits.
 * Arguments, ownership, synchronisation and errors are those of the 64-bit calls of the same name; levelRange
 * still has CS_NUM_LEVEL_OFFSETS entries (those past level 11 equal numNodes).  The tree stages widen keys and
 * leaf arrays into the context's workspace (the first call allocates 26 bytes per leaf of capacity for it).
 */
#define CS_MAX_LEVEL32 10u
#define CS_KEY_END32 (1u << 30)

/* curve: CS_CURVE_MORTON or CS_CURVE_HILBERT */
cs_status cs_computeKeys32(cs_context* ctx, const double* x, const double* y, const double* z, uint64_t n,
                           const double* box6, int curve, uint32_t* keys, void* stream);
cs_status cs_sortKeys32(cs_context* ctx, uint32_t* keys, uint32_t* perm, uint64_t n, void* stream);
cs_status cs_buildLeaves32(cs_context* ctx, const uint32_t* sortedKeys, uint64_t n, uint32_t bucketSize,
                           const uint32_t* prevLeaves, uint32_t prevNumLeaves, uint32_t maxRounds, uint32_t* leaves,
                           uint32_t* counts, uint32_t leafCapacity, uint32_t* numLeaves, uint32_t* rounds, void* stream);
cs_status cs_linkOctree32(cs_context* ctx, const uint32_t* leaves, uint32_t numLeaves, uint32_t* prefixes,
                          uint32_t* levels, uint32_t* childOffsets, uint32_t* parents, uint32_t* levelRange,
                          uint32_t* leafToNode, uint32_t* nodeToLeaf, uint32_t nodeCapacity, uint32_t* numNodes,
                          void* stream);

typedef struct cs_octree_buffers32 {   /* cs_octree_buffers with 32-bit keys, leaves and prefixes */
    double*   box6;
    uint32_t* keys;
    uint32_t* perm;
    uint32_t* leaves;
    uint32_t* counts;
    uint32_t* prefixes;
    uint32_t* levels;        /* nullable */
    uint32_t* childOffsets;
    uint32_t* parents;       /* nullable */
    uint32_t* levelRange;
    uint32_t* leafToNode;    /* nullable */
    uint32_t* nodeToLeaf;
    uint32_t* nodeFirst;
    uint32_t* nodeCount;
    uint32_t  leafCapacity;
    uint32_t  nodeCapacity;
} cs_octree_buffers32;

/* box, 30-bit keys (on the curve of cs_setCurve), sort, leaves from {0, 8^10}, links and node counts in one call. */
cs_status cs_buildOctree32(cs_context* ctx, const double* x, const double* y, const double* z, uint64_t n,
                           uint32_t bucketSize, const cs_octree_buffers32* buffers, cs_octree_sizes* sizes,
                           void* stream);

/* ---- the distributed build of Sec. 6, as the calls ONE rank makes (Eq. 11) -----------------------
 *
 * "Let us assume that the particles are distributed across multiple compute nodes ... f_glob = f_r o f, where f is
 * applied to the particles on each node separately and f_r is the element-wise sum of the counts arrays ... computed
 * with a single call to MPI_Allreduce.  Then we can apply g to N and K as before".  The library
 * offers f and g as separate calls so that the caller's collective sits between them; it does not communicate:
 *
 *     cs_countLeaves(ctx, myKeys, n, K, nl, N)                    f on this rank's particles (async)
 *     all-reduce(sum, uint32, nl) of N over the ranks             f_r, the caller's (e.g. ncclAllReduce on `stream`)
 *     cs_rebalance(ctx, K, N, nl, bucket, K', cap, &nl', &changed)  g: identical on every rank
 *     ... repeat with K', nl' while changed ...
 *     cs_partitionLeaves(ctx, N, nl, numRanks, bounds)            SFC domain decomposition
 *     cs_linkOctree(K ...), cs_nodeCountsFromLeaves(K, N ...)     the replicated global octree and its node counts
 *
 * All array arguments are device pointers owned by the caller.
 */

/* cs_countLeaves -- f alone (Eq. 3): counts[i] = number of keys of sortedKeys in [K_i, K_{i+1}).
 *   sortedKeys: n ascending keys (this rank's particles).  leaves: numLeaves + 1 keys of a cornerstone array
 *   (precondition: ascending; Eq. 2 is checked by cs_rebalance).  counts: numLeaves uint32 out.
 *   One merge pass over sortedKeys and leaves.  Does not synchronise.
 *   Errors: INVALID_ARG, CAPACITY (n > maxParticles, numLeaves > maxLeaves), CUDA. */
cs_status cs_countLeaves(cs_context* ctx, const uint64_t* sortedKeys, uint64_t n, const uint64_t* leaves,
                         uint32_t numLeaves, uint32_t* counts, void* stream);

/* cs_rebalance -- g = g3 o g2 o g1 alone (Eqs. 4-9) on leaves K and given counts N (any counts: one
 *   rank's, or the element-wise sum over ranks of Eq. 11).  g1: O_i = 8 if N_i > bucketSize and the leaf is above
 *   depth L (A7); 0 if the leaf is not the first of 8 sibling leaves that hold <= bucketSize particles together (A8;
 *   the root never merges, A9); else 1.  g2: exclusive prefix sum O'.  g3: K'[O'_i] = K_i, or K'[O'_i + j] = K_i +
 *   j delta_i / 8 for j = 0..7 (A10); K'[O'_{nl}] = 8^21 (A11).
 *   newLeaves: out, capacity leafCapacity + 1, must not alias leaves.  newNumLeaves, changed: host out; changed = 0
 *   iff O_i = 1 for all i (the confirming round: then newLeaves == leaves).  Synchronises `stream`.
 *   Errors: NOT_CORNERSTONE (leaves violate Eq. 2), CAPACITY (result exceeds leafCapacity or the context's maxLeaves;
 *   newLeaves untouched), INVALID_ARG, CUDA. */
cs_status cs_rebalance(cs_context* ctx, const uint64_t* leaves, const uint32_t* counts, uint32_t numLeaves,
                       uint32_t bucketSize, uint64_t* newLeaves, uint32_t leafCapacity, uint32_t* newNumLeaves,
                       uint32_t* changed, void* stream);

/* cs_partitionLeaves -- SFC domain decomposition: "the global domain can then be partitioned into n_ranks subdomains
 *   by grouping K into n_ranks bins of consecutive leaves such that each bin contains approximately N_tot / n_ranks
 *   of the total particle count".  The paper gives no rule for "approximately"; DESIGN.md reading
 *   A29: with C_i = N_0 + ... + N_{i-1}, bounds[0] = 0, bounds[numRanks] = numLeaves and, for 0 < r < numRanks,
 *   bounds[r] = the first leaf boundary i with C_i * numRanks >= r * N_tot (exact integer comparison).  Rank r owns
 *   the leaves [bounds[r], bounds[r+1]), i.e. the keys [K[bounds[r]], K[bounds[r+1]]).
 *   counts: numLeaves uint32 (their sum may exceed 2^32).  bounds: numRanks + 1 uint32 out.  Does not synchronise. */
cs_status cs_partitionLeaves(cs_context* ctx, const uint32_t* counts, uint32_t numLeaves, uint32_t numRanks,
                             uint32_t* bounds, void* stream);

/* cs_partitionLeavesStatic -- cs_partitionLeaves for callers that must not allocate (code under CUDA graph capture,
 *   serving loops, harnesses that forbid cudaMalloc): same arguments without the context, same result (PAPER.md:202-204,
 *   reading A29), and no cudaMalloc / cudaFree or allocating library call on any path: there is no context, and the
 *   kernel's scratch (one 64-bit sum per 2048 counts, and a ticket) is a fixed __device__ array inside the library,
 *   64.25 KB on every GPU that loads it, held until the process exits.
 *   Limit: numLeaves <= CS_STATIC_PARTITION_MAX_LEAVES (2^24; BASELINE's largest tree has 14.2 M leaves); beyond it
 *   the call returns CS_ERR_CAPACITY and touches nothing.  numRanks: any (bounds holds numRanks + 1 uint32).
 *   counts, bounds: device pointers on the CURRENT device (there is no context to name one).  Enqueues a 8-byte memset
 *   node (the ticket must start at zero; the sums need no clearing, they are overwritten before they are read) and one
 *   kernel on `stream`; does not synchronise; capturable.
 *   All calls on a device share the scratch array: calls that overlap on the GPU (different streams, or host threads
 *   on streams that are not ordered with each other) race and give wrong bounds; the caller orders them.
 *   cs_partitionLeavesStaticSetup looks up the array's device address for the current device (cudaGetSymbolAddress,
 *   once per device; the entry point does the same on its first call there): call it before a capture begins.
 *   Errors: INVALID_ARG (null pointer, numLeaves or numRanks 0), CAPACITY (see above), CUDA.  cs_lastError(NULL) has
 *   the message. */
#define CS_STATIC_PARTITION_MAX_LEAVES (1u << 24)
cs_status cs_partitionLeavesStatic(const uint32_t* counts, uint32_t numLeaves, uint32_t numRanks, uint32_t* bounds,
                                   void* stream);
cs_status cs_partitionLeavesStaticSetup(void);
uint32_t  cs_partitionLeavesStaticMax(void);   /* CS_STATIC_PARTITION_MAX_LEAVES of the loaded library */

/* cs_nodeCountsFromLeaves -- particle ranges of the nodes of a linked octree from the counts of its leaves, without
 *   the particles (the upward pass of PAPER.md:258; for the replicated global octree the counts are the all-reduced
 *   ones): nodeCount[i] = sum of leafCounts over the leaves inside node i, nodeFirst[i] = sum over the leaves before
 *   it (sums modulo 2^32: N_tot < 2^32).  leaves / leafCounts: the cornerstone array and its counts; prefixes: NK from
 *   cs_linkOctree of the same leaves.  Does not synchronise. */
cs_status cs_nodeCountsFromLeaves(cs_context* ctx, const uint64_t* leaves, const uint32_t* leafCounts, uint32_t numLeaves,
                                  const uint64_t* prefixes, uint32_t numNodes, uint32_t* nodeFirst, uint32_t* nodeCount,
                                  void* stream);

/* ---- node properties on the linked octree (first row past the hot path: "additional octree
 *      node properties ... can be stored in separate arrays of length n"; readings A25-A27) --------
 * All arrays are device pointers owned by the caller; the calls enqueue on `stream` and return.  Three-component
 * outputs are structure-of-arrays: component d of node i at [d * numNodes + i].
 */

/* cs_gatherParticles -- the coordinates in SFC order: xs[j] = x[perm[j]] (perm as written by cs_sortKeys,
 *   PAPER.md:168).  Not in place.  n == 0 is a no-op. */
cs_status cs_gatherParticles(cs_context* ctx, const double* x, const double* y, const double* z, const uint32_t* perm,
                             uint64_t n, double* xs, double* ys, double* zs, void* stream);

/* cs_nodeGeometry -- the cell of every node in the bounding box: a node with placeholder-bit key NK of `level`
 *   octal digits is cell (ix, iy, iz) of the 2^level grid (digit = 4 xbit + 2 ybit + zbit);
 *   edge h_d = (hi_d - lo_d) / 2^level, centers[d] = lo_d + (i_d + 0.5) * h_d, halfSizes[d] = 0.5 * h_d, one
 *   binary64 rounding per operation.  box6: dev, as written by cs_computeBox. */
cs_status cs_nodeGeometry(cs_context* ctx, const uint64_t* prefixes, uint32_t numNodes, const double* box6,
                          double* centers, double* halfSizes, void* stream);

/* cs_nodeGeometryHilbert -- the same for a tree built on Hilbert keys (cs_computeKeysHilbert / cs_setCurve; DESIGN.md
 *   reading A28): the digits of NK are positions along the curve, and the cell is found by walking the curve backwards
 *   from the root (in orientation (e, d) the w-th sub-cube is the octant rotl(gc(w), d + 1) xor e).  Same arithmetic on
 *   the cell, same arguments. */
cs_status cs_nodeGeometryHilbert(cs_context* ctx, const uint64_t* prefixes, uint32_t numNodes, const double* box6,
                                 double* centers, double* halfSizes, void* stream);

/* cs_nodeMassCenters -- centres of mass (unit masses) by an upward pass over the links: a leaf's
 *   is the sum of its particles' sorted coordinates xs[first .. first + count) in that order over count, an
 *   internal node's the sum over its 8 children in order of count_c * com_c over its count, an empty node takes
 *   its geometric centre.  xs, ys, zs: coordinates in SFC order (cs_gatherParticles); nodeFirst / nodeCount /
 *   childOffsets / levelRange: as written by cs_linkOctree + cs_nodeCounts or cs_buildOctree; centers: from
 *   cs_nodeGeometry.  Two launches (the leaves of all levels; then the internal nodes level by level, deepest
 *   first, behind grid barriers); no host synchronisation. */
cs_status cs_nodeMassCenters(cs_context* ctx, const double* xs, const double* ys, const double* zs,
                             const uint32_t* nodeFirst, const uint32_t* nodeCount, const uint32_t* childOffsets,
                             const double* centers, const uint32_t* levelRange, uint32_t numNodes, double* com,
                             void* stream);

/* cs_macMinDistance -- the minimum-distance multipole acceptance criterion, Eq. 12: pass[i] = 1
 *   iff r_min > l / theta for source node i and the axis-aligned target box focus6 = {xmin, xmax, ymin, ymax, zmin,
 *   zmax} (HOST array; "with respect to any point in F").  r_min^2 = sum of squared per-dimension
 *   gaps max(|c - fc| - (h + fh), 0), l = 2 * max_d h_d, decided as r_min^2 * theta^2 > l^2 in binary64.
 *   Errors: INVALID_ARG (null pointer, theta <= 0). */
cs_status cs_macMinDistance(cs_context* ctx, const double* centers, const double* halfSizes, uint32_t numNodes,
                            const double* focus6, double theta, uint8_t* pass, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* CORNERSTONE_B200_H */
