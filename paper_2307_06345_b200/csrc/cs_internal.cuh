// Internal declarations shared by the translation units of libcornerstone_b200.so.
// sm_100a only.  Nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

#include "../../include/cornerstone.h"

namespace cs {

typedef unsigned long long u64;
typedef unsigned int u32;

constexpr int kL = 21;
constexpr u64 kKeyEnd = 1ull << 63;          // 8^L
constexpr int kMaxRounds = kL + 1;           // DESIGN.md A12
constexpr int kRoundSlots = kMaxRounds + 2;

// ---- radix sort geometry -------------------------------------------------------------
#ifndef CS_RADIX_BITS
#define CS_RADIX_BITS 9
#endif
constexpr int kRadixBits = CS_RADIX_BITS;
constexpr int kRadix = 1 << kRadixBits;
constexpr int kSortPasses = (63 + kRadixBits - 1) / kRadixBits;   // 63 key bits: 7 passes of 9 bits
// Sort plans (cs_sort.cu): the plain plan sorts by all digits; a plan with first digit F sorts by the digits F .. 6 and
// orders the bits below inside runs of equal leading digits in its last pass: the default plan (F = kSortTopFirst: bits
// 18..62, 5 passes), the short plan (F = 3: bits 27..62, 4 passes: fits while no cell of octree level 12 holds more than
// 257 particles) and the tiny plan (F = kSortMaxFirst = 4: bits 36..62, 3 passes: no such cell on level 9; what uniform
// particles allow up to billions of them).  A plan whose last pass finds a run too long is redone on the device and the
// context moves to the next plan for a while (the ladder of CS_SORT_AUTO).  Plans are numbered finest first.
enum { kPlanTiny = 0, kPlanShort = 1, kPlanDefault = 2, kPlanPlain = 3 };
constexpr int kSortTopFirst = 2;
constexpr int kSortShortFirst = 3;
constexpr int kSortMaxFirst = 4;
constexpr int kPlainHold = 16;        // sorts on the plain plan after the default plan needed the redo, before it is tried again
constexpr int kShortHold = 256;       // sorts before a plan that needed the redo is tried again (doubles with every failure)
constexpr int kShortHoldMax = 1 << 14;
inline int planFirstDigit(int plan) { return plan == kPlanPlain ? 0 : kSortMaxFirst - plan; }
inline int planPasses(int plan) { return kSortPasses - planFirstDigit(plan); }
#ifndef CS_SORT_BLOCK
#define CS_SORT_BLOCK 512
#endif
#ifndef CS_SORT_ITEMS
#define CS_SORT_ITEMS 13
#endif
#ifndef CS_SORT_MINBLOCKS
#define CS_SORT_MINBLOCKS 2
#endif
constexpr int kSortBlock = CS_SORT_BLOCK;
constexpr int kSortMinBlocks = CS_SORT_MINBLOCKS;   // resident CTAs per SM the radix pass is compiled for
constexpr int kSortItems = CS_SORT_ITEMS;
constexpr int kSortTile = kSortBlock * kSortItems;   // 6656 keys per tile
constexpr int kSortLastTile = kSortTile - 320;       // nominal tile of the pass that also orders the low bits (cs_sort.cu)

// ---- leaf refinement / link geometry -------------------------------------------------
constexpr int kLeafBlock = 256;
constexpr int kLeafItems = 8;
constexpr int kLeafTile = kLeafBlock * kLeafItems;   // 2048 leaves per tile

constexpr int kLinkBlock = 256;
constexpr int kLinkItems = 4;
constexpr int kLinkTile = kLinkBlock * kLinkItems;   // 1024 leaf boundaries per tile
constexpr int kLinkBins = 2 * (kL + 1);              // per level: all nodes, internal nodes

// one-pass leaf build (cs_leaves_direct.cu): particle boundaries per tile, largest bucketSize it takes
constexpr int kDirectTileLog2 = 11;
constexpr int kDirectMaxBucket = 1024;
#ifndef CS_DIR_COMPACT
#define CS_DIR_COMPACT 256
#endif
constexpr int kDirectCompact = CS_DIR_COMPACT;   // leaf starts per tile that the levels kernel hands over as a compact list

constexpr int kScanBlock = 256;
constexpr int kScanItems = 8;
constexpr int kScanTile = kScanBlock * kScanItems;

// Device-resident control block: every size the path produces stays here, so the whole
// build can be enqueued without a host round trip.
struct DeviceCtrl {
    u32 nl[kRoundSlots];         // leaf count entering round r (nl[r+1] = after round r)
    u32 ticket[kRoundSlots];     // tile tickets of round r
    u32 tilesDone[kRoundSlots];
    u32 changed[kRoundSlots];    // some O_i != 1 in round r
    u32 taskCount[kRoundSlots];  // split leaves of round r with a short particle range (counted linearly)
    u32 searchCount[kRoundSlots];// split leaves of round r with a long particle range (searched)
    u32 done;                    // refinement finished (converged / maxRounds / error)
    u32 rounds;                  // rounds performed
    u32 converged;
    u32 status;                  // cs_status of the device-side checks
    u32 numLeaves;               // final leaf count
    u32 numNodes;
    u32 linkTicket;
    u32 scanTicket;
    u32 levelTotals[kLinkBins];  // link: nodes per level (all / internal)
    u32 levelRange[kL + 2];
    u32 directBuild;             // the leaves in leafK[0] come from the one-pass build (cs_leaves_direct.cu)
    u32 pad[6];
};

struct HostCtrl {                // pinned mirror read back once per call
    DeviceCtrl c;
    u32 sortRedo;                // the sort's fix-up gave up and the plain passes ran (cs_sort.cu)
    u32 sortRedoHint;            // the same flag, copied behind every default-plan sort without a synchronisation
    u32 epochBase;               // replayed builds (CUDA graph): the look-back epoch before this replay, copied to the device by the graph's first node
};

// A whole cs_buildOctree call captured as a CUDA graph (small inputs are bound by launch overhead, not by the device):
// valid while every argument and mode it was captured with stays the same.
struct BuildGraphKey {   // `plain` holds the sort plan
    const void* x; const void* y; const void* z;
    u64 n;
    u32 bucket, prevNumLeaves, maxRounds;
    const void* prevLeaves;
    cs_octree_buffers buffers;
    int plain, curve, leafMode;
    cudaStream_t stream;
};
constexpr int kSortRedoSlot = 63;   // ctx->sortTickets[kSortRedoSlot]: that flag on the device

}  // namespace cs

struct cs_context {
    int device = 0;
    uint64_t maxParticles = 0;
    uint32_t maxLeaves = 0;
    uint32_t maxNodes = 0;
    int numSMs = 148;

    char* slab = nullptr;
    size_t slabBytes = 0;

    // sort
    cs::u64* keysAlt = nullptr;
    cs::u32* permAlt = nullptr;
    cs::u32* sortHist = nullptr;       // [kSortPasses][kRadix] + kSortPasses tickets
    cs::u32* sortTickets = nullptr;
    cs::u64* sortLookback = nullptr;   // [tiles][kRadix]
    cs::u32 epoch = 0;                 // look-back epoch, bumped per launch that uses a look-back array
    cs::u32* epochWords = nullptr;     // device: [0] = 0 for ever, [1] = epoch base of the replayed graph (kernels add *base to their epoch argument)
    bool capturing = false;            // a build is being captured: epochs are handed out relative to [1]
    cs::u32 captureEpochs = 0;         // epochs the captured build uses
    cudaStream_t captureStream = nullptr;
    cudaGraphExec_t buildGraph = nullptr;
    cs::BuildGraphKey buildGraphKey = {};
    cs::BuildGraphKey buildGraphCandidate = {};   // arguments of the previous call (a graph is captured when they repeat)
    bool buildGraphSeen = false;
    cs::u32 buildGraphEpochs = 0;      // epochs one replay consumes
    uint64_t buildGraphLaunches = 0;   // kernels one replay launches
    uint64_t graphMaxParticles = 1ull << 32;   // builds of at most this many particles are captured and replayed (all)
    int sortMode = CS_SORT_AUTO;       // cs_setSortMode
    int autoPlainLeft = 0;             // CS_SORT_AUTO: sorts left on the plain plan after the default plan needed the redo
    int planLeft[cs::kPlanDefault] = {0, 0};                             // CS_SORT_AUTO: sorts left before the tiny / short plan is tried again
    int planHold[cs::kPlanDefault] = {cs::kShortHold, cs::kShortHold};   // the next value of planLeft[] (back-off)
    int lastPlan = cs::kPlanDefault;   // plan of the last sort enqueued (whose redo flag may still arrive)
    cs::u32 redoGrid = 0;              // CTAs of onesweepRedoKernel that are resident together (cooperative launch)

    // keys
    unsigned short* hilbertTable = nullptr;   // [24][512] three-level transitions of the Hilbert curve (cs_particles.cu)
    unsigned char* hilbertInverse = nullptr;  // [24][8] one-level inverse transitions (node geometry, cs_props.cu)
    int curve = CS_CURVE_MORTON;              // cs_setCurve: the curve cs_buildOctree computes keys on

    // box
    double* boxPartials = nullptr;     // [grid][6]
    cs::u32* boxCounter = nullptr;

    // leaves
    cs::u64* leafK[2] = {nullptr, nullptr};
    cs::u32* leafOff[2] = {nullptr, nullptr};
    unsigned char* divLevel = nullptr; // one-pass build: d_j = level of the deepest internal node above particle j
    uint4* leafTasks = nullptr;        // (first child slot, particle range, shift of the child digit) per split leaf
    cs::u32 maxTasks = 0;
    cs::u32* leafOffFinal = nullptr;   // off[] of the returned leaves (prefix sum of counts), n_l + 1 entries
    cs::u64* tileLookback = nullptr;   // [tiles] look-back words of the leaf rounds and the scan
    cs::u32* leafOpk = nullptr;        // [leaf tiles][kLeafBlock] rounds: O of 8 leaves per word (decide -> scatter phase)
    uint4* leafTileInfo = nullptr;     // [leaf tiles] rounds: sum of O, split leaves per tile
    cs::u32 roundsGrid = 0;            // CTAs of leafRoundsKernel that are resident together (cooperative launch)
    unsigned char* dirFlags = nullptr; // one-pass leaf build: bit j set <=> position j owns entries of K
    cs::u32* dirTotals = nullptr;      // [tiles] K entries owned by the positions of a tile
    cs::u32* dirBases = nullptr;       // [tiles + 1] exclusive prefix of dirTotals
    cs::u32* dirListSize = nullptr;    // [tiles] leaf starts of the tile, or ~0u if they exceed kDirectCompact (then flags / levels serve)
    ulonglong2* dirListKeys = nullptr; // [tiles][kDirectCompact] the two keys around each leaf start
    cs::u32* dirListMeta = nullptr;    // [tiles][kDirectCompact] position | levels | entry count of each leaf start
    int leafMode = 0;                  // cs_setLeafMode
    cs::u32* linkTileHist = nullptr;   // [tiles][kLinkBins] node counts per tile, level and kind
    cs::DeviceCtrl* ctrl = nullptr;
    cs::HostCtrl* hostCtrl = nullptr;  // pinned

    // 64-bit staging of the L = 10 entry points (cs_api32.cu; allocated on first use)
    char* wideSlab = nullptr;
    cs::u64* wideLeaves = nullptr;     // [maxLeaves + 2]
    cs::u64* widePrev = nullptr;       // [maxLeaves + 2]
    cs::u64* widePrefixes = nullptr;   // [maxNodes + 2]

    // buffers for cs_buildOctreeHost (allocated lazily)
    char* hostPathSlab = nullptr;
    size_t hostPathBytes = 0;
    cudaStream_t copyStream = nullptr;   // the upload runs here, chunk by chunk, while the box of earlier chunks is reduced
    cudaEvent_t copyEvents[9] = {};
    bool boxReady = false;               // cs_buildOctreeHost: buffers->box6 is already filled, the build skips the box stage

    // profiling
    bool profiling = false;
    cudaEvent_t evBegin[CS_NUM_STAGES] = {};
    cudaEvent_t evEnd[CS_NUM_STAGES] = {};
    bool evUsed[CS_NUM_STAGES] = {};
    uint64_t launches = 0;

    std::string lastError;
};

namespace cs {

// ---- error plumbing --------------------------------------------------------------------
cs_status fail(cs_context* ctx, cs_status st, const char* fmt, ...);
cs_status cudaFail(cs_context* ctx, cudaError_t e, const char* what);
#define CS_CUDA(ctx, call)                                                     \
    do {                                                                       \
        cudaError_t e__ = (call);                                              \
        if (e__ != cudaSuccess) return ::cs::cudaFail((ctx), e__, #call);      \
    } while (0)
#define CS_TRY(expr)                                   \
    do {                                               \
        cs_status s__ = (expr);                        \
        if (s__ != CS_OK) return s__;                  \
    } while (0)
#define CS_LAUNCH_CHECK(ctx, name)                                             \
    do {                                                                       \
        (ctx)->launches++;                                                     \
        cudaError_t e__ = cudaGetLastError();                                  \
        if (e__ != cudaSuccess) return ::cs::cudaFail((ctx), e__, name);       \
    } while (0)

// Launch `kernel` so that it may be scheduled before the kernel in front of it on the stream has finished (programmatic
// dependent launch: the launch latency and the prologue of one kernel hide behind the tail of the one before; what a
// small build is made of).  ONLY for kernels whose first statement is chainEnter() (cs_device.cuh): that is where they
// wait for the data of their predecessors.  Works under stream capture (a programmatic edge of the graph); behind a
// memset, copy or event node, or a kernel without chainEnter(), it is an ordinary launch.
#ifndef CS_CHAIN
#define CS_CHAIN 1
#endif
template <typename... KArgs, typename... Args>
inline void launchChained(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, Args&&... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = CS_CHAIN ? 1 : 0;
    cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);     // errors: cudaGetLastError in CS_LAUNCH_CHECK
}

struct DeviceGuard {              // makes `dev` current for the scope and restores the caller's device
    int prev = -1;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(int dev)
    {
        cudaGetDevice(&prev);
        if (prev != dev) err = cudaSetDevice(dev);
        else prev = -1;
    }
    ~DeviceGuard()
    {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

struct StageTimer {               // records CUDA events around a stage when profiling is on
    cs_context* ctx; int stage; cudaStream_t s;
    StageTimer(cs_context* c, int st, cudaStream_t stream) : ctx(c), stage(st), s(stream)
    {
        if (ctx->profiling) { cudaEventRecord(ctx->evBegin[stage], s); }
    }
    ~StageTimer()
    {
        if (ctx->profiling) { cudaEventRecord(ctx->evEnd[stage], s); ctx->evUsed[stage] = true; }
    }
};

inline u32 divUp(u64 a, u64 b) { return (u32)((a + b - 1) / b); }
u32 nextEpoch(cs_context* ctx, cudaStream_t s);
inline const u32* epochBase(const cs_context* ctx) { return ctx->epochWords + (ctx->capturing ? 1 : 0); }
u32 reserveEpochs(cs_context* ctx, u32 count, cudaStream_t s);   // first of `count` consecutive look-back epochs

// ---- stage enqueue functions (no synchronisation; sizes device-resident) ---------------
cs_status enqueueBox(cs_context*, const double* x, const double* y, const double* z, u64 n, double* box6,
                     cudaStream_t);
cs_status enqueueBoxFold(cs_context*, const double* chunkBoxes, int chunks, double* box6, cudaStream_t);
// histFrom: also accumulate the digit histograms of the radix sort, digits histFrom..6, into ctx->sortHist (-1: none)
cs_status enqueueKeys(cs_context*, const double* x, const double* y, const double* z, u64 n, const double* box6,
                      u64* keys, int histFrom, int curve, cudaStream_t, u32* keys32 = nullptr /*30-bit keys instead*/);
void hilbertBuildTable(unsigned short* table /*[24 * 512], host*/);
void hilbertBuildInverse(unsigned char* inv /*[24 * 8], host*/);
cs_status sortInit(cs_context*);            // per-device kernel attributes, called by cs_create
cs_status leavesDirectInit(cs_context*);
cs_status leavesInit(cs_context*);
cs_status enqueueSortReset(cs_context*, cudaStream_t);
u64* sortSource(cs_context*, u64* keys, int plan);   // where the first radix pass reads the unsorted keys
cs_status enqueueSort32(cs_context*, u32* keys, u32* perm, u64 n, cudaStream_t);   // 30-bit keys: 4 plain passes
int sortDecidePlan(cs_context*);              // plan of the next sort (kPlanTiny .. kPlanPlain)
void sortPlanOutcome(cs_context*, int plan, bool redone);   // what the host learnt about a finished sort
int sortPeekPlainPasses(const cs_context*);   // plain passes of the next sort (cs_sortPasses)
cs_status enqueueSort(cs_context*, u64* keys, u32* perm, u64 n, bool fused, int plan, cudaStream_t);
// maxLevel: depth below which no leaf is split: kL, or 10 for 30-bit keys held in the top 10 digits (cs_api32.cu)
cs_status enqueueLeaves(cs_context*, const u64* sortedKeys, u64 n, u32 bucketSize, const u64* prevLeaves,
                        u32 prevNumLeaves, u32 maxRounds, u64* leaves, u32* counts, u32 leafCapacity, u32 maxLevel,
                        cudaStream_t);
bool leavesDirectSupported(const cs_context*, u32 bucketSize);
cs_status enqueueLeavesDirect(cs_context*, const u64* sortedKeys, u64 n, u32 bucketSize, u32 cap, u32 maxLevel, cudaStream_t);
// leaves/numLeaves: if dNumLeaves is null the host value is used
cs_status enqueueLink(cs_context*, const u64* leaves, const u32* dNumLeaves, u32 hNumLeaves, u32 leafBound,
                      u64* prefixes, u32* levels, u32* childOffsets, u32* parents, u32* levelRange,
                      u32* leafToNode, u32* nodeToLeaf, u32 nodeCapacity, const u32* leafOffsets /*nullable*/,
                      u32* nodeFirst, u32* nodeCount, cudaStream_t);
cs_status enqueueNodeCounts(cs_context*, const u64* sortedKeys, u64 n, const u64* prefixes, const u32* dNumNodes,
                            u32 hNumNodes, u32 nodeBound, const u32* leafOffsets, const u32* nodeToLeaf,
                            u32* nodeFirst, u32* nodeCount, cudaStream_t);
// device-wide exclusive scan of u32 (decoupled look-back): out[i] = sum_{j<i} in[j], out[n] = total
cs_status enqueueExclusiveScan(cs_context*, const u32* in, u32* out, u32 n, cudaStream_t);
cs_status enqueueReadCtrl(cs_context*, cudaStream_t);   // D2H of the control block
cs_status readCtrl(cs_context*, cudaStream_t);   // D2H of the control block + stream sync
// the distributed build (cs_global.cu): f alone, g alone, SFC partition, node counts from leaf counts
cs_status enqueueCountLeaves(cs_context*, const u64* sortedKeys, u64 n, const u64* leaves, u32 numLeaves, u32* counts,
                             cudaStream_t);
cs_status enqueueRebalance(cs_context*, const u64* leaves, const u32* counts, u32 numLeaves, u32 bucketSize, u32 maxLevel,
                           u64* newLeaves, u32 cap, cudaStream_t);
cs_status enqueuePartition(cs_context*, const u32* counts, u32 numLeaves, u32 numRanks, u32* bounds, cudaStream_t);
cs_status enqueueNodeCountsFromLeaves(cs_context*, const u64* leaves, const u32* counts, u32 numLeaves, const u64* prefixes,
                                      u32 numNodes, u32* nodeFirst, u32* nodeCount, cudaStream_t);
// node properties on the linked tree (cs_props.cu)
cs_status enqueueGather(cs_context*, const double* x, const double* y, const double* z, const u32* perm, u64 n,
                        double* xs, double* ys, double* zs, cudaStream_t);
cs_status enqueueNodeGeometry(cs_context*, const u64* prefixes, u32 n, const double* box6, int curve, double* centers,
                              double* halfSizes, cudaStream_t);
cs_status enqueueMassCenters(cs_context*, const double* xs, const double* ys, const double* zs, const u32* nodeFirst,
                             const u32* nodeCount, const u32* childOffsets, const double* centers, const u32* levelRange,
                             u32 n, double* com, cudaStream_t);
cs_status enqueueMac(cs_context*, const double* centers, const double* halfSizes, u32 n, const double* focus6,
                     double theta, unsigned char* pass, cudaStream_t);

}  // namespace cs
