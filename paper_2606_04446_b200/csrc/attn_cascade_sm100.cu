// Stage (c), fused: cascade tree-verify attention in ONE launch on tcgen05 / TMEM / TMA (sm_100a).
// PAPER.md:52, :124, :154.
//
// Every tree query of every branch and every GQA head of one kv head is a row of one batched query
// matrix (row r = t*G + hh), cut into 128-row M tiles.  The keys of a request are the committed
// prefix followed by the tree-local keys, cut into 128-key tiles: prefix tiles 0..np-1
// (np = ceil(L/128)) and tree tiles np..np+nt-1 (nt = ceil(T/128)); the tree tiles are ordinary key
// tiles whose scores additionally pass the node's ancestor-mask bits.
//
// Work decomposition.  A query tile is either half of a "pair item" (tiles 2p, 2p+1) or a "split item"
// of its own; the launch plan decides (api.cu: up to three query tiles in the one-wave regime are all
// split items).  The key-tile sequence of the request is cut into chunks; one CTA serves (request b, kv
// head g, item, chunk) and owns two accumulator SLOTS that strictly alternate in the unit stream
// (one unit = one M tile x one 128-key tile):
//
//   pair item   : slot s = M tile 2p+s; every key tile of the chunk feeds both slots (the KV tile crosses
//                 the L2->SM crossbar once per 256 query rows; two partial states leave the CTA)
//   split item  : both slots hold the same M tile; slot s takes the chunk's key tiles of parity s
//                 (two running softmax states over disjoint keys, merged in registers in the epilogue:
//                 one partial state of 128 rows leaves the CTA)
//
// so that the tensor phase of one slot (P.V, then the next Q.K^T, which cannot start earlier because P
// overwrites S in TMEM) runs under the other slot's softmax.  The eight softmax warps serve one unit
// at a time, two threads per query row.
// Per unit:
//
//   S[128 x 128] = Q_m[128 x 128] . K_j^T    tcgen05.mma, A/B from 128B-swizzled SMEM (TMA), D in TMEM
//   P            = exp2(c*(S - m_run))       softmax thread per row (TMEM lane), P -> TMEM over S
//   O_m[128x128] += P[128 x 128] . V_j       tcgen05.mma, A = P from TMEM, B = V (MN-major SMEM)
//
// TMEM (512 columns): O_0, O_1 (128 fp32 columns each), S_0/P_0, S_1/P_1 (128 each).
// Warp roles (384 threads): warps 0..7 = softmax (warps 0..3 key columns 0..63, warps 4..7 columns
// 64..127 of every S tile), warp 8 = TMA producer, warps 9 / 10 = MMA issuers of slot 0 / 1 (one
// thread each; warp 10 also owns the TMEM allocation), warp 11 = zeroes the V rows behind a
// ragged tile end (they are multiplied by exact zeros and may hold anything, NaN included).  The
// control warpgroup gives registers to the softmax warpgroups (setmaxnreg).  The running max is only
// raised when a tile maximum exceeds it by more than 2^8 (lazy rescale), in which case the owning
// thread rescales its O row in TMEM before the next P.V.
//
// Cascade merge in the same launch (log-sum-exp state merge): every CTA writes its
// partial state(s) (normalised O fp32, LSE) to the workspace (bulk copies from a shared-memory
// staging image; it stays in L2), publishes it with a release-increment of its group's arrival
// counter (group = request, kv head, item), waits until all non-empty chunks of the group have
// arrived, and then merges ITS share of the group's rows and writes the bf16 output and the LSE.
// The counters reset themselves (last CTA out), so the workspace header only has to be zero before
// the first call (d2sd_cascade_workspace_init).  The wait is safe because a group is a run of
// consecutive blocks of the grid's linear order: the oldest unfinished group always has all its
// CTAs resident or done; the spin is bounded and traps instead of hanging.
// The launch is a programmatic dependent launch: the prologue (barriers, TMEM, tensor-map prefetch)
// overlaps the tail of the preceding kernel; no global memory is touched before griddepcontrol.wait.
#include <cuda.h>

#include "common.cuh"

namespace d2sd {
namespace {

constexpr int kD = 128;
constexpr int kTileM = 128;
constexpr int kTileN = 128;
constexpr int kRing = 5;        // ring of K / V tiles (K_j, V_j, K_j+1, ...)
constexpr int kThreads = 384;
constexpr uint32_t kQTileBytes = kTileM * kD * 2;   // 32 KiB: [d_hi 2][128 rows][128 B]
constexpr uint32_t kKvTileBytes = kTileN * kD * 2;  // 32 KiB: [d_hi 2][128 keys][128 B]
constexpr uint32_t kOffQ = 0;
constexpr uint32_t kOffRing = 2 * kQTileBytes;
constexpr uint32_t kOffBar = kOffRing + kRing * kKvTileBytes;
constexpr uint32_t kOffX = kOffBar + 256;                 // softmax exchange: fp32 [2][2][128]
constexpr uint32_t kSmemUsed = kOffX + 2 * 2 * kTileM * 4;
constexpr uint32_t kSmemBytes = 232448;                   // the whole 227 KiB: kSmemUsed + alignment slack
constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kTmemS = 256;  // S/P buffers of the two slots behind the two O accumulators
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kRescaleThreshold = 8.0f;  // log2 units
constexpr uint32_t kRegsControl = 80, kRegsSoftmax = 208;  // setmaxnreg targets

// barrier slots (8 bytes each) at kOffBar.  S-ready / P-ready exist PER SLOT (phase = unit
// count of that slot) and are only ever waited on by that slot's team and the MMA thread.
enum : uint32_t {
    kBarQFull = 0,                     // [2]
    kBarFull = 2,                      // [kRing]
    kBarEmpty = kBarFull + kRing,      // [kRing]
    kBarSFull = kBarEmpty + kRing,     // [2]
    kBarPFull = kBarSFull + 2,         // [2][4]: P is released to the tensor pipe in four 32-key pieces
    kBarAllDone = kBarPFull + 8,       // every MMA of the CTA has completed
    kBarVFix = kBarAllDone + 1,        // [2] warp 11 has zeroed the V rows behind a ragged tile end; a CTA
                                       // meets at most two ragged tiles (last prefix tile, last tree tile)
    kBarMerge = kBarVFix + 2,          // the group's partial O rows of this CTA's share have landed in shared memory
    kNumBars = kBarMerge + 1,
    kTmemSlot = kNumBars  // uint32 written by tcgen05.alloc
};
static_assert((kNumBars + 1) * 8 <= 256, "barrier area");
static_assert(kSmemUsed + 512 <= kSmemBytes, "shared memory budget");

// ---- PTX wrappers -------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
// Bounded wait: a protocol bug traps (reported as a launch failure) instead of hanging the GPU.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t spins = 0;
    while (!mbar_try_wait(bar, parity)) {
        if (++spins > (1u << 26)) __trap();
    }
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int c0, int c1, int c2,
                                            int c3, uint64_t hint) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
        " [%0], [%1, {%3, %4, %5, %6}], [%2], %7;" ::"r"(dst),
        "l"(reinterpret_cast<uint64_t>(tm)), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "l"(hint)
        : "memory");
}
__device__ __forceinline__ void tma_load_5d(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int c0, int c1, int c2,
                                            int c3, int c4, uint64_t hint) {
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
        " [%0], [%1, {%3, %4, %5, %6, %7}], [%2], %8;" ::"r"(dst),
        "l"(reinterpret_cast<uint64_t>(tm)), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "l"(hint)
        : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* tm) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(tm)) : "memory");
}
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void named_bar_arrive(uint32_t id, uint32_t threads) {
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(threads) : "memory");
}
__device__ __forceinline__ void named_bar_sync(uint32_t id, uint32_t threads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}
constexpr uint64_t kEvictNormal = 0x1000000000000000ull;  // KV: read by the 2-3 sibling CTAs of the kv head within a few
                                                          // microseconds (evict-first measured 3% slower on configs 3, 4)
constexpr uint64_t kEvictLast = 0x14F0000000000000ull;   // re-read by every chunk CTA of the head: Q

// D[tmem] (+)= A[smem] . B[smem]
__device__ __forceinline__ void umma_ss(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc,
                                        uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// D[tmem] (+)= A[tmem] . B[smem]
__device__ __forceinline__ void umma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc,
                                        uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem),
        "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}

// Shared-memory matrix descriptor, 128B swizzle, descriptor version 1 (Blackwell).
//   K-major  operand: rows of 128 B (64 bf16 along K); 8-row groups SBO = 1024 B apart; LBO unused (1).
//   MN-major operand: rows of 128 B (64 bf16 along MN); the next 64 along MN is LBO bytes away, the next
//                     8 along K is SBO = 1024 B away.
// The start-address field holds (addr >> 4); advancing an operand by `bytes` adds (bytes >> 4).
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    return (uint64_t)((addr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) |
           ((uint64_t)(sbo_bytes >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// Instruction descriptor, kind::f16: fp32 accumulate, bf16 x bf16.
__host__ __device__ constexpr uint32_t idesc(uint32_t M, uint32_t N, uint32_t b_mn_major) {
    return (1u << 4) | (1u << 7) | (1u << 10) | (b_mn_major << 16) | ((N >> 3) << 17) | ((M >> 4) << 24);
}
constexpr uint32_t kIdescPV = idesc(kTileM, kD, 1);

#define D2SD_R32(r, o)                                                                                     \
    "=r"(r[o + 0]), "=r"(r[o + 1]), "=r"(r[o + 2]), "=r"(r[o + 3]), "=r"(r[o + 4]), "=r"(r[o + 5]),         \
        "=r"(r[o + 6]), "=r"(r[o + 7]), "=r"(r[o + 8]), "=r"(r[o + 9]), "=r"(r[o + 10]), "=r"(r[o + 11]),   \
        "=r"(r[o + 12]), "=r"(r[o + 13]), "=r"(r[o + 14]), "=r"(r[o + 15]), "=r"(r[o + 16]), "=r"(r[o + 17]), \
        "=r"(r[o + 18]), "=r"(r[o + 19]), "=r"(r[o + 20]), "=r"(r[o + 21]), "=r"(r[o + 22]), "=r"(r[o + 23]), \
        "=r"(r[o + 24]), "=r"(r[o + 25]), "=r"(r[o + 26]), "=r"(r[o + 27]), "=r"(r[o + 28]), "=r"(r[o + 29]), \
        "=r"(r[o + 30]), "=r"(r[o + 31])
#define D2SD_W32(r, o)                                                                                     \
    "r"(r[o + 0]), "r"(r[o + 1]), "r"(r[o + 2]), "r"(r[o + 3]), "r"(r[o + 4]), "r"(r[o + 5]), "r"(r[o + 6]),   \
        "r"(r[o + 7]), "r"(r[o + 8]), "r"(r[o + 9]), "r"(r[o + 10]), "r"(r[o + 11]), "r"(r[o + 12]),         \
        "r"(r[o + 13]), "r"(r[o + 14]), "r"(r[o + 15]), "r"(r[o + 16]), "r"(r[o + 17]), "r"(r[o + 18]),      \
        "r"(r[o + 19]), "r"(r[o + 20]), "r"(r[o + 21]), "r"(r[o + 22]), "r"(r[o + 23]), "r"(r[o + 24]),      \
        "r"(r[o + 25]), "r"(r[o + 26]), "r"(r[o + 27]), "r"(r[o + 28]), "r"(r[o + 29]), "r"(r[o + 30]),      \
        "r"(r[o + 31])
#define D2SD_TMEM_LD32(taddr, r, o)                                                                         \
    asm volatile(                                                                                           \
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"    \
        "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"                          \
        : D2SD_R32(r, o)                                                                                    \
        : "r"(taddr))
#define D2SD_TMEM_ST32(taddr, r, o)                                                                         \
    asm volatile(                                                                                           \
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15," \
        "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};" ::"r"(taddr),               \
        D2SD_W32(r, o)                                                                                      \
        : "memory")
#define D2SD_TMEM_ST16(taddr, r)                                                                            \
    asm volatile(                                                                                           \
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15," \
        "%16};" ::"r"(taddr),                                                                               \
        "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]),   \
        "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])                    \
        : "memory")
// Scheduling fence for 32 registers: the values are "rewritten" here, \
        so everything computed from them
// stays behind the preceding asm volatile statements (the compiler would otherwise hoist all 128
// exponentials above the first piece-wise release of P).
#define D2SD_PIN32(r, \
        o) asm volatile("" : \
        "+r"(r[o + 0]), \
        "+r"(r[o + 1]), \
        "+r"(r[o + 2]), \
        "+r"(r[o + 3]), \
        "+r"(r[o + 4]), \
        "+r"(r[o + 5]), \
        "+r"(r[o + 6]), \
        "+r"(r[o + 7]), \
        "+r"(r[o + 8]), \
        "+r"(r[o + 9]), \
        "+r"(r[o + 10]), \
        "+r"(r[o + 11]), \
        "+r"(r[o + 12]), \
        "+r"(r[o + 13]), \
        "+r"(r[o + 14]), \
        "+r"(r[o + 15]), \
        "+r"(r[o + 16]), \
        "+r"(r[o + 17]), \
        "+r"(r[o + 18]), \
        "+r"(r[o + 19]), \
        "+r"(r[o + 20]), \
        "+r"(r[o + 21]), \
        "+r"(r[o + 22]), \
        "+r"(r[o + 23]), \
        "+r"(r[o + 24]), \
        "+r"(r[o + 25]), \
        "+r"(r[o + 26]), \
        "+r"(r[o + 27]), \
        "+r"(r[o + 28]), \
        "+r"(r[o + 29]), \
        "+r"(r[o + 30]), \
        "+r"(r[o + 31]))
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

__device__ __forceinline__ float ex2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// Same, but ordered against the other volatile statements (TMEM stores / waits, barrier arrivals): the
// softmax loop uses it to keep a piece's exponentials ahead of the wait for the previous piece's store.
__device__ __forceinline__ float ex2_ordered(float x) {
    float y;
    asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ uint32_t pack2_bf16(float lo, float hi) {
    __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&v);
}

// One lane of a fully active warp; unlike `lane == 0` it lets ptxas keep the MMA operands on the uniform
// datapath (no per-instruction elect loop around every tcgen05.mma).
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
// shared -> global bulk copy (bytes % 16 == 0), one bulk group per call site
__device__ __forceinline__ void bulk_store(void* gdst, uint32_t ssrc, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(ssrc), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }


// What one CTA does: which item / chunk, which rows its two slots hold, which key tiles it streams.
enum : int { kModePair = 0, kModeSplit = 2 };
struct Work {
    int b, g, item, chunk;
    int mode;          // pair: both slots on every key tile; split: one query tile, slot = key-tile parity
    int lay_pair;      // partial-state layout of the group: 1 = pair item (256 rows per chunk), 0 = 128 rows
    int row_base;      // first query row (t*G + hh) of the item
    int rows0, rows1;  // valid query rows of slot 0 / 1 (0 = slot unused)
    int np, nt;        // prefix / tree key tiles of the request (after the mode bits)
    int j_begin, n_tiles;
    int n_chunks;      // non-empty chunks of the group = CTAs that arrive at the group counter
    int group;         // (b*Hkv + g)*n_items + item
    int T, L, rows_valid;
    int rows_item;     // valid query rows of the whole item (<= 256 for a pair item)
    __device__ __forceinline__ int rows(int s) const { return s ? rows1 : rows0; }
    // slot's first row relative to row_base (0 / 128 for a pair, 0 / 0 for a split)
    __device__ __forceinline__ int row_off(int s) const { return mode == kModeSplit ? 0 : s * kTileM; }
    __device__ __forceinline__ uint32_t uses(int jj) const {  // slots fed by the chunk's jj-th key tile
        return mode == kModePair ? 3u : (1u << (jj & 1));
    }
    // partial-state row of (slot s, row rl of the slot's tile) inside the group's partial block
    __device__ __forceinline__ int part_row0(int s) const {
        return lay_pair ? chunk * 2 * kTileM + s * kTileM : chunk * kTileM;
    }
};

struct TileInfo {
    int valid;      // keys of the tile that exist (1..128)
    int row;        // first row of the tile in its tensor map
    bool tree;      // tree tile (ancestor mask applies), else prefix tile
    int tt;         // tree tile index (tree tiles only)
    int j;          // key tile index within the request (prefix tiles first)
};

// -------------------------------------------------------------------------------------------------
// Cascade merge of one group's rows (log-sum-exp state merge):
//   LSE = log sum_p e^{LSE_p};  O = sum_p e^{LSE_p - LSE} O_p   over the partial states that hold the row.
// CTA `ci` of the group's `nc` CTAs takes a contiguous range of the item's rows.  A pair item has one
// state per chunk and query tile (at partial rows c*256 + row), a split item one per chunk (at c*128 + row).
// One bulk copy per state brings the range's O rows (512 B each, stored with their 16-byte chunks
// XOR-swizzled by the row, undone here) into shared memory -- all copies in flight at once, one L2
// round trip -- while the LSEs are staged with plain loads.  Warp w then
// merges rows w, w+8, ... of the range.  The partial states were written by other SMs through the
// async proxy and published with a release; they are read at L2 (bulk copy / ld.global.cg).
__device__ __forceinline__ void merge_rows(const AttnPlan& pl, const AttnArgs& a, float* dbg_rows, const Work& wk,
                                           uint32_t smem_stage, unsigned char* stage_gen, uint32_t bar_merge,
                                           int warp, int lane) {
    const int G = pl.G;
    const bool split = !wk.lay_pair;
    const int rows_item = wk.rows_item;
    const int n_rel = wk.n_chunks;  // <= 64 states
    const size_t grp0 = (size_t)wk.group * pl.grp_rows;
    const int stride = split ? kTileM : 2 * kTileM;
    const int r0 = rows_item * wk.chunk / wk.n_chunks, r1 = rows_item * (wk.chunk + 1) / wk.n_chunks;
    const int nrows = r1 - r0;  // nrows * n_rel <= 320 rows of 512 B: fits the freed Q + ring area
    if (nrows <= 0) return;
    if (warp == 0) {
        if (lane == 0) mbar_expect_tx(bar_merge, (uint32_t)(n_rel * nrows) * 512u);
        __syncwarp();
        for (int i = lane; i < n_rel; i += 32)
            asm volatile(
                "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                    smem_stage + (uint32_t)(i * nrows) * 512u),
                "l"(a.part_o + (grp0 + (size_t)i * stride + r0) * kD), "r"((uint32_t)nrows * 512u), "r"(bar_merge)
                : "memory");
    }
    // the LSEs of the range's rows, all states, into shared memory behind the O block (one round trip)
    float* lse_sm = reinterpret_cast<float*>(stage_gen + 320u * 512u);
    const int tid = warp * 32 + lane;
    for (int e = tid; e < n_rel * nrows; e += 256) {
        const int i = e / nrows, r = e - i * nrows;
        const float v = __ldcg(a.part_lse + grp0 + (size_t)i * stride + r0 + r);
        lse_sm[e] = v;
    }
    named_bar_sync(1, 256);
    auto out_row = [&](int r) {  // index of query row r0 + r of the item in out / lse: [b][t][h]
        const int ra = wk.row_base + r0 + r, t = ra / G;
        return ((size_t)wk.b * pl.T_cap + t) * pl.Hq + wk.g * G + (ra - t * G);
    };
    // step 1, one thread per row: LSE = m + log sum_p e^{LSE_p - m}; the LSEs in shared memory are
    // replaced by the normalised weights e^{LSE_p - LSE} (a state without any key: weight 0)
    if (tid < nrows) {
        float* col0 = lse_sm + tid;
        float m = -INFINITY;
#pragma unroll 4
        for (int i = 0; i < n_rel; ++i) m = fmaxf(m, col0[i * nrows]);
        float wsum = 0.f;
#pragma unroll 4
        for (int i = 0; i < n_rel; ++i) {
            const float v = col0[i * nrows];
            const float wv = v == -INFINITY ? 0.f : __expf(v - m);
            wsum += wv;
            col0[i * nrows] = wv;
        }
        const float inv = wsum > 0.f ? 1.f / wsum : 0.f;  // no key at all (L = 0, prefix-only mode): O = 0, LSE = -inf
#pragma unroll 4
        for (int i = 0; i < n_rel; ++i) col0[i * nrows] *= inv;
        const float lse = wsum > 0.f ? m + logf(wsum) : -INFINITY;
        const size_t orow = out_row(tid);
        if (dbg_rows) dbg_rows[orow * (kD + 1) + kD] = lse;
        else if (a.lse) a.lse[orow] = lse;
    }
    named_bar_sync(1, 256);
    mbar_wait(bar_merge, 0);  // the O rows have landed
    // step 2, one thread per (row, 16-byte chunk): O = sum_p weight_p O_p.  States without any key hold
    // zeros (their CTA wrote them), so no value needs guarding.
#pragma unroll 1
    for (int item = tid; item < nrows * 32; item += 256) {
        const int r = item >> 5;  // == warp-uniform row; chunk position == lane
        const float4* o_ptr = reinterpret_cast<const float4*>(stage_gen + (size_t)r * 512u) + lane;
        const float* w_ptr = lse_sm + r;
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 4
        for (int i = 0; i < n_rel; ++i) {
            const float wv = w_ptr[i * nrows];
            const float4 o = o_ptr[(size_t)(i * nrows) * 32];
            acc.x += wv * o.x; acc.y += wv * o.y; acc.z += wv * o.z; acc.w += wv * o.w;
        }
        const size_t orow = out_row(r);
        const int col = 4 * (lane ^ ((r0 + r) & 7));  // undo the staging swizzle: this lane holds columns col..col+3
        if (dbg_rows) {  // fp32 state for tests
            float* d0 = dbg_rows + orow * (kD + 1);
            d0[col + 0] = acc.x; d0[col + 1] = acc.y; d0[col + 2] = acc.z; d0[col + 3] = acc.w;
            continue;
        }
        __nv_bfloat162 lo = __floats2bfloat162_rn(acc.x, acc.y);
        __nv_bfloat162 hi = __floats2bfloat162_rn(acc.z, acc.w);
        uint2 pk;
        pk.x = *reinterpret_cast<uint32_t*>(&lo);
        pk.y = *reinterpret_cast<uint32_t*>(&hi);
        *reinterpret_cast<uint2*>(a.out + orow * kD + col) = pk;
    }
}

// mode bits: 1 = include the prefix tiles, 2 = include the tree tiles (3 = the whole cascade).
__global__ void __launch_bounds__(kThreads, 1)
attn_cascade_tc_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
                       const __grid_constant__ CUtensorMap tm_v, const __grid_constant__ CUtensorMap tm_tk,
                       const __grid_constant__ CUtensorMap tm_tv, AttnPlan pl, AttnArgs a, int mode,
                       float* dbg_rows) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    const uint32_t smem_raw_u32 = (uint32_t)__cvta_generic_to_shared(smem_raw);
    const uint32_t smem = (smem_raw_u32 + 1023u) & ~1023u;  // 128B swizzle atoms need 1024 B alignment
    if (smem - smem_raw_u32 + kSmemUsed > kSmemBytes) __trap();
    unsigned char* smem_gen = smem_raw + (smem - smem_raw_u32);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t bar0 = smem + kOffBar;
    auto bar = [&](uint32_t i) { return bar0 + 8u * i; };
    volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem_gen + kOffBar + 8u * kTmemSlot);

    // ---- prologue that touches no global memory (overlaps the preceding kernel's tail under PDL) ----
    if (warp == 8 && lane == 0) {
        mbar_init(bar(kBarQFull + 0), 1);
        mbar_init(bar(kBarQFull + 1), 1);
        for (int i = 0; i < kRing; ++i) {
            mbar_init(bar(kBarFull + i), 1);
            mbar_init(bar(kBarEmpty + i), 3);  // the two MMA issuers' commits + the V sanitiser
        }
        for (int s = 0; s < 2; ++s) {
            mbar_init(bar(kBarSFull + s), 1);
            for (int q = 0; q < 4; ++q) mbar_init(bar(kBarPFull + 4 * s + q), kTileM);
        }
        mbar_init(bar(kBarAllDone), 2);
        mbar_init(bar(kBarVFix + 0), 1);
        mbar_init(bar(kBarVFix + 1), 1);
        mbar_init(bar(kBarMerge), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        tma_prefetch_desc(&tm_q);
        tma_prefetch_desc(&tm_k);
        tma_prefetch_desc(&tm_v);
        tma_prefetch_desc(&tm_tk);
        tma_prefetch_desc(&tm_tv);
    }
    if (warp == 10) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(bar(kTmemSlot)),
                     "r"(kTmemCols)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    pdl_launch_dependents();  // the next kernel may begin its own prologue as SMs free up
    pdl_wait();               // everything before this kernel in the stream is complete and visible

    // ---- this CTA's work ----
    Work wk;
    {
        const int G = pl.G;
        wk.g = blockIdx.y;
        wk.b = blockIdx.z;
        int x = blockIdx.x, n_static;
        if (x < pl.n_pair * pl.chunks_a) {
            wk.item = x / pl.chunks_a; wk.chunk = x - wk.item * pl.chunks_a; n_static = pl.chunks_a;
            wk.mode = kModePair;
        } else {
            x -= pl.n_pair * pl.chunks_a;
            wk.item = pl.n_pair + x / pl.chunks_b; wk.chunk = x % pl.chunks_b; n_static = pl.chunks_b;
            wk.mode = kModeSplit;
        }
        wk.T = a.tree_len[wk.b];
        wk.L = a.ctx_len[wk.b];
        wk.rows_valid = wk.T * G;
        wk.row_base = wk.item < pl.n_pair ? wk.item * 2 * kTileM
                                          : (pl.n_pair * 2 + (wk.item - pl.n_pair)) * kTileM;
        wk.group = (wk.b * pl.Hkv + wk.g) * (pl.n_pair + pl.n_single) + wk.item;
        const int left = wk.rows_valid - wk.row_base;
        wk.rows0 = max(0, min(kTileM, left));
        if (wk.mode == kModePair) {
            wk.rows1 = max(0, min(kTileM, left - kTileM));
            // a pair item whose second query tile is empty (short tree): run the one tile as a split item
            // (both slots, key-tile parity), keep the pair item's partial-state layout
            if (wk.rows1 == 0) wk.mode = kModeSplit;
        }
        wk.lay_pair = wk.item < pl.n_pair;
        wk.rows_item = max(0, min(wk.lay_pair ? 2 * kTileM : kTileM, left));
        if (wk.mode == kModeSplit) wk.rows1 = wk.rows0;
        wk.np = (mode & 1) ? (wk.L + kTileN - 1) / kTileN : 0;
        wk.nt = (mode & 2) ? (wk.T + kTileN - 1) / kTileN : 0;
        const int nk = wk.np + wk.nt;
        const int tps = max(max(1, pl.tps_min), (nk + n_static - 1) / n_static);
        wk.n_chunks = max(1, (nk + tps - 1) / tps);  // chunk 0 always takes part (nk = 0: state (0, -inf))
        wk.j_begin = wk.chunk * tps;
        wk.n_tiles = max(0, min(nk, wk.j_begin + tps) - wk.j_begin);
    }
    // whole items past the tree's rows, and chunks past the request's key tiles, leave at once:
    // nobody waits for them (n_chunks counts the non-empty chunks only)
    const bool idle = wk.rows0 == 0 || wk.chunk >= wk.n_chunks;
    const int kv_row0 = a.kv_indptr ? a.kv_indptr[wk.b] : 0;
    auto tile_info = [&](int jj) {
        const int j = wk.j_begin + jj;
        TileInfo ti;
        ti.j = j;
        ti.tree = j >= wk.np;
        ti.tt = j - wk.np;
        ti.valid = ti.tree ? min(kTileN, wk.T - ti.tt * kTileN) : min(kTileN, wk.L - j * kTileN);
        ti.row = ti.tree ? wk.b * pl.T_cap + ti.tt * kTileN : kv_row0 + j * kTileN;  // (contiguous KV)
        return ti;
    };

    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    // the control warpgroup hands registers to the two softmax warpgroups (one instruction per warpgroup)
    if (warp >= 8) {
      asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsControl));
      if (idle) {
        // fall through to the TMEM release
      } else if (warp == 8) {
        // ===== TMA producer: K_0 first (the first MMA needs it), then the Q tiles, then the ring.
        // Contiguous KV: lane 0 issues one 32 KiB box per tile.  Paged KV (page = 16 keys): a 128-key
        // tile is 8 pages; lane 2p+hi issues the 2 KiB box (page p, d half hi) of the tile, so a tile is
        // 16 loads in flight at once.  Only the ceil(valid/16) pages that exist are loaded: the MMAs
        // never read past ceil16(valid) keys.  The page ids of the next tile are fetched one tile ahead. =====
        const bool paged = pl.page_size > 0;
        int x = 0;  // ring position of the next tile to load
        auto page_of = [&](int jj) {
            int pg = 0;
            if (paged && jj < wk.n_tiles) {
                const TileInfo t2 = tile_info(jj);
                const int p = lane >> 1;
                if (!t2.tree && lane < 16 && p * 16 < t2.valid) pg = __ldg(a.kv_indices + kv_row0 + t2.j * 8 + p);
            }
            return pg;
        };
        int page_cur = page_of(0);
        for (int jj = 0; jj < wk.n_tiles; ++jj) {
            const TileInfo ti = tile_info(jj);
            const int page_next = page_of(jj + 1);
            for (int kv = 0; kv < 2; ++kv, ++x) {
                const int i = x % kRing;
                const uint32_t dst = smem + kOffRing + i * kKvTileBytes;
                if (paged && !ti.tree) {
                    const int n_pages = (ti.valid + 15) >> 4;
                    if (lane == 0) {
                        mbar_wait(bar(kBarEmpty + i), ((x / kRing) & 1) ^ 1);
                        mbar_expect_tx(bar(kBarFull + i), (uint32_t)n_pages * 4096u);
                    }
                    __syncwarp();
                    if (lane < 2 * n_pages)
                        tma_load_5d(dst + (uint32_t)(lane & 1) * (kKvTileBytes / 2) + (uint32_t)(lane >> 1) * 2048u,
                                    kv ? &tm_v : &tm_k, bar(kBarFull + i), 0, 0, lane & 1, wk.g, page_cur, kEvictNormal);
                } else if (lane == 0) {
                    mbar_wait(bar(kBarEmpty + i), ((x / kRing) & 1) ^ 1);
                    mbar_expect_tx(bar(kBarFull + i), kKvTileBytes);
                    const CUtensorMap* tm = ti.tree ? (kv ? &tm_tv : &tm_tk) : (kv ? &tm_v : &tm_k);
                    tma_load_4d(dst, tm, bar(kBarFull + i), 0, ti.row, 0, wk.g, ti.tree ? kEvictLast : kEvictNormal);
                }
                if (x == 0 && lane == 0) {
                    // a split item holds one M tile (Q buffer 0 serves both slots)
                    const int nq = wk.mode == kModePair ? 2 : 1;
                    for (int s = 0; s < nq; ++s) {
                        const int t0 = wk.b * pl.T_cap + (wk.row_base + s * kTileM) / pl.G;
                        mbar_expect_tx(bar(kBarQFull + s), kQTileBytes);
                        tma_load_5d(smem + kOffQ + s * kQTileBytes, &tm_q, bar(kBarQFull + s), 0, 0, t0, 0, wk.g,
                                    kEvictLast);
                    }
                }
                __syncwarp();
            }
            page_cur = page_next;
        }
      } else if (warp == 9 || warp == 10) {
        // ===== MMA issuers: one elected thread per SLOT (warp 9 -> slot 0, warp 10 -> slot 1).  The two
        // slots' chains (Q.K^T -> softmax -> P.V -> next Q.K^T) are independent, so each thread simply
        // walks its own chain and the tensor pipe interleaves them.  The chain's tensor phase is kept
        // short: the next unit's K tile is waited for BEFORE the P pieces, and the next Q.K^T is issued
        // right behind the last P.V piece (S and P share TMEM columns, so it cannot go earlier).
        // Both threads release every ring tile; a tile the slot does not use is released as soon as
        // its fill has been observed (so the arrival can only count for that fill). =====
        if (elect_one()) {
            const int s = warp - 9;
            const uint64_t qd = smem_desc(smem + kOffQ + (wk.mode == kModePair && s ? kQTileBytes : 0u), 16, 1024);
            const uint32_t sd = tmem + kTmemS + s * kTileN;  // S, overwritten by P (bf16, 64 columns)
            const uint32_t od = tmem + s * kD;
            uint32_t acc = 0, par = 0, n_ragged = 0;
            int jj = 0, ki = 0, kpar = 0;  // current tile and the ring slot / fill parity of its K
            auto ring_next = [&](int& i, int& p) { if (++i == kRing) { i = 0; p ^= 1; } };
            auto is_used = [&](int j) { return ((wk.uses(j) >> s) & 1u) != 0; };
            auto valid_of = [&](int j) { return tile_info(j).valid; };
            // Walk from tile nj to the slot's next used tile: an unused tile is released once its fills
            // have been observed; at a used tile, its K fill is awaited.  Non-blocking mode gives up at the
            // first fill that has not landed yet (returns false) and can be resumed.
            int nj = 0, nki = 0, nkpar = 0, nsub = 0;
            auto advance = [&](bool blocking) {
                while (nj < wk.n_tiles) {
                    if (is_used(nj)) {
                        if (blocking) mbar_wait(bar(kBarFull + nki), nkpar);
                        else if (!mbar_try_wait(bar(kBarFull + nki), nkpar)) return false;
                        return true;
                    }
                    while (nsub < 2) {
                        if (blocking) mbar_wait(bar(kBarFull + nki), nkpar);
                        else if (!mbar_try_wait(bar(kBarFull + nki), nkpar)) return false;
                        tc_commit(bar(kBarEmpty + nki));
                        ring_next(nki, nkpar);
                        ++nsub;
                    }
                    if (valid_of(nj) & 15) ++n_ragged;
                    nsub = 0;
                    ++nj;
                }
                return true;
            };
            auto issue_qk = [&](int j, int i) {
                const int tile_n = (valid_of(j) + 15) & ~15;  // MMA N (multiple of 16)
                const uint64_t kd = smem_desc(smem + kOffRing + i * kKvTileBytes, 16, 1024);
                const uint32_t id_qk = idesc(kTileM, (uint32_t)tile_n, 0);
                tc_fence_after();
#pragma unroll
                for (int kk = 0; kk < kD / 16; ++kk) {
                    const uint64_t off = (uint64_t)(((kk >> 2) * (kQTileBytes / 2) + (kk & 3) * 32) >> 4);
                    umma_ss(sd, qd + off, kd + off, id_qk, kk > 0);
                }
                tc_commit(bar(kBarSFull + s));
                tc_commit(bar(kBarEmpty + i));  // K_j is free once this Q.K^T has completed
            };
            advance(true);
            jj = nj; ki = nki; kpar = nkpar;
            if (jj < wk.n_tiles) {
                mbar_wait(bar(kBarQFull + (wk.mode == kModePair ? s : 0)), 0);
                issue_qk(jj, ki);
            }
            while (jj < wk.n_tiles) {
                const int valid = valid_of(jj);
                const int ksteps = ((valid + 15) & ~15) >> 4;  // K extent of P.V in 16-key steps
                int vi = ki, vpar = kpar;
                ring_next(vi, vpar);
                mbar_wait(bar(kBarFull + vi), vpar);
                if (valid & 15) mbar_wait(bar(kBarVFix + n_ragged++), 0);
                // the next unit of this slot and its K tile, before the P pieces arrive
                nj = jj + 1; nki = vi; nkpar = vpar; nsub = 0;
                ring_next(nki, nkpar);
                const bool next_ready = advance(false);
                const uint64_t vd = smem_desc(smem + kOffRing + vi * kKvTileBytes, kKvTileBytes / 2, 1024);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    // Every piece is awaited, also the ones past a ragged tile's end that feed no MMA: the
                    // softmax threads still store (zero) P there, and the next Q.K^T of the slot overwrites
                    // the same TMEM columns.
                    mbar_wait(bar(kBarPFull + 4 * s + q), par);
                    tc_fence_after();
#pragma unroll
                    for (int ks = 2 * q; ks < 2 * q + 2; ++ks)
                        if (ks < ksteps) umma_ts(od, sd + ks * 8, vd + (uint64_t)(ks * (2048 >> 4)), kIdescPV, acc | ks);
                }
                acc = 1;
                par ^= 1;
                tc_commit(bar(kBarEmpty + vi));  // V_j is free once these P.V pieces have completed
                if (!next_ready) advance(true);
                if (nj < wk.n_tiles) issue_qk(nj, nki);
                jj = nj; ki = nki; kpar = nkpar;
            }
            tc_commit(bar(kBarAllDone));
        }
      } else if (warp == 11) {
        // ===== V sanitiser: the P.V MMA runs over ceil16(valid) keys; rows valid..ceil16(valid)-1 of a
        // ragged V tile belong to nobody (next request, tree padding) and are multiplied by P = 0
        // exactly, so they must not hold NaN/Inf: zero them in shared memory.  A row is 2 x 128 B
        // (d halves); the 128B swizzle permutes 16-byte chunks inside a row's 128 B only.
        // The warp observes EVERY fill of every ring slot in order (a parity wait is only sound
        // then) and is the second arriver on each slot's empty barrier, so it can never be lapped. =====
        int x = 0, n_ragged = 0;
        for (int jj = 0; jj < wk.n_tiles; ++jj) {
            const int valid = tile_info(jj).valid;
            for (int kv = 0; kv < 2; ++kv, ++x) {
                const int i = x % kRing;
                mbar_wait(bar(kBarFull + i), (x / kRing) & 1);
                if (kv == 1 && (valid & 15) != 0) {
                    const int n_rows = ((valid + 15) & ~15) - valid;
                    for (int e = lane; e < n_rows * 16; e += 32) {  // 16 x 16 B per row
                        const int row = valid + (e >> 4), c16 = e & 15;
                        const uint32_t addr = smem + kOffRing + i * kKvTileBytes +
                                              (uint32_t)(c16 >> 3) * (kKvTileBytes / 2) + (uint32_t)row * 128u +
                                              (uint32_t)(c16 & 7) * 16u;
                        asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(addr), "r"(0u) : "memory");
                    }
                    fence_async_smem();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar(kBarVFix + n_ragged));
                    ++n_ragged;
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(kBarEmpty + i));
            }
        }
      }
    } else {
      asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegsSoftmax));
      if (!idle) {
        // ===== softmax: all eight warps serve ONE unit at a time, two threads per query row: warps 0..3
        // take key columns 0..63 of the S tile, warps 4..7 columns 64..127; thread (w, lane) of either
        // half owns query row w*32 + lane (TMEM lane).  Two warps per scheduler keep the MUFU pipe
        // saturated (a single warp reaches only ~2/3 of it), and because the units alternate between
        // the two slots, the tensor phase of one slot (P.V, next Q.K^T) runs under the other slot's
        // softmax.  The halves exchange their row maxima through shared memory once per unit. =====
        const int h = warp >> 2;
        const int w = warp & 3;
        const int rl = w * 32 + lane;  // row within the tile
        const uint32_t lane_addr = (uint32_t)(w * 32) << 16;
        const float c2 = pl.sm_scale * kLog2e;
        const float thr = kRescaleThreshold / c2;  // in raw score units
        float* xm = reinterpret_cast<float*>(smem_gen + kOffX);  // [2 unit parity][2 halves][128 rows]
        // per-slot running state in scalars (selected by the unrolled s)
        float m_run0 = -INFINITY, m_run1 = -INFINITY, l_run0 = 0.f, l_run1 = 0.f;
        int kcnt0 = 0, kcnt1 = 0;
        int n = 0;
        for (int jj = 0; jj < wk.n_tiles; ++jj) {
            const uint32_t use = wk.uses(jj);
            const TileInfo ti = tile_info(jj);
            const bool masked_tile = ti.tree || ti.valid < kTileN;
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                if (!((use >> s) & 1u)) continue;
                const int k = s ? kcnt1 : kcnt0;
                float m_cur = s ? m_run1 : m_run0, l_cur = s ? l_run1 : l_run0;
                const bool warp_active = w * 32 < wk.rows(s);
                const uint32_t sbuf = tmem + kTmemS + s * kTileN + lane_addr;
                const uint32_t o_addr = tmem + s * kD + h * 64 + lane_addr;
                mbar_wait(bar(kBarSFull + s), k & 1);
                uint32_t sv[64];
                float mxh = -INFINITY;
                if (warp_active) {
                    tc_fence_after();
                    D2SD_TMEM_LD32(sbuf + h * 64, sv, 0);
                    D2SD_TMEM_LD32(sbuf + h * 64 + 32, sv, 32);
                    tmem_wait_ld();
                    if (masked_tile) {
                        // keys past the tile's end, and (tree tiles) keys that are not ancestors-or-self of
                        // this row's node: bits 64h..64h+63 of the tile's 128 mask bits, -> -inf
                        uint32_t mw0 = 0xFFFFFFFFu, mw1 = 0xFFFFFFFFu;
                        if (ti.tree) {
                            const int t = min((wk.row_base + wk.row_off(s) + rl) / pl.G, wk.T - 1);
                            const uint32_t* mrow = a.mask + ((size_t)wk.b * pl.T_cap + t) * pl.W;
                            const int wi = ti.tt * 4 + h * 2;
                            mw0 = wi < pl.W ? mrow[wi] : 0u;
                            mw1 = wi + 1 < pl.W ? mrow[wi + 1] : 0u;
                        }
                        const int lim = ti.valid - h * 64;  // columns [lim, 64) of this half are past the end
#pragma unroll
                        for (int c = 0; c < 64; ++c) {
                            const uint32_t bit = ((c < 32 ? mw0 : mw1) >> (c & 31)) & 1u;
                            if (c >= lim || !bit) sv[c] = 0xFF800000u;
                        }
                    }
                    float mx0 = -INFINITY, mx1 = -INFINITY, mx2 = -INFINITY, mx3 = -INFINITY;
#pragma unroll
                    for (int c = 0; c < 64; c += 4) {
                        mx0 = fmaxf(mx0, __uint_as_float(sv[c]));
                        mx1 = fmaxf(mx1, __uint_as_float(sv[c + 1]));
                        mx2 = fmaxf(mx2, __uint_as_float(sv[c + 2]));
                        mx3 = fmaxf(mx3, __uint_as_float(sv[c + 3]));
                    }
                    mxh = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3));
                }
                xm[((n & 1) * 2 + h) * kTileM + rl] = mxh;
                named_bar_sync(1, 256);  // also orders "both halves have read S" before "P overwrites S"
                if (warp_active) {
                    const float mx = fmaxf(mxh, xm[((n & 1) * 2 + (h ^ 1)) * kTileM + rl]);
                    // lazy rescale: raise the running max only when it is exceeded by more than 2^8
                    const bool need = mx > m_cur + thr;
                    if (k == 0) {
                        m_cur = mx;
                    } else if (__any_sync(0xffffffffu, need)) {
                        const float alpha = need ? ex2((m_cur - mx) * c2) : 1.f;
                        // S_k ready implies the previous P.V into this O has landed (tcgen05.commit covers
                        // every earlier MMA of the issuing thread)
                        tc_fence_after();
#pragma unroll 1
                        for (int c0 = 0; c0 < 64; c0 += 32) {  // this half's 64 of the 128 O columns
                            uint32_t o[32];
                            D2SD_TMEM_LD32(o_addr + c0, o, 0);
                            tmem_wait_ld();
#pragma unroll
                            for (int c = 0; c < 32; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * alpha);
                            D2SD_TMEM_ST32(o_addr + c0, o, 0);
                        }
                        tmem_wait_st();
                        // The P.V of this unit accumulates into all 128 O columns as soon as ONE half has
                        // released its first piece: both halves of these 32 rows (warps w and w + 4 take the
                        // same decision, they see the same maxima) finish their rescale before either releases.
                        tc_fence_before();
                        named_bar_sync(2 + w, 64);
                        if (need) {
                            m_cur = mx;
                            l_cur *= alpha;
                        }
                    }
                    // a row with every key so far masked has m_run = -inf: exp2(-inf - 0) = 0, not NaN
                    const float ms = m_cur == -INFINITY ? 0.f : m_cur * c2;
                    float sum0 = 0.f, sum1 = 0.f;
                    // P[128 x 128] bf16 = 64 TMEM columns; this half writes columns 32h..32h+31 in two
                    // pieces (key quarters 2h, 2h+1), each released to the tensor pipe on its own.  The
                    // store of a piece is only waited for after the next piece's exponentials.
#pragma unroll
                    for (int q = 0; q < 2; ++q) {
                        float ev[32];
#pragma unroll
                        for (int c = 0; c < 32; ++c) ev[c] = ex2_ordered(__uint_as_float(sv[q * 32 + c]) * c2 - ms);
                        if (q > 0) {
                            tmem_wait_st();
                            tc_fence_before();
                            mbar_arrive(bar(kBarPFull + 4 * s + 2 * h));
                        }
                        uint32_t p[16];
                        float t0 = 0.f, t1 = 0.f, t2 = 0.f, t3 = 0.f;
#pragma unroll
                        for (int c = 0; c < 16; c += 2) {
                            t0 += ev[2 * c]; t1 += ev[2 * c + 1]; t2 += ev[2 * c + 2]; t3 += ev[2 * c + 3];
                            p[c] = pack2_bf16(ev[2 * c], ev[2 * c + 1]);
                            p[c + 1] = pack2_bf16(ev[2 * c + 2], ev[2 * c + 3]);
                        }
                        sum0 += t0 + t1;
                        sum1 += t2 + t3;
                        D2SD_TMEM_ST16(sbuf + h * 32 + q * 16, p);
                    }
                    l_cur += sum0 + sum1;
                    tmem_wait_st();
                    tc_fence_before();
                    mbar_arrive(bar(kBarPFull + 4 * s + 2 * h + 1));
                } else {
                    mbar_arrive(bar(kBarPFull + 4 * s + 2 * h));
                    mbar_arrive(bar(kBarPFull + 4 * s + 2 * h + 1));
                }
                if (s) { m_run1 = m_cur; l_run1 = l_cur; ++kcnt1; } else { m_run0 = m_cur; l_run0 = l_cur; ++kcnt0; }
                ++n;
            }
        }
        // ---- epilogue: O / l -> swizzled staging image in shared memory -> bulk copies to the partial
        // state (row r of the image: 32 chunks of 16 B, chunk c stored at position c ^ (r & 7)).  A pair
        // item writes one state per slot.  A split item first merges its two slots (two running states of
        // the same rows over disjoint keys) in registers and writes ONE state: the exchange through L2
        // carries 128 rows per CTA, not 256. ----
        mbar_wait(bar(kBarAllDone), 0);  // every MMA done: the ring is free for staging
        const bool split = wk.mode == kModeSplit;
        xm[(0 * 2 + h) * kTileM + rl] = l_run0;  // row sums of this half, both slots
        xm[(1 * 2 + h) * kTileM + rl] = l_run1;
        named_bar_sync(1, 256);
        const float l_tot0 = l_run0 + xm[(0 * 2 + (h ^ 1)) * kTileM + rl];
        const float l_tot1 = l_run1 + xm[(1 * 2 + (h ^ 1)) * kTileM + rl];
        const int n_out = wk.mode == kModePair ? 2 : 1;
#pragma unroll 1
        for (int o = 0; o < n_out; ++o) {
            // out state o = w0 * O_slot0 + w1 * O_slot1 (use0 / use1 are uniform over the CTA: a slot
            // without any unit holds an uninitialised accumulator and is not read at all)
            bool use0, use1;
            float w0, w1, lse_v;
            int rows_o;
            if (split) {
                use0 = kcnt0 > 0;
                use1 = kcnt1 > 0;
                const float m0 = use0 ? m_run0 : -INFINITY, m1 = use1 ? m_run1 : -INFINITY;
                const float m = fmaxf(m0, m1);
                const float a0 = m0 == -INFINITY ? 0.f : ex2((m0 - m) * c2);
                const float a1 = m1 == -INFINITY ? 0.f : ex2((m1 - m) * c2);
                const float l = a0 * l_tot0 + a1 * l_tot1;
                const float inv = l > 0.f ? 1.f / l : 0.f;  // l = 0: every key of the chunk masked
                w0 = a0 * inv;
                w1 = a1 * inv;
                lse_v = l > 0.f ? m * pl.sm_scale + logf(l) : -INFINITY;
                rows_o = wk.rows0;
            } else {
                const bool any = (o ? kcnt1 : kcnt0) > 0;  // false: empty chunk 0 -> state (0, -inf)
                use0 = any && o == 0;
                use1 = any && o == 1;
                const float lt = o ? l_tot1 : l_tot0, mf = o ? m_run1 : m_run0;
                const float inv = any && lt > 0.f ? 1.f / lt : 0.f;
                w0 = use0 ? inv : 0.f;
                w1 = use1 ? inv : 0.f;
                lse_v = any && lt > 0.f ? mf * pl.sm_scale + logf(lt) : -INFINITY;
                rows_o = wk.rows(o);
            }
            const size_t prow0 = (size_t)wk.group * pl.grp_rows + wk.part_row0(o);
            float* po = a.part_o + prow0 * kD;
            float* plse = a.part_lse + prow0;
            const bool row_ok = rl < rows_o;
            const bool warp_active = w * 32 < rows_o;
            const uint32_t stage = smem + kOffRing + (uint32_t)o * (2 * kKvTileBytes);
            if (warp_active) {
                tc_fence_after();
                const uint32_t srow = stage + (uint32_t)rl * 512u;
                const uint32_t o_addr = tmem + h * 64 + lane_addr;
#pragma unroll
                for (int c0 = 0; c0 < 64; c0 += 32) {
                    uint32_t ov0[32], ov1[32];
                    if (use0) D2SD_TMEM_LD32(o_addr + c0, ov0, 0);
                    if (use1) D2SD_TMEM_LD32(o_addr + kD + c0, ov1, 0);
                    tmem_wait_ld();
                    float acc[32];
#pragma unroll
                    for (int c = 0; c < 32; ++c) {
                        acc[c] = use0 ? __uint_as_float(ov0[c]) * w0 : 0.f;
                        if (use1) acc[c] += __uint_as_float(ov1[c]) * w1;
                    }
#pragma unroll
                    for (int c = 0; c < 32; c += 4) {
                        const uint32_t chunk = (uint32_t)((h * 64 + c0 + c) >> 2);
                        const uint32_t phys = chunk ^ ((uint32_t)rl & 7u);
                        asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(srow + phys * 16u), "f"(acc[c]),
                                     "f"(acc[c + 1]), "f"(acc[c + 2]), "f"(acc[c + 3])
                                     : "memory");
                    }
                }
                if (h == 0 && row_ok) plse[rl] = lse_v;
                fence_async_smem();
            }
            named_bar_sync(1, 256);  // both halves of every row are staged
            if (warp_active && h == (o & 1) && lane == 0) {
                // this warp's rows: one contiguous piece of the image and of the partial state
                const int nrows = min(32, rows_o - w * 32);
                bulk_store(po + (size_t)(w * 32) * kD, stage + (uint32_t)(w * 32) * 512u, (uint32_t)nrows * 512u);
                bulk_commit();
            }
        }
        if (lane == 0) {
            bulk_wait_all();
            asm volatile("fence.proxy.async;" ::: "memory");
        }
        __syncwarp();

        // ---- publish this CTA's partial states, wait for the group, merge this CTA's share of rows ----
        const unsigned expected = (unsigned)wk.n_chunks;
        unsigned* cnt = a.counters + 2 * wk.group;  // [0] arrivals, [1] done
        named_bar_sync(1, 256);  // every thread's partial-state writes happen before the leader's release
        unsigned done_before = 0;
        if (warp == 0 && lane == 0) {
            asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(cnt) : "memory");
            unsigned seen, spins = 0;
            do {
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(cnt) : "memory");
                if (seen < expected) {
                    __nanosleep(20);
                    if (++spins > (1u << 24)) __trap();  // a scheduling assumption broke: fail, do not hang
                }
            } while (seen < expected);
            // this CTA is past the wait: count it out now, the round trip hides behind the merge
            done_before = atomicAdd(cnt + 1, 1u);
        }
        named_bar_sync(1, 256);
        asm volatile("fence.proxy.async;" ::: "memory");  // the bulk copies below read what the acquire made visible
        merge_rows(pl, a, dbg_rows, wk, smem + kOffQ, smem_gen + kOffQ, bar(kBarMerge), warp, lane);
        if (warp == 0 && lane == 0) {
            if (done_before == expected - 1) {  // last CTA out: everybody is past the wait
                cnt[0] = 0;
                cnt[1] = 0;
            }
        }
      }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 10) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(kTmemCols) : "memory");
    }
}

// ---- host side ----------------------------------------------------------------------------------
using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

int32_t encode(CUtensorMap* tm, const void* base, int rank, const cuuint64_t* dims, const cuuint64_t* strides,
               const cuuint32_t* box, const char* what) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return set_error(D2SD_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
    cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, (cuuint32_t)rank, const_cast<void*>(base), dims, strides, box,
                    estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return set_error(D2SD_ERR_CUDA, "cuTensorMapEncodeTiled(%s) failed with CUresult %d", what, (int)r);
    return D2SD_OK;
}

}  // namespace

bool attn_cascade_tc_supported(const AttnPlan& pl) {
    // contiguous or 16-key-paged KV, rows of one query tile must be whole tree nodes (128 % G == 0),
    // and the tensor-map extents must fit.
    return (pl.page_size == 0 || pl.page_size == 16) && pl.d == kD && pl.G <= 128 && (128 % pl.G) == 0 &&
           (int64_t)pl.B * pl.T_cap < (1ll << 31) && pl.kv_rows < (1ll << 31);
}

int32_t launch_attn_cascade_tc(const AttnPlan& pl, const AttnArgs& a, int mode, float* dbg_rows, cudaStream_t s) {
    static unsigned long long attr_done = 0;
    if (first_use_on_device(attr_done))
        D2SD_CHECK_CUDA(cudaFuncSetAttribute(attn_cascade_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)kSmemBytes));
    CUtensorMap tm_q, tm_k, tm_v, tm_tk, tm_tv;
    {   // Q [B*T_cap, Hq, d] viewed as (d_lo 64, hh G, t B*T_cap, d_hi 2, g Hkv): one box = one 128-row query tile
        const cuuint64_t dims[5] = {64, (cuuint64_t)pl.G, (cuuint64_t)pl.B * pl.T_cap, 2, (cuuint64_t)pl.Hkv};
        const cuuint64_t strides[4] = {(cuuint64_t)kD * 2, (cuuint64_t)pl.Hq * kD * 2, 128, (cuuint64_t)pl.G * kD * 2};
        const cuuint32_t box[5] = {64, (cuuint32_t)pl.G, (cuuint32_t)(kTileM / pl.G), 2, 1};
        if (int32_t st = encode(&tm_q, a.q, 5, dims, strides, box, "q")) return st;
    }
    {   // K/V [rows, Hkv, d] viewed as (d_lo 64, row, d_hi 2, g): one box = one 128-key tile.  Rows past the
        // end of the tensor are zero-filled by TMA; the kernel masks every key past a tile's valid count.
        const cuuint64_t strides[3] = {(cuuint64_t)pl.Hkv * kD * 2, 128, (cuuint64_t)kD * 2};
        const cuuint32_t box[4] = {64, kTileN, 2, 1};
        const cuuint64_t tdims[4] = {64, (cuuint64_t)pl.B * pl.T_cap, 2, (cuuint64_t)pl.Hkv};
        if (int32_t st = encode(&tm_tk, a.tree_k, 4, tdims, strides, box, "tree_k")) return st;
        if (int32_t st = encode(&tm_tv, a.tree_v, 4, tdims, strides, box, "tree_v")) return st;
        if (pl.kv_rows > 0 && a.k_cache && a.v_cache && pl.page_size > 0) {
            // paged pool [P, 16, Hkv, d] viewed as (d_lo 64, slot 16, d_hi 2, g, page): one box = one d half
            // of one page of one kv head (2 KiB); 16 boxes make a 128-key tile in the same shared-memory
            // image as a contiguous tile (the 128B swizzle is a function of the shared-memory address)
            const cuuint64_t pdims[5] = {64, 16, 2, (cuuint64_t)pl.Hkv, (cuuint64_t)(pl.kv_rows / 16)};
            const cuuint64_t pstrides[4] = {(cuuint64_t)pl.Hkv * kD * 2, 128, (cuuint64_t)kD * 2,
                                            (cuuint64_t)16 * pl.Hkv * kD * 2};
            const cuuint32_t pbox[5] = {64, 16, 1, 1, 1};
            if (int32_t st = encode(&tm_k, a.k_cache, 5, pdims, pstrides, pbox, "k_pool")) return st;
            if (int32_t st = encode(&tm_v, a.v_cache, 5, pdims, pstrides, pbox, "v_pool")) return st;
        } else if (pl.kv_rows > 0 && a.k_cache && a.v_cache) {
            const cuuint64_t dims[4] = {64, (cuuint64_t)pl.kv_rows, 2, (cuuint64_t)pl.Hkv};
            if (int32_t st = encode(&tm_k, a.k_cache, 4, dims, strides, box, "k_cache")) return st;
            if (int32_t st = encode(&tm_v, a.v_cache, 4, dims, strides, box, "v_cache")) return st;
        } else {  // no committed prefix at all (max_ctx_len == 0): the maps are never used
            tm_k = tm_tk;
            tm_v = tm_tv;
        }
    }
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(pl.n_pair * pl.chunks_a + pl.n_single * pl.chunks_b, pl.Hkv, pl.B);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = kSmemBytes;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;  // PDL: see the file header
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    D2SD_CHECK_CUDA(cudaLaunchKernelEx(&cfg, attn_cascade_tc_kernel, tm_q, tm_k, tm_v, tm_tk, tm_tv, pl, a, mode, dbg_rows));
    D2SD_CHECK_LAUNCH("attn_cascade_tc_kernel");
    return D2SD_OK;
}


}  // namespace d2sd
