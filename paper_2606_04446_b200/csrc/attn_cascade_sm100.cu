// Stage (c), fused: cascade tree-verify attention in ONE launch on tcgen05 / TMEM / TMA (sm_100a).
// PAPER.md:52, :124, :154.
//
// Every tree query of every branch and every GQA head of one kv head is a row of one batched query
// matrix (row r = t*G + hh), cut into 128-row M tiles; up to three M tiles form an "M group".  The
// keys of a request are the committed prefix followed by the tree-local keys, cut into 128-key
// tiles: prefix tiles 0..np-1 (np = ceil(L/128)) and tree tiles np..np+nt-1 (nt = ceil(T/128)); the
// tree tiles are ordinary key tiles whose scores additionally pass the node's ancestor-mask bits.
// The tile sequence is cut into `num_splits` chunks.  One work item = (request b, kv head g, M
// group, chunk) and is served by a PAIR of CTAs (rank 0 / 1) that stream the same K/V chunk:
//
//   M tiles in the group   rank 0 computes                rank 1 computes
//   3                      tile 0 (all key tiles)         tile 1 (all key tiles)
//                          + tile 2 on even key tiles     + tile 2 on odd key tiles
//   2                      tile 0                         tile 1
//   1                      tile 0 on even key tiles       tile 0 on odd key tiles
//
// so each CTA holds at most two fp32 O accumulators (2 x 128 TMEM columns) and two S/P buffers
// (2 x 128 columns) -- the whole 512-column TMEM -- and the tensor work of the 3-tile case is split
// evenly.  Per unit (one M tile x one 128-key tile):
//
//   S[128 x 128] = Q_m[128 x 128] . K_j^T    tcgen05.mma, A/B from 128B-swizzled SMEM (TMA), D in TMEM
//   P            = exp2(c*(S - m_run))       softmax warpgroup, one thread per row (TMEM lane), P -> TMEM
//   O_m[128x128] += P[128 x 128] . V_j       tcgen05.mma, A = P from TMEM, B = V (MN-major SMEM)
//
// N = 128 keys per MMA keeps the tensor pipe MMA-bound (measured: 67 cycles per M128 N128 K16
// instruction against 64 ideal; N = 64 instructions are issue/SMEM-bound at 54 cycles against 32).
//
// Warp roles (384 threads): warp 0 = TMA producer, warp 1 = MMA issuer (one thread), warp 2 = TMEM
// allocator, warp 3 = zeroes the V rows behind a ragged tile end (they are multiplied by exact zeros
// and may hold anything, NaN included), warps 4..11 = softmax: two threads per query row (TMEM
// lane), warps 4..7 on key columns 0..63 and warps 8..11 on columns 64..127 of every S tile, so that
// two warps per scheduler share the MUFU pipe; the halves exchange row maxima through shared
// memory.  Running max / sum stay in registers; the running max is only raised when a tile maximum
// exceeds it by more than 2^8 (lazy rescale), in which case the owning threads rescale their O row
// in TMEM before the next P.V.
//
// Cascade merge in the same launch (log-sum-exp state merge): every CTA writes one
// partial state (normalised O fp32, LSE) per accumulator slot to the workspace (it stays in L2),
// publishes it with a release-increment of its group's arrival counter, waits until all
// 2*num_splits CTAs of the group (same b, g, M group) have arrived, and then merges ITS share of the
// group's rows (rows are dealt round-robin to the group's softmax warps) and writes the bf16 output
// and the LSE.  The counters reset themselves (last CTA out), so the workspace header only has to
// be zero before the first call (d2sd_cascade_workspace_init).  The wait is safe because a group is
// 2*num_splits consecutive blocks of the grid's linear order: the oldest unfinished group always
// has all its CTAs resident or done; the spin is bounded and traps instead of hanging.
// Workspace layout (private to this file): header of arrival/done counters, then O
// [b][slot][g][rows_pad][128] fp32 (XOR-swizzled 16-byte chunks are undone before the store) and
// LSE [b][slot][g][rows_pad].
#include <cuda.h>

#include "common.cuh"

namespace d2sd {
namespace {

constexpr int kD = 128;
constexpr int kTileM = 128;
constexpr int kTileN = 128;
constexpr int kGroupTiles = 3;  // M tiles per M group
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
constexpr uint32_t kTmemS = 256;  // two S/P buffers of 128 columns behind the two O accumulators
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kRescaleThreshold = 8.0f;  // log2 units

// barrier slots (8 bytes each) at kOffBar.  S-ready / P-ready / O-ready exist PER ACCUMULATOR SLOT
// (phase = unit count of that slot): a parity wait is only sound if the waiter observes every phase,
// so barriers are never shared between the two softmax warpgroups.
enum : uint32_t {
    kBarQFull = 0,                     // [2]
    kBarFull = 2,                      // [kRing]
    kBarEmpty = kBarFull + kRing,      // [kRing]
    kBarSFull = kBarEmpty + kRing,     // [2]
    kBarPFull = kBarSFull + 2,         // [2]
    kBarODone = kBarPFull + 2,         // [2]
    kBarAllDone = kBarODone + 2,       // every MMA of the CTA has completed
    kBarVFix = kBarAllDone + 1,        // [2] warp 3 has zeroed the V rows behind a ragged tile end; a CTA
                                       // meets at most two ragged tiles (last prefix tile, last tree tile)
    kNumBars = kBarVFix + 2,
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
__device__ __forceinline__ void named_bar_sync(uint32_t id, uint32_t threads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}
constexpr uint64_t kEvictFirst = 0x12F0000000000000ull;  // streamed: KV
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
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

__device__ __forceinline__ float ex2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ uint32_t pack2_bf16(float lo, float hi) {
    __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&v);
}

// Which accumulator slots of a CTA are live, and on which key tiles the shared slot runs.
struct SlotPlan {
    int tile[2];   // M tile (within the M group) of slot 0 (own) / slot 1 (shared), or -1
    __device__ __forceinline__ bool own() const { return tile[0] >= 0; }
    __device__ __forceinline__ bool shared_on(int j, int rank) const { return tile[1] >= 0 && (j & 1) == rank; }
    __device__ __forceinline__ bool used(int j, int rank) const { return own() || shared_on(j, rank); }
};
__device__ __forceinline__ SlotPlan make_slots(int MT, int rank) {
    SlotPlan s;
    s.tile[0] = MT >= 2 ? rank : -1;
    s.tile[1] = (MT & 1) ? MT - 1 : -1;
    return s;
}

#ifdef D2SD_TIMELINE
// Debug builds only (-DD2SD_TIMELINE): per-CTA cycle stamps of pipeline events, read back with
// d2sd_debug_timeline().  Not part of the C ABI.
__device__ long long g_timeline[256][128];
#define TL(slot)                                                                                    \
    do {                                                                                            \
        const int _c = blockIdx.x + gridDim.x * blockIdx.y;                                         \
        if (_c < 256 && (slot) < 128) g_timeline[_c][(slot)] = clock64() - tl_t0;                   \
    } while (0)
#else
#define TL(slot) do {} while (0)
#endif

// -------------------------------------------------------------------------------------------------
// Cascade merge of one group's rows (log-sum-exp state merge):
//   LSE = log sum_p e^{LSE_p};  O = sum_p e^{LSE_p - LSE} O_p   over the slots that hold the row's M tile.
// Warp `gw` of `n_gw` takes rows gw, gw + n_gw, ... of the group; lane i first fetches the LSE of
// relevant slot i, then the warp sweeps the slots' O rows (512 B each, coalesced).  The partial
// states were written by other SMs: read them at L2 (ld.global.cg).
__device__ __forceinline__ void merge_rows(const AttnPlan& pl, const AttnArgs& a, float* dbg_rows, int b, int g,
                                           int row_base, int rows_g, int MT, int gw, int n_gw, int lane) {
    const int G = pl.G;
    for (int rr = gw; rr < rows_g; rr += n_gw) {
        const int r = row_base + rr;
        const int tl = rr / kTileM;
        const bool own = MT >= 2 && tl < 2;  // tile owned by rank tl; otherwise shared by both ranks
        const int n_rel = own ? pl.num_splits : 2 * pl.num_splits;  // relevant slots
        auto row_of = [&](int i) {
            const int slot = own ? 2 * i + tl : i;
            return (((size_t)b * pl.NSLOT + slot) * pl.Hkv + g) * pl.rows_pad + r;
        };
        float m = -INFINITY, wsum = 0.f;
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int base = 0; base < n_rel; base += 32) {
            const int i = base + lane;
            const float l = i < n_rel ? __ldcg(a.part_lse + row_of(i)) : -INFINITY;
            float mb = l;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) mb = fmaxf(mb, __shfl_xor_sync(0xffffffffu, mb, o));
            if (mb == -INFINITY) continue;
            if (mb > m) {  // rescale what has been accumulated so far (only with > 32 relevant slots)
                const float sc = m == -INFINITY ? 0.f : __expf(m - mb);
                acc.x *= sc; acc.y *= sc; acc.z *= sc; acc.w *= sc;
                wsum *= sc;
                m = mb;
            }
            const float wl = l == -INFINITY ? 0.f : __expf(l - m);
            const int cnt = min(32, n_rel - base);
#pragma unroll 6
            for (int q = 0; q < cnt; ++q) {
                const float w = __shfl_sync(0xffffffffu, wl, q);
                if (w == 0.f) continue;
                const float4 o = __ldcg(reinterpret_cast<const float4*>(a.part_o + row_of(base + q) * kD) + lane);
                wsum += w;
                acc.x += w * o.x; acc.y += w * o.y; acc.z += w * o.z; acc.w += w * o.w;
            }
        }
        const float inv = wsum > 0.f ? 1.f / wsum : 0.f;  // no key at all (L = 0, prefix-only mode): O = 0, LSE = -inf
        const float lse = wsum > 0.f ? m + logf(wsum) : -INFINITY;
        const int t = r / G;
        const size_t orow = ((size_t)b * pl.T_cap + t) * pl.Hq + g * G + (r - t * G);
        if (dbg_rows) {  // fp32 state for tests: d values of O, then the LSE
            float* d0 = dbg_rows + orow * (kD + 1);
            d0[lane * 4 + 0] = acc.x * inv; d0[lane * 4 + 1] = acc.y * inv;
            d0[lane * 4 + 2] = acc.z * inv; d0[lane * 4 + 3] = acc.w * inv;
            if (lane == 0) d0[kD] = lse;
            continue;
        }
        __nv_bfloat162 lo = __floats2bfloat162_rn(acc.x * inv, acc.y * inv);
        __nv_bfloat162 hi = __floats2bfloat162_rn(acc.z * inv, acc.w * inv);
        uint2 pk;
        pk.x = *reinterpret_cast<uint32_t*>(&lo);
        pk.y = *reinterpret_cast<uint32_t*>(&hi);
        *reinterpret_cast<uint2*>(a.out + orow * kD + lane * 4) = pk;
        if (a.lse && lane == 0) a.lse[orow] = lse;
    }
}

// mode bits: 1 = include the prefix tiles, 2 = include the tree tiles (3 = the whole cascade).
struct TileInfo {
    int valid;      // keys of the tile that exist (1..128)
    int row;        // first row of the tile in its tensor map
    bool tree;      // tree tile (ancestor mask applies), else prefix tile
    int tt;         // tree tile index (tree tiles only)
};

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
#ifdef D2SD_TIMELINE
    const long long tl_t0 = clock64();
#endif
    const int rank = blockIdx.x & 1, split = blockIdx.x >> 1, g = blockIdx.y;
    const int b = blockIdx.z / pl.n_mgroups, mg = blockIdx.z - b * pl.n_mgroups;
    const int G = pl.G;
    const int T = a.tree_len[b];
    const int rows_valid = T * G;
    const int row_base = mg * (kGroupTiles * kTileM);
    if (row_base >= rows_valid) return;  // the whole group returns: nobody waits for it
    const int rows_g = min(kGroupTiles * kTileM, rows_valid - row_base);
    const int MT = (rows_g + kTileM - 1) / kTileM;
    const SlotPlan sp = make_slots(MT, rank);
    const int L = a.ctx_len[b];
    // key tiles of this request: prefix tiles [0, np), tree tiles [np, np + nt); this chunk: [j_begin, j_end)
    const int np = (mode & 1) ? (L + kTileN - 1) / kTileN : 0;
    const int nt = (mode & 2) ? (T + kTileN - 1) / kTileN : 0;
    const int tps = max(1, (np + nt + pl.num_splits - 1) / pl.num_splits);
    const int j_begin = split * tps;
    const int n_tiles = max(0, min(np + nt, j_begin + tps) - j_begin);
    const int slot_id = 2 * split + rank;
    const size_t slot_row0 = (((size_t)b * pl.NSLOT + slot_id) * pl.Hkv + g) * pl.rows_pad;
    float* po = a.part_o + slot_row0 * kD;
    float* plse = a.part_lse + slot_row0;
    const int kv_row0 = a.kv_indptr ? a.kv_indptr[b] : 0;
    auto tile_info = [&](int jj) {
        const int j = j_begin + jj;
        TileInfo ti;
        ti.tree = j >= np;
        ti.tt = j - np;
        ti.valid = ti.tree ? min(kTileN, T - ti.tt * kTileN) : min(kTileN, L - j * kTileN);
        ti.row = ti.tree ? b * pl.T_cap + ti.tt * kTileN : kv_row0 + j * kTileN;
        return ti;
    };

    const uint32_t bar0 = smem + kOffBar;
    auto bar = [&](uint32_t i) { return bar0 + 8u * i; };
    volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem_gen + kOffBar + 8u * kTmemSlot);

    if (warp == 0 && lane == 0) {
        mbar_init(bar(kBarQFull + 0), 1);
        mbar_init(bar(kBarQFull + 1), 1);
        for (int i = 0; i < kRing; ++i) {
            mbar_init(bar(kBarFull + i), 1);
            mbar_init(bar(kBarEmpty + i), 2);  // the MMA's commit + the V sanitiser
        }
        for (int s = 0; s < 2; ++s) {
            mbar_init(bar(kBarSFull + s), 1);
            mbar_init(bar(kBarPFull + s), 2 * kTileM);
            mbar_init(bar(kBarODone + s), 1);
        }
        mbar_init(bar(kBarAllDone), 1);
        mbar_init(bar(kBarVFix + 0), 1);
        mbar_init(bar(kBarVFix + 1), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        tma_prefetch_desc(&tm_q);
        tma_prefetch_desc(&tm_k);
        tma_prefetch_desc(&tm_v);
        tma_prefetch_desc(&tm_tk);
        tma_prefetch_desc(&tm_tv);
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(bar(kTmemSlot)),
                     "r"(kTmemCols)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    if (tid == 0) TL(0);

    if (warp == 0) {
        // ===== TMA producer: K_0 first (the first MMA needs it), then the Q tiles, then the ring =====
        if (lane == 0) {
            int x = 0;  // ring position of the next tile to load
            bool q_sent = false;
            for (int j = 0; j < n_tiles; ++j) {
                if (!sp.used(j, rank)) continue;
                const TileInfo ti = tile_info(j);
                for (int kv = 0; kv < 2; ++kv, ++x) {
                    const int i = x % kRing;
                    mbar_wait(bar(kBarEmpty + i), ((x / kRing) & 1) ^ 1);
                    mbar_expect_tx(bar(kBarFull + i), kKvTileBytes);
                    const CUtensorMap* tm = ti.tree ? (kv ? &tm_tv : &tm_tk) : (kv ? &tm_v : &tm_k);
                    tma_load_4d(smem + kOffRing + i * kKvTileBytes, tm, bar(kBarFull + i), 0, ti.row, 0, g,
                                ti.tree ? kEvictLast : kEvictFirst);
                    if (!q_sent) {
                        q_sent = true;
                        for (int s = 0; s < 2; ++s) {
                            if (sp.tile[s] < 0) continue;
                            const int t0 = b * pl.T_cap + (row_base + sp.tile[s] * kTileM) / G;
                            mbar_expect_tx(bar(kBarQFull + s), kQTileBytes);
                            tma_load_5d(smem + kOffQ + s * kQTileBytes, &tm_q, bar(kBarQFull + s), 0, 0, t0, 0, g,
                                        kEvictLast);
                        }
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (one thread).  Issue order: QK(n+1) before PV(n), so that the tensor pipe
        // works on the next S while the softmax warpgroup turns S_n into P_n. =====
        if (lane == 0) {
            const uint64_t qd[2] = {smem_desc(smem + kOffQ, 16, 1024), smem_desc(smem + kOffQ + kQTileBytes, 16, 1024)};
            int n = 0, x = 0;
            int cnt_qk[2] = {0, 0}, cnt_pv[2] = {0, 0};
            // the PV that is still owed (unit n-1)
            bool pend = false, pend_last = false;
            int pend_slot = 0, pend_sbuf = 0, pend_vx = 0, pend_n = 0;
            bool v_waited = false, pend_ragged = false;
            int n_ragged = 0;
            auto do_pv = [&]() {
                const int s = pend_slot, vi = pend_vx % kRing;
                mbar_wait(bar(kBarPFull + s), cnt_pv[s] & 1);
                if (!v_waited) {
                    mbar_wait(bar(kBarFull + vi), (pend_vx / kRing) & 1);
                    if (pend_ragged) mbar_wait(bar(kBarVFix + n_ragged++), 0);
                    v_waited = true;
                }
                tc_fence_after();
                const uint64_t vd = smem_desc(smem + kOffRing + vi * kKvTileBytes, kKvTileBytes / 2, 1024);
                const uint32_t pa = tmem + kTmemS + pend_sbuf * kTileN;
                const uint32_t od = tmem + s * kD;
                const int ksteps = pend_n >> 4;
#pragma unroll 1
                for (int ks = 0; ks < ksteps; ++ks)
                    umma_ts(od, pa + ks * 8, vd + (uint64_t)(ks * (2048 >> 4)), kIdescPV, (cnt_pv[s] | ks) != 0);
                tc_commit(bar(kBarODone + s));
                if (pend_last) tc_commit(bar(kBarEmpty + vi));
                ++cnt_pv[s];
                pend = false;
            };
            for (int j = 0; j < n_tiles; ++j) {
                if (!sp.used(j, rank)) continue;
                const int kx = x, vx = x + 1;
                x += 2;
                const int ki = kx % kRing;
                const int valid = tile_info(j).valid;
                const int tile_n = (valid + 15) & ~15;  // MMA N of Q.K^T and K extent of P.V (multiple of 16)
                const bool sh = sp.shared_on(j, rank);
                mbar_wait(bar(kBarFull + ki), (kx / kRing) & 1);
                const uint64_t kd = smem_desc(smem + kOffRing + ki * kKvTileBytes, 16, 1024);
                const uint32_t id_qk = idesc(kTileM, (uint32_t)tile_n, 0);
                for (int s = 0; s < 2; ++s) {
                    if (s == 0 ? !sp.own() : !sh) continue;
                    const bool last_of_tile = (s == 1) || !sh;
                    if (cnt_qk[s] == 0) mbar_wait(bar(kBarQFull + s), 0);
                    TL(16 + 3 * n);
                    tc_fence_after();
                    const uint32_t sd = tmem + kTmemS + (n & 1) * kTileN;
#pragma unroll
                    for (int kk = 0; kk < kD / 16; ++kk) {
                        const uint64_t off = (uint64_t)(((kk >> 2) * (kQTileBytes / 2) + (kk & 3) * 32) >> 4);
                        umma_ss(sd, qd[s] + off, kd + off, id_qk, kk > 0);
                    }
                    tc_commit(bar(kBarSFull + s));
                    if (last_of_tile) tc_commit(bar(kBarEmpty + ki));
                    ++cnt_qk[s];
                    if (pend) {
                        do_pv();
                        TL(16 + 3 * (n - 1) + 2);
                    }
                    pend = true; pend_slot = s; pend_sbuf = n & 1; pend_vx = vx; pend_n = tile_n;
                    pend_last = last_of_tile;
                    pend_ragged = (valid & 15) != 0;
                    if (s == 0 || !sp.own()) v_waited = false;  // first unit of this key tile: V_j not yet waited for
                    ++n;
                }
            }
            if (pend) do_pv();
            tc_commit(bar(kBarAllDone));
        }
    } else if (warp == 3) {
        // ===== V sanitiser: the P.V MMA runs over ceil16(valid) keys; rows valid..ceil16(valid)-1 of a
        // ragged V tile belong to nobody (next request, tree padding) and are multiplied by P = 0
        // exactly, so they must not hold NaN/Inf: zero them in shared memory.  A row is 2 x 128 B
        // (d halves); the 128B swizzle permutes 16-byte chunks inside a row's 128 B only.
        // The warp observes EVERY fill of every ring slot in order (a parity wait is only sound
        // then) and is the second arriver on each slot's empty barrier, so it can never be lapped. =====
        int x = 0, n_ragged = 0;
        for (int j = 0; j < n_tiles; ++j) {
            if (!sp.used(j, rank)) continue;
            const int valid = tile_info(j).valid;
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
    } else if (warp >= 4) {
        // ===== softmax: warps 4..7 take key columns 0..63 of every S tile, warps 8..11 columns 64..127;
        // thread (w, lane) of either half owns query row w*32 + lane (TMEM lane).  The two halves
        // exchange their row maxima through shared memory once per unit. =====
        const int h = (warp - 4) >> 2;
        const int w = warp & 3;
        const int rl = w * 32 + lane;  // row within the tile
        const uint32_t lane_addr = (uint32_t)(w * 32) << 16;
        const float c2 = pl.sm_scale * kLog2e;
        const float thr = kRescaleThreshold / c2;  // in raw score units
        float* xm = reinterpret_cast<float*>(smem_gen + kOffX);  // [2 unit parity][2 halves][128 rows]
        float m_run[2] = {-INFINITY, -INFINITY}, l_run[2] = {0.f, 0.f};
        int kcnt[2] = {0, 0};
        int n = 0;
        for (int j = 0; j < n_tiles; ++j) {
            if (!sp.used(j, rank)) continue;
            const bool sh = sp.shared_on(j, rank);
            const TileInfo ti = tile_info(j);
            const bool masked_tile = ti.tree || ti.valid < kTileN;
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                if (s == 0 ? !sp.own() : !sh) continue;
                const int k = kcnt[s];
                const bool warp_active = (row_base + sp.tile[s] * kTileM + w * 32) < rows_valid;
                const uint32_t sbuf = tmem + kTmemS + (n & 1) * kTileN + lane_addr;
                const uint32_t o_addr = tmem + s * kD + h * 64 + lane_addr;
                mbar_wait(bar(kBarSFull + s), k & 1);
                if (warp == 4 && lane == 0) TL(64 + 2 * n);
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
                            const int t = min((row_base + sp.tile[s] * kTileM + rl) / G, T - 1);
                            const uint32_t* mrow = a.mask + ((size_t)b * pl.T_cap + t) * pl.W;
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
                bool saw_o = false;      // every phase of O-done must be observed (parity waits)
                if (warp_active) {
                    const float mx = fmaxf(mxh, xm[((n & 1) * 2 + (h ^ 1)) * kTileM + rl]);
                    // lazy rescale: raise the running max only when it is exceeded by more than 2^8
                    const bool need = mx > m_run[s] + thr;
                    if (k == 0) {
                        m_run[s] = mx;
                    } else if (__any_sync(0xffffffffu, need)) {
                        const float alpha = need ? ex2((m_run[s] - mx) * c2) : 1.f;
                        mbar_wait(bar(kBarODone + s), (k - 1) & 1);  // previous P.V into this O has landed
                        saw_o = true;
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
                        if (need) {
                            m_run[s] = mx;
                            l_run[s] *= alpha;
                        }
                    }
                    // a row with every key so far masked has m_run = -inf: exp2(-inf - 0) = 0, not NaN
                    const float ms = m_run[s] == -INFINITY ? 0.f : m_run[s] * c2;
                    float sum0 = 0.f, sum1 = 0.f;
                    uint32_t p[32];
#pragma unroll
                    for (int c = 0; c < 32; c += 2) {
                        const float e0 = ex2(__uint_as_float(sv[2 * c]) * c2 - ms);
                        const float e1 = ex2(__uint_as_float(sv[2 * c + 1]) * c2 - ms);
                        const float e2 = ex2(__uint_as_float(sv[2 * c + 2]) * c2 - ms);
                        const float e3 = ex2(__uint_as_float(sv[2 * c + 3]) * c2 - ms);
                        sum0 += e0 + e1;
                        sum1 += e2 + e3;
                        p[c] = pack2_bf16(e0, e1);
                        p[c + 1] = pack2_bf16(e2, e3);
                    }
                    l_run[s] += sum0 + sum1;
                    // P[128 x 128] bf16 = 64 columns (2 keys per column): this half writes columns 32h..32h+31
                    D2SD_TMEM_ST32(sbuf + h * 32, p, 0);
                    tmem_wait_st();
                    tc_fence_before();
                }
                mbar_arrive(bar(kBarPFull + s));
                if (warp == 4 && lane == 0) TL(64 + 2 * n + 1);
                if (k > 0 && !saw_o) mbar_wait(bar(kBarODone + s), (k - 1) & 1);
                ++kcnt[s];
                ++n;
            }
        }
        // ---- epilogue: O / l -> shared staging -> coalesced stores of the slot's partial state ----
        mbar_wait(bar(kBarAllDone), 0);  // every MMA done: the ring is free for staging
        if (warp == 4 && lane == 0) TL(100);
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            if (sp.tile[s] < 0) continue;
            const int tile_row0 = row_base + sp.tile[s] * kTileM;
            const int r = tile_row0 + rl;
            const bool row_ok = r < rows_valid;
            if (kcnt[s] == 0) {  // this rank had no unit for the slot (shared tile, single key tile)
                if (h == 0 && row_ok) plse[r] = -INFINITY;
                continue;
            }
            const bool warp_active = (tile_row0 + w * 32) < rows_valid;
            xm[h * kTileM + rl] = l_run[s];
            named_bar_sync(1, 256);
            const float l_tot = l_run[s] + xm[(h ^ 1) * kTileM + rl];
            const uint32_t stage = smem + kOffRing + (uint32_t)s * (2 * kKvTileBytes);
            if (warp_active) {
                tc_fence_after();
                const float inv = l_tot > 0.f ? 1.f / l_tot : 0.f;  // l = 0: every key of the chunk masked
                const uint32_t srow = stage + (uint32_t)rl * 512u;
                const uint32_t o_addr = tmem + s * kD + h * 64 + lane_addr;
#pragma unroll
                for (int c0 = 0; c0 < 64; c0 += 32) {
                    uint32_t o[32];
                    D2SD_TMEM_LD32(o_addr + c0, o, 0);
                    tmem_wait_ld();
#pragma unroll
                    for (int c = 0; c < 32; c += 4) {
                        const uint32_t chunk = (uint32_t)((h * 64 + c0 + c) >> 2);
                        const uint32_t phys = (chunk & ~7u) | ((chunk ^ (uint32_t)rl) & 7u);
                        asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(srow + phys * 16u),
                                     "f"(__uint_as_float(o[c]) * inv), "f"(__uint_as_float(o[c + 1]) * inv),
                                     "f"(__uint_as_float(o[c + 2]) * inv), "f"(__uint_as_float(o[c + 3]) * inv)
                                     : "memory");
                    }
                }
                if (h == 0 && row_ok) plse[r] = l_tot > 0.f ? m_run[s] * pl.sm_scale + logf(l_tot) : -INFINITY;
            }
            named_bar_sync(1, 256);
            // warp q of the eight stores rows q*16 .. q*16+15, one 512-byte row per instruction
            const int nrows = min(kTileM, rows_valid - tile_row0);
            const int q = warp - 4;
            const uint32_t chunk = (uint32_t)lane;
#pragma unroll 4
            for (int i = 0; i < 16; ++i) {
                const int row = q * 16 + i;
                if (row < nrows) {
                    const uint32_t phys = (chunk & ~7u) | ((chunk ^ (uint32_t)row) & 7u);
                    float4 v;
                    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                                 : "r"(stage + (uint32_t)row * 512u + phys * 16u));
                    *reinterpret_cast<float4*>(po + (size_t)(tile_row0 + row) * kD + lane * 4) = v;
                }
            }
        }
        if (warp == 4 && lane == 0) TL(101);

        // ---- publish this CTA's partial states, wait for the group, merge this CTA's share of rows ----
        const unsigned expected = gridDim.x;  // 2 * num_splits CTAs per (b, g, M group)
        unsigned* cnt = a.counters + 2 * (blockIdx.z * gridDim.y + blockIdx.y);  // [0] arrivals, [1] done
        __threadfence();
        named_bar_sync(1, 256);
        if (warp == 4 && lane == 0) {
            asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(cnt) : "memory");
            unsigned seen, spins = 0;
            do {
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(cnt) : "memory");
                if (seen < expected) {
                    __nanosleep(32);
                    if (++spins > (1u << 24)) __trap();  // a scheduling assumption broke: fail, do not hang
                }
            } while (seen < expected);
        }
        named_bar_sync(1, 256);
        if (warp == 4 && lane == 0) TL(102);
        merge_rows(pl, a, dbg_rows, b, g, row_base, rows_g, MT, (int)blockIdx.x * 8 + (warp - 4), (int)gridDim.x * 8,
                   lane);
        named_bar_sync(1, 256);
        if (warp == 4 && lane == 0) {
            if (atomicAdd(cnt + 1, 1u) == expected - 1) {  // last CTA out: everybody is past the wait
                cnt[0] = 0;
                cnt[1] = 0;
            }
            TL(103);
        }
    }

    tc_fence_before();
    __syncthreads();
    if (tid == 0) TL(2);
    if (warp == 2) {
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
    // contiguous KV only (paged KV stays on the mma.sync path), rows of one query tile must be whole
    // tree nodes (128 % G == 0), and the tensor-map extents must fit.
    return pl.page_size == 0 && pl.d == kD && pl.G <= 128 && (128 % pl.G) == 0 &&
           (int64_t)pl.B * pl.T_cap < (1ll << 31) && pl.kv_rows < (1ll << 31);
}

int32_t launch_attn_cascade_tc(const AttnPlan& pl, const AttnArgs& a, int mode, float* dbg_rows, cudaStream_t s) {
    static bool attr_set = false;
    if (!attr_set) {
        D2SD_CHECK_CUDA(cudaFuncSetAttribute(attn_cascade_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)kSmemBytes));
        attr_set = true;
    }
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
        if (pl.kv_rows > 0 && a.k_cache && a.v_cache) {
            const cuuint64_t dims[4] = {64, (cuuint64_t)pl.kv_rows, 2, (cuuint64_t)pl.Hkv};
            if (int32_t st = encode(&tm_k, a.k_cache, 4, dims, strides, box, "k_cache")) return st;
            if (int32_t st = encode(&tm_v, a.v_cache, 4, dims, strides, box, "v_cache")) return st;
        } else {  // no committed prefix at all (max_ctx_len == 0): the maps are never used
            tm_k = tm_tk;
            tm_v = tm_tv;
        }
    }
    dim3 grid(2 * pl.num_splits, pl.Hkv, pl.B * pl.n_mgroups);
    attn_cascade_tc_kernel<<<grid, kThreads, kSmemBytes, s>>>(tm_q, tm_k, tm_v, tm_tk, tm_tv, pl, a, mode, dbg_rows);
    D2SD_CHECK_LAUNCH("attn_cascade_tc_kernel");
    return D2SD_OK;
}

#ifdef D2SD_TIMELINE
extern "C" int32_t d2sd_debug_timeline(long long* host_buf /* [256][128] */) {
    return cudaMemcpyFromSymbol(host_buf, g_timeline, sizeof(long long) * 256 * 128) == cudaSuccess ? 0 : -4;
}
#endif

}  // namespace d2sd
