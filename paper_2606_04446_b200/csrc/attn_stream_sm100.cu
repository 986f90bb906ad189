// Stage (c), fused: cascade tree-verify attention in ONE launch on tcgen05 / TMEM / TMA (sm_100a).
// PAPER.md:52, :124, :154.
//
// Every tree query of every branch and every GQA head of one kv head is a row of one batched query
// matrix (row r = t*G + hh), cut into 128-row M tiles.  The keys of a request are the committed
// prefix followed by the tree-local keys, cut into 128-key tiles: prefix tiles 0..np-1
// (np = ceil(L/128)) and tree tiles np..np+nt-1 (nt = ceil(T/128)); a tree tile is an ordinary key
// tile whose scores additionally pass the node's ancestor-mask bits.
//
// Work decomposition.  One CTA serves (request b, kv head g, M tile, context chunk): ONE query tile and
// a run of key tiles ("units").  The launch is made of 2-CTA clusters: the CTAs of M tiles (2p, 2p+1)
// over the same chunk form a SHARING pair -- rank 0 loads every K tile, rank 1 every V tile, each TMA
// multicast into both CTAs' rings, so a KV tile crosses the L2->SM fabric once per 256 query rows --
// and the chunks of an odd last M tile are paired without sharing.
//
// TMEM (512 columns): O (128 fp32 columns), S_0..S_3 (64 each), P_0..P_3 (32 each, bf16 pairs).
// A 128-key tile is processed as two 64-key SUB-UNITS; sub-unit n uses buffers n & 3.  S and P are
// separate columns, so Q.K^T of sub-unit n+4 is issued as soon as the softmax has READ S_n (it does not
// wait for P.V of sub-unit n), and the softmax never waits for the tensor pipe in steady state:
//
//   S_n[128 x 64] = Q[128 x 128] . K_n^T         tcgen05.mma, A/B from 128B-swizzled SMEM (TMA)
//   P_n           = exp2(c*(S_n - m_ref))        one softmax thread per row (TMEM lane)
//   O[128 x 128] += P_n[128 x 64] . V_n          tcgen05.mma, A = P from TMEM, B = V (MN-major SMEM)
//
// Warp roles (640 threads): warps 0..15 = four softmax teams of four warps, team t owns the sub-units
// n = t (mod 4), thread (w, lane) of a team owns query row w*32 + lane (TMEM lane) and the 64 scores of
// the sub-unit; warp 16 = K producer (+ Q), warp 17 = V producer (also zeroes the V rows behind a
// ragged tile end: they are multiplied by exact zeros and may hold anything, NaN included), warp 18 =
// Q.K^T issuer (one elected thread; owns the TMEM allocation), warp 19 = P.V issuer.  A single softmax warp runs
// at ~0.2 instructions per clock (dependent chains of the maxima, exponentials, packs): four teams keep
// four warps per scheduler busy on four different sub-units, so one team's loads / maxima / packs
// overlap the others' exponentials on the shared MUFU pipe, inside the register file's 64 Ki registers
// (64 scores per thread: 112 registers).
//
// One accumulator, four teams: the row's reference maximum m_ref travels with the sub-unit sequence.
// The owner of sub-unit n reads m_ref(n-1) from shared memory (published by the previous team's warp of
// the same rows, ordered by an mbarrier per (team, warp)), raises it only when the tile maximum exceeds
// it by more than 2^8 (lazy rescale), publishes m_ref(n), and -- only when it raised it -- waits for
// P.V of sub-unit n-1 and rescales its O row in TMEM before it releases P_n.  Each thread keeps its own
// row sum relative to the last reference it has seen; the four sums meet in the epilogue.
//
// Cascade merge in the same launch (log-sum-exp state merge): every CTA writes its
// normalised partial state (O fp32, LSE) to the workspace straight from registers (tcgen05.ld 16x256b
// gives four adjacent lanes 32 contiguous bytes of a row: full-sector stores; it stays in L2),
// publishes it with a release-increment of its group's arrival counter (group = request, kv head,
// M tile), waits until all non-empty chunks of the group have arrived, and merges ITS share of the
// group's rows (coalesced 16-byte loads, all in flight at once).  The counters reset themselves.
// The wait needs the group's CTAs (<= 64) to be co-resident; the plan sizes one-wave grids so that
// they are, multi-wave grids are safe because a group is a run of consecutive blocks of the grid's
// linear order.  A wait that does not end sets an error word in the workspace header instead of
// trapping (d2sd.h).
// The launch is a programmatic dependent launch: the prologue (barriers, TMEM, tensor-map prefetch)
// overlaps the tail of the preceding kernel.  Before griddepcontrol.wait nothing is read for use and nothing is
// written: one warp reads the request's lengths as they stand (possibly stale) only to aim an L2 prefetch hint at
// the chunk's first K / V tiles; every value the kernel computes with is read after the wait.
// Pace: one-thread roles (the two MMA issuers, the producers) and one-shot code (prologue, epilogue) cost
// (instructions) x 5-8 clk, and a barrier test keeps a thread 100-250 clk; they, not the softmax warps, set the
// kernel's pace (profiles/r02_experiments.md, "Per-thread timeline"), so their loops carry their state incrementally
// (no division, no per-tile decode) and probe the barriers of a tile together.
#include "tc_ptx.cuh"

namespace d2sd {
namespace {

constexpr int kRingK = 3, kRingV = 3;  // K tiles / V tiles in flight or in use (2 + 4 measured the same: what counts is the 192 KiB in flight)
constexpr int kThreads = 640;      // 16 softmax warps (4 teams) + 4 control warps
constexpr int kTeams = 4;
constexpr int kSubN = 64;          // keys per sub-unit (one S / P buffer)
constexpr uint32_t kOffQ = 0;
constexpr uint32_t kOffK = kQTileBytes;
constexpr uint32_t kOffV = kOffK + kRingK * kKvTileBytes;
constexpr uint32_t kOffBar = kOffV + kRingV * kKvTileBytes;
constexpr uint32_t kOffX = kOffBar + 512;                 // reference-maximum hand-off: fp32 [4 teams][128 rows]
constexpr uint32_t kOffXL = kOffX;                        // epilogue: the teams' row sums take the same place
constexpr uint32_t kSmemUsed = kOffX + kTeams * kTileM * 4;
constexpr uint32_t kSmemBytes = 232448;                   // the whole 227 KiB: kSmemUsed + alignment slack
constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kTmemS = 128;   // S_0..S_3 behind O (64 fp32 columns each)
constexpr uint32_t kTmemP = 384;   // P_0..P_3 (32 columns of bf16 pairs each)
constexpr float kRescaleThreshold = 8.0f;  // log2 units
constexpr int kPrefetchTiles = 3;           // key tiles per CTA hinted into L2 in the prologue (measured: 1-3 equal, 4 and 6 slower)
constexpr uint32_t kRegsControl = 64, kRegsSoftmax = 104;  // setmaxnreg targets: 512 x 104 + 128 x 64 = 60 Ki registers (the launch allocation)

// barrier slots (8 bytes each) at kOffBar
enum : uint32_t {
    kBarQFull = 0,
    kBarKFull = 1,                       // [kRingK]
    kBarKEmpty = kBarKFull + kRingK,     // [kRingK]
    kBarVFull = kBarKEmpty + kRingK,     // [kRingV]
    kBarVEmpty = kBarVFull + kRingV,     // [kRingV]
    kBarSFull = kBarVEmpty + kRingV,     // [4] Q.K^T of a sub-unit has completed
    kBarSFree = kBarSFull + kTeams,      // [4] the owning team has read S into registers
    kBarPFull = kBarSFree + kTeams,      // [4] the owning team has written P
    kBarPFree = kBarPFull + kTeams,      // [8] P.V of sub-unit n has completed: barrier n & 7 (P buffer reusable, O current)
    kBarRef = kBarPFree + 8,             // [4 teams][4 warps] the team's warp has published its rows' reference maxima
    kBarVFix = kBarRef + 4 * kTeams,     // [2] V rows behind a ragged tile end are zero (<= 2 ragged tiles per CTA)
    kBarAllDone = kBarVFix + 2,
    kNumBars = kBarAllDone + 1,
    kTmemSlot = kNumBars  // uint32 written by tcgen05.alloc
};
static_assert((kNumBars + 1) * 8 <= 512, "barrier area");
static_assert(kSmemUsed + 512 <= kSmemBytes, "shared memory budget");  // the kernel checks the actual alignment slack

// ---- cluster (2-CTA sharing pair) ---------------------------------------------------------------
// tcgen05.commit that arrives on the barrier at the same offset in every CTA of `mask`
__device__ __forceinline__ void tc_commit_mc(uint32_t bar, uint16_t mask) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(bar),
                 "h"(mask)
                 : "memory");
}
__device__ __forceinline__ void tma_load_4d_mc(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int c0, int c1, int c2,
                                               int c3, uint16_t mask, uint64_t hint) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster.L2::cache_hint"
        " [%0], [%1, {%3, %4, %5, %6}], [%2], %7, %8;" ::"r"(dst),
        "l"(reinterpret_cast<uint64_t>(tm)), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "h"(mask), "l"(hint)
        : "memory");
}
__device__ __forceinline__ void tma_load_5d_mc(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int c0, int c1, int c2,
                                               int c3, int c4, uint16_t mask, uint64_t hint) {
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster.L2::cache_hint"
        " [%0], [%1, {%3, %4, %5, %6, %7}], [%2], %8, %9;" ::"r"(dst),
        "l"(reinterpret_cast<uint64_t>(tm)), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "h"(mask), "l"(hint)
        : "memory");
}

// What one CTA does: which M tile / chunk, which key tiles it streams, whom it shares them with.
struct Work {
    int b, g, tile, chunk;
    int share;         // 1: sharing pair (this CTA and its cluster peer stream the same key tiles)
    int rank;          // rank in the cluster (sharing pair: 0 loads K, 1 loads V)
    int row_base;      // first query row (t*G + hh) of the tile
    int rows;          // valid query rows of the tile (0: nothing to do)
    int np, nt;        // prefix / tree key tiles of the request (after the mode bits)
    int j_begin, n_tiles;
    int n_chunks;      // non-empty chunks of the group = CTAs that arrive at the group counter
    int group;         // (b*Hkv + g)*n_mt + tile
    int T, L;
};

struct TileInfo {
    int valid;      // keys of the tile that exist (1..128)
    int row;        // first row of the tile in its tensor map
    bool tree;      // tree tile (ancestor mask applies), else prefix tile
    int tt;         // tree tile index (tree tiles only)
    int j;          // key tile index within the request (prefix tiles first)
};

// partial states are read at L2 (written by other SMs; this SM's L1 may hold the previous launch's lines)
__device__ __forceinline__ float ld_cg_f32(const float* p) {
    float v;
    asm volatile("ld.global.cg.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ uint4 ld_cg_u4(const __nv_bfloat16* p) {
    uint4 v;
    asm volatile("ld.global.cg.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}
// Row sums of the partial states: the workspace's O region is sized for fp32 rows (common.cuh), this kernel's bf16
// rows fill its first half; the sums sit right behind them.
__device__ __forceinline__ float* part_sum(const AttnPlan& pl, const AttnArgs& a) {
    const size_t rows_all = (size_t)pl.B * pl.Hkv * pl.n_mt * pl.grp_rows;
    return reinterpret_cast<float*>(a.part_o16 + rows_all * kD);
}
__device__ __forceinline__ float bf_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf_hi(uint32_t w) { return __uint_as_float(w & 0xFFFF0000u); }

// -------------------------------------------------------------------------------------------------
// Cascade merge of one group's rows (log-sum-exp state merge):
//   LSE = log sum_p e^{LSE_p};  O = sum_p e^{LSE_p - LSE} O_p   over the group's chunk states.
// CTA `chunk` of the group's n_chunks CTAs takes a contiguous range of the tile's rows.  One THREAD takes 8
// columns of one row (16 threads a row, 512 threads = 32 rows a pass): it loads the row's LSE of every state and
// its 16-byte piece of every state's O row (all requested at once: one L2 round trip), forms the weights itself
// (no shuffles) and writes 16 bytes of the output.  The decomposition matters more than the traffic: a warp
// executes a dependent instruction every 5-8 clk, so the merge costs (instructions per thread) x that, and the
// earlier warp-per-two-rows form (shuffled weights, ~600 instructions per thread) took 4.6k-8.6k clk.
// The partial states were written by other SMs and published with a release; the loads follow the group wait's
// acquire fence.
__device__ __forceinline__ void merge_rows(const AttnPlan& pl, const AttnArgs& a, float* dbg_rows, const Work& wk,
                                           int r0, int r1, int warp, int lane) {
    const int G = pl.G;
    const int nc = wk.n_chunks;  // <= 64 states
    const size_t grp0 = (size_t)wk.group * pl.grp_rows;
    const int nrows = r1 - r0;  // <= 128
    const int g_shift = __ffs(G) - 1;  // G divides 128 (attn_stream_supported): a power of two
    constexpr int kSB = 8;      // states per batch
    for (int idx = warp * 32 + lane; idx < nrows * 16; idx += 512) {
        const int r = r0 + (idx >> 4), cg = idx & 15;
        const float* lp = a.part_lse + grp0 + r;
        const __nv_bfloat16* op = a.part_o16 + (grp0 + r) * kD + cg * 8;
        const float* sp = part_sum(pl, a) + grp0 + r;
        float mv[kSB], sv[kSB];
        uint4 v[kSB];
#pragma unroll
        for (int i = 0; i < kSB; ++i) {
            mv[i] = i < nc ? ld_cg_f32(lp + (size_t)i * kTileM) : 0.f;
            sv[i] = i < nc ? ld_cg_f32(sp + (size_t)i * kTileM) : 0.f;
        }
#pragma unroll
        for (int i = 0; i < kSB; ++i)
            if (i < nc) v[i] = ld_cg_u4(op + (size_t)i * kTileM * kD);
        // O = sum_i 2^(m_i - M) O_i / sum_i 2^(m_i - M) l_i over the states that saw a key (l_i > 0)
        float m = -INFINITY;
#pragma unroll
        for (int i = 0; i < kSB; ++i) m = sv[i] > 0.f ? fmaxf(m, mv[i]) : m;
#pragma unroll 1
        for (int i = kSB; i < nc; ++i)  // more than eight chunks
            if (ld_cg_f32(sp + (size_t)i * kTileM) > 0.f) m = fmaxf(m, ld_cg_f32(lp + (size_t)i * kTileM));
        float ws = 0.f, wv[kSB];
#pragma unroll
        for (int i = 0; i < kSB; ++i) {
            wv[i] = sv[i] > 0.f ? ex2(mv[i] - m) : 0.f;
            ws += wv[i] * sv[i];
        }
#pragma unroll 1
        for (int i = kSB; i < nc; ++i) {
            const float l = ld_cg_f32(sp + (size_t)i * kTileM);
            if (l > 0.f) ws += ex2(ld_cg_f32(lp + (size_t)i * kTileM) - m) * l;
        }
        const float inv = ws > 0.f ? __fdividef(1.f, ws) : 0.f;  // no key at all (L = 0, prefix-only mode): O = 0, LSE = -inf
        const float lse = ws > 0.f ? (m + __log2f(ws)) * (1.f / kLog2e) : -INFINITY;
        float acc[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) acc[c] = 0.f;
#pragma unroll
        for (int i = 0; i < kSB; ++i)
            if (i < nc) {  // states without any key hold zeros (their CTA wrote them)
                const float w1 = wv[i] * inv;
                acc[0] += w1 * bf_lo(v[i].x); acc[1] += w1 * bf_hi(v[i].x);
                acc[2] += w1 * bf_lo(v[i].y); acc[3] += w1 * bf_hi(v[i].y);
                acc[4] += w1 * bf_lo(v[i].z); acc[5] += w1 * bf_hi(v[i].z);
                acc[6] += w1 * bf_lo(v[i].w); acc[7] += w1 * bf_hi(v[i].w);
            }
#pragma unroll 1
        for (int i = kSB; i < nc; ++i) {
            const float l = ld_cg_f32(sp + (size_t)i * kTileM);
            const float w1 = l > 0.f ? ex2(ld_cg_f32(lp + (size_t)i * kTileM) - m) * inv : 0.f;
            const uint4 x = ld_cg_u4(op + (size_t)i * kTileM * kD);
            acc[0] += w1 * bf_lo(x.x); acc[1] += w1 * bf_hi(x.x);
            acc[2] += w1 * bf_lo(x.y); acc[3] += w1 * bf_hi(x.y);
            acc[4] += w1 * bf_lo(x.z); acc[5] += w1 * bf_hi(x.z);
            acc[6] += w1 * bf_lo(x.w); acc[7] += w1 * bf_hi(x.w);
        }
        const int ra = wk.row_base + r, t = ra >> g_shift;  // query row of the tile -> out / lse row [b][t][h]
        const size_t orow = ((size_t)wk.b * pl.T_cap + t) * pl.Hq + wk.g * G + (ra - (t << g_shift));
        if (dbg_rows) {  // fp32 state for tests
            float* d0 = dbg_rows + orow * (kD + 1) + cg * 8;
#pragma unroll
            for (int c = 0; c < 8; ++c) d0[c] = acc[c];
            if (cg == 0) dbg_rows[orow * (kD + 1) + kD] = lse;
            continue;
        }
        uint4 pk;
        pk.x = pack2_bf16(acc[0], acc[1]);
        pk.y = pack2_bf16(acc[2], acc[3]);
        pk.z = pack2_bf16(acc[4], acc[5]);
        pk.w = pack2_bf16(acc[6], acc[7]);
        *reinterpret_cast<uint4*>(a.out + orow * kD + cg * 8) = pk;
        if (cg == 0 && a.lse) a.lse[orow] = lse;
    }
}

// mode bits: 1 = include the prefix tiles, 2 = include the tree tiles (3 = the whole cascade).
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads, 1)
attn_stream_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
                   const __grid_constant__ CUtensorMap tm_v, const __grid_constant__ CUtensorMap tm_tk,
                   const __grid_constant__ CUtensorMap tm_tv, AttnPlan pl, AttnArgs a, int mode, float* dbg_rows) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    const uint32_t smem_raw_u32 = (uint32_t)__cvta_generic_to_shared(smem_raw);
    const uint32_t smem = (smem_raw_u32 + 1023u) & ~1023u;  // 128B swizzle atoms need 1024 B alignment
    if (smem - smem_raw_u32 + kSmemUsed > kSmemBytes) __trap();
    unsigned char* smem_gen = smem_raw + (smem - smem_raw_u32);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t bar0 = smem + kOffBar;
    auto bar = [&](uint32_t i) { return bar0 + 8u * i; };
    volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem_gen + kOffBar + 8u * kTmemSlot);

    // static part of the work decode (no global memory): which cluster kind this CTA belongs to
    const int n_pairs = pl.n_mt >> 1;
    const int pair_ctas = n_pairs * 2 * pl.chunks_a;
    const bool pair = (int)blockIdx.x < pair_ctas;  // cluster of M tiles (2p, 2p+1) over one chunk

    // ---- prologue that touches no global memory (overlaps the preceding kernel's tail under PDL) ----
    if (warp == 16 && lane == 0) {
        mbar_init(bar(kBarQFull), 1);
        for (int i = 0; i < kRingK; ++i) {
            mbar_init(bar(kBarKFull + i), 1);
            mbar_init(bar(kBarKEmpty + i), pair ? 2 : 1);  // released by both CTAs of a pair cluster
        }
        for (int i = 0; i < kRingV; ++i) {
            mbar_init(bar(kBarVFull + i), 1);
            mbar_init(bar(kBarVEmpty + i), pair ? 2 : 1);
        }
        for (int t = 0; t < kTeams; ++t) {
            mbar_init(bar(kBarSFull + t), 1);
            mbar_init(bar(kBarSFree + t), 4);  // one elected arrival per warp of the owning team
            mbar_init(bar(kBarPFull + t), 4);
            mbar_init(bar(kBarPFree + t), 1);
            mbar_init(bar(kBarPFree + 4 + t), 1);
            for (int w = 0; w < 4; ++w) mbar_init(bar(kBarRef + 4 * t + w), 1);
        }
        mbar_init(bar(kBarVFix + 0), 1);
        mbar_init(bar(kBarVFix + 1), 1);
        mbar_init(bar(kBarAllDone), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        tma_prefetch_desc(&tm_q);
        tma_prefetch_desc(&tm_k);
        tma_prefetch_desc(&tm_v);
        tma_prefetch_desc(&tm_tk);
        tma_prefetch_desc(&tm_tv);
    }
    if (warp == 18) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(bar(kTmemSlot)),
                     "r"(kTmemCols)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    // the peer's barriers must be initialised before anything remote reaches them: arrive now, wait after the
    // work decode (the peer has long arrived by then)
    if (pair) asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    pdl_launch_dependents();  // the next kernel may begin its own prologue as SMs free up

    // ---- this CTA's work: the part that needs no global memory ----
    Work wk;
    int n_static;
    bool pad = false;
    {
        wk.g = blockIdx.y;
        wk.b = blockIdx.z;
        int x = blockIdx.x;
        if (pair) {
            const int p = x / (2 * pl.chunks_a), r = x - p * 2 * pl.chunks_a;
            wk.chunk = r >> 1; wk.rank = r & 1; wk.tile = 2 * p + wk.rank; n_static = pl.chunks_a;
        } else {
            x -= pair_ctas;
            wk.chunk = x; wk.rank = x & 1; wk.tile = pl.n_mt - 1; n_static = pl.chunks_b;
            pad = x >= pl.chunks_b;  // the odd tile's chunk count rounded up to whole clusters
        }
        wk.row_base = wk.tile * kTileM;
        wk.group = (wk.b * pl.Hkv + wk.g) * pl.n_mt + wk.tile;
    }
    // the chunk's key tiles from the request's lengths
    auto cut = [&](int T, int L) {
        wk.T = T;
        wk.L = L;
        wk.np = (mode & 1) ? (L + kTileN - 1) / kTileN : 0;
        wk.nt = (mode & 2) ? (T + kTileN - 1) / kTileN : 0;
        const int nk = wk.np + wk.nt;
        const int tps = max(max(1, pl.tps_min), (nk + n_static - 1) / n_static);
        wk.n_chunks = max(1, (nk + tps - 1) / tps);  // chunk 0 always takes part (nk = 0: state (0, -inf))
        wk.j_begin = wk.chunk * tps;
        wk.n_tiles = max(0, min(nk, wk.j_begin + tps) - wk.j_begin);
    };
    // L2 prefetch of the chunk's first ring of K / V tiles, issued BEFORE the grid dependency resolves, from lengths
    // that may be stale (the preceding kernel may be the one that writes them): a prefetch is a hint, a wrong guess
    // fetches other lines of the same tensors.  The first tiles' DRAM latency (2.2k-2.9k clk, and the whole
    // launch asks for its first 9 MB at once) then runs under the dependency wait and the work decode.
    if (warp == 17 && pl.page_size == 0 && !pad) {
        int T0, L0, kv0 = 0;
        asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(T0) : "l"(a.tree_len + wk.b) : "memory");
        asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(L0) : "l"(a.ctx_len + wk.b) : "memory");
        if (a.kv_indptr) asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(kv0) : "l"(a.kv_indptr + wk.b) : "memory");
        if (T0 >= 0 && T0 <= pl.T_cap && L0 >= 0 && L0 <= pl.max_ctx_len) {
            cut(T0, L0);
            const int jj = lane >> 1, j = wk.j_begin + jj;
            const bool v_side = lane & 1;
            // a sharing pair: rank 0 will load K, rank 1 V (short trees do not share: then both sides are needed
            // anyway and the other CTA's hint is merely redundant)
            const bool mine = !pair || wk.rank == (v_side ? 1 : 0);
            if (lane < 2 * kPrefetchTiles && jj < wk.n_tiles && j < wk.np && mine)
                tma_prefetch_4d(v_side ? &tm_v : &tm_k, 0, kv0 + j * kTileN, 0, wk.g);
        }
    }
    pdl_wait();  // everything before this kernel in the stream is complete and visible
    {
        const int G = pl.G;
        cut(a.tree_len[wk.b], a.ctx_len[wk.b]);
        const int rows_valid = wk.T * G;
        wk.rows = pad ? 0 : max(0, min(kTileM, rows_valid - wk.row_base));
        // a pair shares its key tiles when both M tiles hold rows (a short tree leaves the odd tile empty)
        wk.share = pair && rows_valid > (wk.tile | 1) * kTileM;
    }
    // M tiles past the tree's rows, and chunks past the request's key tiles, leave at once:
    // nobody waits for them (n_chunks counts the non-empty chunks only)
    const bool idle = wk.rows == 0 || wk.chunk >= wk.n_chunks;
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
    if (pair) asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
    const uint16_t mc_mask = wk.share ? 3 : (uint16_t)(1u << (blockIdx.x & 1));

    // the control warpgroup hands registers to the two softmax warpgroups (one instruction per warpgroup)
    if (warp >= 16) {
      asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsControl));
      if (idle) {
        // fall through to the TMEM release
      } else if (warp == 16 || warp == 17) {
        // ===== K producer (warp 8, also loads Q) and V producer (warp 9): one ring of three tiles each.
        // Contiguous KV: lane 0 issues one 32 KiB box per tile.  Paged KV (page = 16 keys): a 128-key
        // tile is 8 pages; lane 2p+hi issues the 2 KiB box (page p, d half hi), so a tile is 16 loads in
        // flight at once; only the ceil(valid/16) pages that exist are loaded (the MMAs never read past
        // ceil16(valid) keys); the page ids of the next tile are fetched one tile ahead.
        // Sharing pair: both CTAs wait for their slot (released by BOTH CTAs' MMAs) and arm their own full
        // barrier; rank 0 issues every K load, rank 1 every V load, multicast into both CTAs' rings.
        // The V producer also zeroes the V rows behind a ragged tile end in its own CTA's copy: the P.V MMA
        // runs over ceil16(valid) keys, rows valid..ceil16(valid)-1 belong to nobody (next request, tree
        // padding), are multiplied by P = 0 exactly and must not hold NaN/Inf.  A row is 2 x 128 B (d
        // halves); the 128B swizzle permutes 16-byte chunks inside a row's 128 B only. =====
        const bool is_v = warp == 17;
        const bool paged = pl.page_size > 0;
        const bool issuer = !wk.share || wk.rank == (is_v ? 1 : 0);
        const int ring = is_v ? kRingV : kRingK;
        const uint32_t ring_off = is_v ? kOffV : kOffK;
        const uint32_t bar_full = is_v ? kBarVFull : kBarKFull, bar_empty = is_v ? kBarVEmpty : kBarKEmpty;
        auto page_of = [&](int jj) {
            int pg = 0;
            if (paged && issuer && jj < wk.n_tiles) {
                const TileInfo t2 = tile_info(jj);
                const int p = lane >> 1;
                if (!t2.tree && lane < 16 && p * 16 < t2.valid) pg = __ldg(a.kv_indices + kv_row0 + t2.j * 8 + p);
            }
            return pg;
        };
        // Q: one box = the 128-row query tile of this kv head; issued by the V producer (its first tile is needed a
        // softmax later than the first K tile, and an issue keeps the thread ~400 clk)
        if (is_v && lane == 0) {
            const int t0 = wk.b * pl.T_cap + wk.row_base / pl.G;
            mbar_expect_tx(bar(kBarQFull), kQTileBytes);
            tma_load_5d(smem + kOffQ, &tm_q, bar(kBarQFull), 0, 0, t0, 0, wk.g, kEvictLast);
        }
        int page_cur = page_of(0);
        int n_ragged = 0;
        int i = 0;            // ring slot of tile jj
        uint32_t round = 0;   // parity of jj / ring
        for (int jj = 0; jj < wk.n_tiles; ++jj) {
            const TileInfo ti = tile_info(jj);
            const int page_next = page_of(jj + 1);
            const uint32_t dst = smem + ring_off + i * kKvTileBytes;
            const uint32_t fb = bar(bar_full + i);
            const bool by_page = paged && !ti.tree;
            const int n_pages = (ti.valid + 15) >> 4;
            if (lane == 0) {
                if (jj >= ring) mbar_wait(bar(bar_empty + i), round ^ 1u);  // (the first fill finds the ring empty)
                mbar_expect_tx(fb, by_page ? (uint32_t)n_pages * 4096u : kKvTileBytes);
            }
            __syncwarp();
            if (issuer) {
                if (by_page) {
                    if (lane < 2 * n_pages) {
                        const uint32_t d2 = dst + (uint32_t)(lane & 1) * (kKvTileBytes / 2) + (uint32_t)(lane >> 1) * 2048u;
                        if (wk.share)
                            tma_load_5d_mc(d2, is_v ? &tm_v : &tm_k, fb, 0, 0, lane & 1, wk.g, page_cur, mc_mask, kEvictNormal);
                        else
                            tma_load_5d(d2, is_v ? &tm_v : &tm_k, fb, 0, 0, lane & 1, wk.g, page_cur, kEvictNormal);
                    }
                } else if (lane == 0) {
                    const CUtensorMap* tm = ti.tree ? (is_v ? &tm_tv : &tm_tk) : (is_v ? &tm_v : &tm_k);
                    const uint64_t hint = ti.tree ? kEvictLast : kEvictNormal;
                    if (wk.share) tma_load_4d_mc(dst, tm, fb, 0, ti.row, 0, wk.g, mc_mask, hint);
                    else tma_load_4d(dst, tm, fb, 0, ti.row, 0, wk.g, hint);
                }
            }
            if (is_v && (ti.valid & 15) != 0) {
                mbar_wait_warp(lane, fb, round);  // this fill has landed (every lane observes it)
                const int n_rows = ((ti.valid + 15) & ~15) - ti.valid;
                for (int e = lane; e < n_rows * 16; e += 32) {  // 16 x 16 B per row
                    const int row = ti.valid + (e >> 4), c16 = e & 15;
                    const uint32_t addr = dst + (uint32_t)(c16 >> 3) * (kKvTileBytes / 2) + (uint32_t)row * 128u +
                                          (uint32_t)(c16 & 7) * 16u;
                    asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(addr), "r"(0u) : "memory");
                }
                fence_async_smem();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(kBarVFix + n_ragged));
                ++n_ragged;
            }
            __syncwarp();
            page_cur = page_next;
            if (++i == ring) { i = 0; round ^= 1u; }
        }
      } else if (warp == 18 || warp == 19) {
        // ===== MMA issuers (warp 18: Q.K^T stream, warp 19: P.V stream): one elected thread each walks the sub-unit sequence (two 64-key halves per key tile, a
        // ragged tile's second half only if it holds keys).  Q.K^T of sub-unit n+4 goes out as soon as the
        // owning team has read S_n (S and P are separate TMEM columns), P.V of sub-unit n as its P arrives;
        // the tensor pipe executes them in this order.  A ring slot is released by the commit behind its
        // last reader (to both CTAs of a sharing pair). =====
        if (elect_one()) {
            const uint64_t qd = smem_desc(smem + kOffQ, 16, 1024);
            const uint32_t od = tmem;
            const int N = wk.n_tiles;
            auto release = [&](uint32_t b) {
                if (wk.share) tc_commit_mc(b, 3);
                else { tc_commit(b); if (pair) tc_commit(b); }  // a pair cluster's barriers count two releases
            };
            // Every key tile of the chunk is whole (128 keys = two sub-units) except the request's last prefix tile
            // and its last tree tile.  The issuer loops are the pace-setters of the kernel (one thread, dependent
            // instructions): no division, no per-tile decode, and the waits of a tile are probed together so that
            // their latencies (~100-200 clk each even when the phase is long complete) overlap.
            const int jr0 = wk.np - 1 - wk.j_begin, jr1 = wk.np + wk.nt - 1 - wk.j_begin;
            const int v0 = wk.L - (wk.np - 1) * kTileN, v1 = wk.T - (wk.nt - 1) * kTileN;
            auto valid_of = [&](int jj) { return jj == jr0 ? v0 : (jj == jr1 ? v1 : kTileN); };
            if (warp == 18) {
                // Q.K^T stream: sub-unit n goes out as soon as its S buffer has been read (sub-unit n-4) and its K
                // tile has landed
                mbar_wait(bar(kBarQFull), 0);  // (also with N = 0: the CTA must not leave with the load in flight)
                auto issue_half = [&](uint32_t t, uint32_t ki, uint32_t hf, int keys) {
                    const int n_cols = (keys + 15) & ~15;  // MMA N (multiple of 16)
                    const uint64_t kd = smem_desc(smem + kOffK + ki * kKvTileBytes + hf * (kSubN * 128u), 16, 1024);
                    const uint32_t id_qk = idesc(kTileM, (uint32_t)n_cols, 0);
                    const uint32_t sd = tmem + kTmemS + t * kSubN;
                    tc_fence_after();
#pragma unroll
                    for (int kk = 0; kk < kD / 16; ++kk) {
                        const uint64_t off = (uint64_t)(((kk >> 2) * (kQTileBytes / 2) + (kk & 3) * 32) >> 4);
                        umma_ss(sd, qd + off, kd + off, id_qk, kk > 0);
                    }
                    tc_commit(bar(kBarSFull + t));
                };
                uint32_t n = 0, ki = 0, kph = 0;
                for (int jj = 0; jj < N; ++jj) {
                    const int valid = valid_of(jj);
                    const bool two = valid > kSubN;
                    const uint32_t t0 = n & 3, t1 = (n + 1) & 3;
                    // (a probe that is not needed asks the Q barrier for its long-complete phase 0)
                    const bool need0 = n >= kTeams, need1 = two && n + 1 >= kTeams;
                    uint32_t ok_k, ok_0, ok_1;
                    mbar_probe3(bar(kBarKFull + ki), kph, need0 ? bar(kBarSFree + t0) : bar(kBarQFull),
                                need0 ? (((n >> 2) & 1) ^ 1) : 0u, need1 ? bar(kBarSFree + t1) : bar(kBarQFull),
                                need1 ? ((((n + 1) >> 2) & 1) ^ 1) : 0u, ok_k, ok_0, ok_1);
                    if (!ok_0) mbar_wait(bar(kBarSFree + t0), ((n >> 2) & 1) ^ 1);
                    if (!ok_k) mbar_wait(bar(kBarKFull + ki), kph);
                    issue_half(t0, ki, 0, min(valid, kSubN));
                    if (two) {
                        if (!ok_1) mbar_wait(bar(kBarSFree + t1), (((n + 1) >> 2) & 1) ^ 1);
                        issue_half(t1, ki, 1, valid - kSubN);
                    }
                    release(bar(kBarKEmpty + ki));  // K is free once the tile's last Q.K^T has completed
                    n += two ? 2u : 1u;
                    if (++ki == (uint32_t)kRingK) { ki = 0; kph ^= 1u; }
                }
            } else {
                // P.V stream: sub-unit n goes out as its P arrives; the last commit covers every P.V, and every
                // Q.K^T has completed before its scores were read
                auto issue_half = [&](uint32_t n, uint32_t vi, uint32_t hf, int keys) {
                    const uint32_t t = n & 3;
                    const int ksteps = ((keys + 15) & ~15) >> 4;  // K extent of this P.V in 16-key steps
                    const uint64_t vd = smem_desc(smem + kOffV + vi * kKvTileBytes, kKvTileBytes / 2, 1024);
                    const uint32_t pd = tmem + kTmemP + t * (kSubN / 2);
                    tc_fence_after();
#pragma unroll
                    for (int ks = 0; ks < kSubN / 16; ++ks)
                        if (ks < ksteps)
                            umma_ts(od, pd + ks * 8, vd + (uint64_t)((hf * (kSubN / 16) + ks) * (2048 >> 4)), kIdescPV, (n > 0) | ks);
                    tc_commit(bar(kBarPFree + (n & 7)));
                };
                uint32_t n = 0, vi = 0, vph = 0, n_ragged = 0;
                for (int jj = 0; jj < N; ++jj) {
                    const int valid = valid_of(jj);
                    const bool two = valid > kSubN;
                    uint32_t ok_v, ok_p, ok_x;
                    mbar_probe3(bar(kBarVFull + vi), vph, bar(kBarPFull + (n & 3)), (n >> 2) & 1, bar(kBarQFull), 0u, ok_v,
                                ok_p, ok_x);
                    if (!ok_v) mbar_wait(bar(kBarVFull + vi), vph);
                    if (valid & 15) mbar_wait(bar(kBarVFix + n_ragged++), 0);
                    if (!ok_p) mbar_wait(bar(kBarPFull + (n & 3)), (n >> 2) & 1);
                    issue_half(n, vi, 0, min(valid, kSubN));
                    if (two) {
                        mbar_wait(bar(kBarPFull + ((n + 1) & 3)), ((n + 1) >> 2) & 1);
                        issue_half(n + 1, vi, 1, valid - kSubN);
                    }
                    release(bar(kBarVEmpty + vi));  // V is free once the tile's last P.V has completed
                    n += two ? 2u : 1u;
                    if (++vi == (uint32_t)kRingV) { vi = 0; vph ^= 1u; }
                }
                tc_commit(bar(kBarAllDone));
            }
        }
      }
      // The pair's last barrier, arrival half: this warp has issued everything it will ever send to the peer (multicast
      // loads, multicast commits).  The wait half sits at the kernel's end, an epilogue later, and costs nothing there.
      __syncwarp();
      if (pair) asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    } else {
      asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegsSoftmax));
      if (idle) {
        if (pair) asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
      } else {
        // ===== softmax: team t (warps 4t..4t+3) owns the sub-units n = t (mod 4); thread (w, lane) owns query
        // row w*32 + lane (TMEM lane) and the sub-unit's 64 scores.  Four warps per scheduler work on four
        // different sub-units: while one is in its exponentials the others load, take maxima, pack, store. =====
        const int t = warp >> 2;       // team
        const int w = warp & 3;
        const int rl = w * 32 + lane;  // row within the tile
        const uint32_t lane_addr = (uint32_t)(w * 32) << 16;
        const float c2 = pl.sm_scale * kLog2e;
        const float thr = kRescaleThreshold / c2;  // in raw score units
        float* xm = reinterpret_cast<float*>(smem_gen + kOffX);  // [team][row]: reference maximum after the team's last sub-unit
        const bool warp_active = w * 32 < wk.rows;
        const int N = wk.n_tiles;
        float m_mine = -INFINITY;  // the reference this thread's row sum is relative to
        float l_mine = 0.f;
        const int t_node = min((wk.row_base + rl) / pl.G, wk.T - 1);
        const uint32_t* mrow = a.mask + ((size_t)wk.b * pl.T_cap + t_node) * pl.W;
        const uint32_t sbuf = tmem + kTmemS + t * kSubN + lane_addr;
        const uint32_t pbuf = tmem + kTmemP + t * (kSubN / 2) + lane_addr;
        const int tp = (t + kTeams - 1) & 3;  // the team that owns sub-unit n-1
        // The sub-unit sequence without a per-tile walk: every key tile of the chunk is whole (two sub-units) except
        // the request's last prefix tile (chunk-local index jr0, v0 keys) and its last tree tile (jr1, v1 keys; the
        // last tile of the chunk if it is there at all); a ragged tile of <= 64 keys is a single sub-unit.
        const int jr0 = wk.np - 1 - wk.j_begin, jr1 = wk.np + wk.nt - 1 - wk.j_begin;
        const int v0 = wk.L - (wk.np - 1) * kTileN, v1 = wk.T - (wk.nt - 1) * kTileN;
        const bool in0 = jr0 >= 0 && jr0 < N, in1 = jr1 >= 0 && jr1 < N && jr1 != jr0;
        const int skip0 = in0 && v0 <= kSubN ? 2 * jr0 : 0x3fffffff;  // sub-units past this index sit one half-tile later
        const int n_sub = 2 * N - (in0 && v0 <= kSubN ? 1 : 0) - (in1 && v1 <= kSubN ? 1 : 0);
        const int j_tree = wk.np - wk.j_begin;  // chunk-local index of the first tree tile
        {
            for (int n = t; n < n_sub; n += kTeams) {
                const int n2 = n + (n > skip0 ? 1 : 0);
                const int jj = n2 >> 1, hf = n2 & 1;
                struct { int valid; bool tree; int tt; } ti;
                ti.valid = jj == jr0 ? v0 : (jj == jr1 ? v1 : kTileN);
                ti.tree = jj >= j_tree;
                ti.tt = jj - j_tree;
                const int par = (n >> 2) & 1;
                const int keys = min(kSubN, ti.valid - hf * kSubN);
                const bool last = n == n_sub - 1;
                mbar_wait(bar(kBarSFull + t), par);
                if (!warp_active) {  // a warp without rows only keeps the barrier phases in step
                    if (lane == 0) {
                        mbar_arrive(bar(kBarSFree + t));
                        if (n >= kTeams) mbar_wait(bar(kBarPFree + ((n - 4) & 7)), ((n - 4) >> 3) & 1);
                        mbar_arrive(bar(kBarPFull + t));
                    }
                    __syncwarp();
                    continue;
                }
                uint32_t sv[kSubN];
                tc_fence_after();
                D2SD_TMEM_LD32(sbuf, sv, 0);
                D2SD_TMEM_LD32(sbuf + 32, sv, 32);
                tmem_wait_ld();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(kBarSFree + t));  // Q.K^T of sub-unit n+4 may overwrite S now
                if (ti.tree || keys < kSubN) {
                    // keys past the tile's end, and (tree tiles) keys that are not ancestors-or-self of this
                    // row's node: the sub-unit's 64 mask bits -> -inf
                    uint32_t mw0 = 0xFFFFFFFFu, mw1 = 0xFFFFFFFFu;
                    if (ti.tree) {
                        const int wi = ti.tt * 4 + hf * 2;
                        mw0 = wi < pl.W ? mrow[wi] : 0u;
                        mw1 = wi + 1 < pl.W ? mrow[wi + 1] : 0u;
                    }
#pragma unroll
                    for (int c = 0; c < kSubN; ++c) {
                        const uint32_t bit = ((c < 32 ? mw0 : mw1) >> (c & 31)) & 1u;
                        if (c >= keys || !bit) sv[c] = 0xFF800000u;
                    }
                }
                float mx0 = -INFINITY, mx1 = -INFINITY, mx2 = -INFINITY, mx3 = -INFINITY;
#pragma unroll
                for (int c = 0; c < kSubN; c += 4) {
                    mx0 = fmaxf(mx0, __uint_as_float(sv[c]));
                    mx1 = fmaxf(mx1, __uint_as_float(sv[c + 1]));
                    mx2 = fmaxf(mx2, __uint_as_float(sv[c + 2]));
                    mx3 = fmaxf(mx3, __uint_as_float(sv[c + 3]));
                }
                const float mx = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3));
                // reference hand-off: m_ref(n-1) from the previous team's warp of the same rows, lazy raise,
                // m_ref(n) to the next team
                float m_prev = -INFINITY;
                if (n > 0) {
                    mbar_wait_warp(lane, bar(kBarRef + 4 * tp + w), ((n - 1) >> 2) & 1);
                    m_prev = xm[tp * kTileM + rl];
                }
                const bool need = n > 0 && mx > m_prev + thr;
                const float m_new = n == 0 ? mx : (need ? mx : m_prev);
                if (!last) {
                    xm[t * kTileM + rl] = m_new;
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar(kBarRef + 4 * t + w));
                }
                if (m_new != m_mine) {  // this thread's own row sum follows the reference
                    l_mine *= m_mine == -INFINITY ? 0.f : ex2((m_mine - m_new) * c2);
                    m_mine = m_new;
                }
                if (__any_sync(0xffffffffu, need)) {
                    // O holds sub-units < n relative to m_prev: wait for P.V of sub-unit n-1, rescale this row.
                    // P.V of sub-unit n cannot start before this thread releases P_n below.
                    // A parity wait is only sound when the barrier's preceding phase is known to be complete and its
                    // next one cannot be: P.V completions are spread over eight barriers (sub-unit n -> barrier n & 7,
                    // a phase every eight sub-units).  For barrier (n-1) & 7: this thread's own P guard at sub-unit n-4
                    // has seen P.V of n-8 complete, hence n-9 (the P.V stream is in order); P.V of n+7 needs P_n.
                    mbar_wait_warp(lane, bar(kBarPFree + ((n - 1) & 7)), ((n - 1) >> 3) & 1);
                    tc_fence_after();
                    const float alpha = need ? (m_prev == -INFINITY ? 0.f : ex2((m_prev - m_new) * c2)) : 1.f;
#pragma unroll 1
                    for (int c0 = 0; c0 < kD; c0 += 16) {
                        uint32_t o[16];
                        asm volatile(
                            "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                            : "=r"(o[0]), "=r"(o[1]), "=r"(o[2]), "=r"(o[3]), "=r"(o[4]), "=r"(o[5]), "=r"(o[6]), "=r"(o[7]),
                              "=r"(o[8]), "=r"(o[9]), "=r"(o[10]), "=r"(o[11]), "=r"(o[12]), "=r"(o[13]), "=r"(o[14]), "=r"(o[15])
                            : "r"(tmem + lane_addr + c0));
                        tmem_wait_ld();
#pragma unroll
                        for (int c = 0; c < 16; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * alpha);
                        D2SD_TMEM_ST16(tmem + lane_addr + c0, o);
                    }
                    tmem_wait_st();
                    tc_fence_before();
                }
                // the P buffer is free once P.V of sub-unit n-4 has completed (this team sees barriers t and t+4 in
                // alternation, each phase after phase)
                if (n >= kTeams) mbar_wait_warp(lane, bar(kBarPFree + ((n - 4) & 7)), ((n - 4) >> 3) & 1);
                // a row with every key so far masked has m_ref = -inf: exp2(-inf - 0) = 0, not NaN
                const float ms = m_new == -INFINITY ? 0.f : m_new * c2;
                float sum0 = 0.f, sum1 = 0.f;
                // P[128 x 64] bf16 = 32 TMEM columns, written in two 32-key pieces (the exponentials replace the
                // scores in place: 64 + 16 live registers)
#pragma unroll
                for (int q = 0; q < 2; ++q) {
#pragma unroll
                    for (int c = 0; c < 32; ++c)
                        sv[q * 32 + c] = __float_as_uint(ex2_ordered(__uint_as_float(sv[q * 32 + c]) * c2 - ms));
                    uint32_t p[16];
                    float t0 = 0.f, t1 = 0.f, t2 = 0.f, t3 = 0.f;
#pragma unroll
                    for (int c = 0; c < 16; c += 2) {
                        const float e0 = __uint_as_float(sv[q * 32 + 2 * c]), e1 = __uint_as_float(sv[q * 32 + 2 * c + 1]);
                        const float e2 = __uint_as_float(sv[q * 32 + 2 * c + 2]), e3 = __uint_as_float(sv[q * 32 + 2 * c + 3]);
                        t0 += e0; t1 += e1; t2 += e2; t3 += e3;
                        p[c] = pack2_bf16(e0, e1);
                        p[c + 1] = pack2_bf16(e2, e3);
                    }
                    sum0 += t0 + t1;
                    sum1 += t2 + t3;
                    D2SD_TMEM_ST16(pbuf + q * 16, p);
                }
                l_mine += sum0 + sum1;
                tmem_wait_st();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(kBarPFull + t));
            }
        }
        // ---- epilogue: the four teams' row sums meet at the final reference; the normalised state leaves the
        // CTA straight from registers through a per-warp transpose in shared memory (the rings are free):
        // thread (team t, w, lane) holds columns 32t..32t+31 of row w*32+lane, the warp writes them as whole
        // 32-byte sectors.  A group with a single chunk writes its rows to `out` directly: no exchange. ----
        const int t_last = (n_sub - 1) & 3;
        mbar_wait_warp(lane, bar(kBarAllDone), 0);  // every MMA done: O is final, the rings are free
        if (pair) asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");  // (see the control warps)
        const bool direct = wk.n_chunks == 1;
        const bool row_ok = rl < wk.rows;
        const size_t prow0 = (size_t)wk.group * pl.grp_rows + (size_t)wk.chunk * kTileM;
        float* xl = reinterpret_cast<float*>(smem_gen + kOffXL);  // (scratch word of the group wait below)
        // per-warp staging: [32 rows][128 B] of fp32 (direct output) or [32 rows][64 B] of bf16 pairs (partial
        // state), 16-byte chunks XOR-swizzled by the row
        const uint32_t region = smem + kOffK + (uint32_t)warp * 4096u;
        // A partial state leaves UNNORMALISED, relative to the row's final reference (which O in TMEM already is): its
        // stores go out first and their way to L2 runs under the row-sum exchange below; the merge divides once.
        if (!direct && warp_active) {
            uint32_t ov[32];
            tc_fence_after();
            if (n_sub > 0) {
                D2SD_TMEM_LD32(tmem + lane_addr + t * 32, ov, 0);
                tmem_wait_ld();
            }
#pragma unroll
            for (int c = 0; c < 32; c += 8) {  // 8 columns = one 16-byte chunk of bf16
                const uint32_t chunk = (uint32_t)(c >> 3) ^ ((uint32_t)(lane >> 1) & 3u);
                uint32_t pk[4];
#pragma unroll
                for (int e = 0; e < 4; ++e)
                    pk[e] = n_sub > 0 ? pack2_bf16(__uint_as_float(ov[c + 2 * e]), __uint_as_float(ov[c + 2 * e + 1])) : 0u;
                asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(region + (uint32_t)lane * 64u + chunk * 16u),
                             "r"(pk[0]), "r"(pk[1]), "r"(pk[2]), "r"(pk[3])
                             : "memory");
            }
            __syncwarp();
#pragma unroll 1
            for (int it = 0; it < 4; ++it) {
                const int row = it * 8 + (lane >> 2), ck = lane & 3;
                uint4 v;
                asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];"
                             : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                             : "r"(region + (uint32_t)row * 64u + (uint32_t)((ck ^ ((row >> 1) & 3)) * 16)));
                const int r = w * 32 + row;  // row of the tile
                if (r < wk.rows) *reinterpret_cast<uint4*>(a.part_o16 + (prow0 + r) * kD + t * 32 + ck * 8) = v;
            }
        }
        // every team's (reference, row sum) of the row through the free V ring, one barrier: the final reference
        // is the one of the last sub-unit's owner, each sum is brought to it
        float2* xp = reinterpret_cast<float2*>(smem_gen + kOffV);
        xp[t * kTileM + rl] = make_float2(m_mine, l_mine);
        named_bar_sync(9, 512);
        const float m_fin = n_sub > 0 ? xp[t_last * kTileM + rl].x : -INFINITY;
        float l_tot = 0.f;
#pragma unroll
        for (int tt = 0; tt < kTeams; ++tt) {
            const float2 ml = xp[tt * kTileM + rl];
            l_tot += ml.x == -INFINITY ? 0.f : ml.y * (ml.x == m_fin ? 1.f : ex2((ml.x - m_fin) * c2));
        }
        if (!direct) {
            // the row's state scalars: reference in log2 units and row sum (l = 0: every key of the chunk masked, or no
            // key at all: the state carries no weight)
            if (t == 0 && row_ok) {
                a.part_lse[prow0 + rl] = l_tot > 0.f ? m_fin * c2 : 0.f;
                part_sum(pl, a)[prow0 + rl] = l_tot;
            }
        } else if (warp_active) {
            const float inv = l_tot > 0.f ? __fdividef(1.f, l_tot) : 0.f;
            const float lse_v = l_tot > 0.f ? m_fin * pl.sm_scale + __logf(l_tot) : -INFINITY;
            const int G = pl.G;
            uint32_t ov[32];
            tc_fence_after();
            if (n_sub > 0) {
                D2SD_TMEM_LD32(tmem + lane_addr + t * 32, ov, 0);
                tmem_wait_ld();
            }
#pragma unroll
            for (int c = 0; c < 32; ++c) ov[c] = n_sub > 0 ? __float_as_uint(__uint_as_float(ov[c]) * inv) : 0u;
#pragma unroll
            for (int c = 0; c < 32; c += 4) {
                const uint32_t chunk = (uint32_t)(c >> 2) ^ ((uint32_t)lane & 7u);
                asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(region + (uint32_t)lane * 128u + chunk * 16u),
                             "r"(ov[c]), "r"(ov[c + 1]), "r"(ov[c + 2]), "r"(ov[c + 3])
                             : "memory");
            }
            __syncwarp();
#pragma unroll 1
            for (int it = 0; it < 8; ++it) {
                const int row = it * 4 + (lane >> 3), ck = lane & 7;
                float4 v;
                asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                             : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                             : "r"(region + (uint32_t)row * 128u + (uint32_t)((ck ^ (row & 7)) * 16)));
                const int r = w * 32 + row;  // row of the tile
                if (r >= wk.rows) continue;
                const int col = t * 32 + ck * 4;
                const int ra = wk.row_base + r, tn = ra / G;
                const size_t orow = ((size_t)wk.b * pl.T_cap + tn) * pl.Hq + wk.g * G + (ra - tn * G);
                if (dbg_rows) {
                    float* d0 = dbg_rows + orow * (kD + 1) + col;
                    d0[0] = v.x; d0[1] = v.y; d0[2] = v.z; d0[3] = v.w;
                } else {
                    uint2 pk;
                    pk.x = pack2_bf16(v.x, v.y);
                    pk.y = pack2_bf16(v.z, v.w);
                    *reinterpret_cast<uint2*>(a.out + orow * kD + col) = pk;
                }
            }
            if (t == 0 && row_ok) {
                const int ra = wk.row_base + rl, tn = ra / G;
                const size_t orow = ((size_t)wk.b * pl.T_cap + tn) * pl.Hq + wk.g * G + (ra - tn * G);
                if (dbg_rows) dbg_rows[orow * (kD + 1) + kD] = lse_v;
                else if (a.lse) a.lse[orow] = lse_v;
            }
        }
        if (!direct) {
            // ---- publish this CTA's partial state and merge.  One wave (every CTA of the launch resident): wait
            // for the group and merge this CTA's SHARE of the rows, so the merge is spread over the group's SMs.
            // Several waves: nobody waits (a waiting CTA would hold an SM that later CTAs need, and its siblings
            // need not be resident); the LAST CTA to arrive merges all rows of the group. ----
            const unsigned expected = (unsigned)wk.n_chunks;
            unsigned* cnt = a.counters + 2 * wk.group;  // [0] arrivals, [1] done
            named_bar_sync(10, 512);  // every thread's partial-state writes happen before the leader's (cumulative) release
            unsigned done_before = 0;
            if (pl.last_merges) {
                if (warp == 0 && lane == 0) {
                    __threadfence();
                    const unsigned before = atomicAdd(cnt, 1u);
                    __threadfence();  // acquire side for the last arriver
                    if (before == expected - 1) cnt[0] = 0;  // the counter is ready for the next launch
                    xl[0] = __int_as_float(before == expected - 1);
                }
                named_bar_sync(9, 512);
                if (__float_as_int(xl[0])) merge_rows(pl, a, dbg_rows, wk, 0, wk.rows, warp, lane);
            } else {
                int ok = 1;
                if (warp == 0 && lane == 0) {
                    // (release at gpu scope, cumulative over the other threads' writes ordered before it by the
                    // barrier above: no separate fence)
                    asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(cnt) : "memory");
                    unsigned seen, spins = 0;
                    do {
                        // relaxed: an acquire here would invalidate the whole L1 on every poll; one fence follows
                        asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(cnt) : "memory");
                        if (seen < expected) {
                            __nanosleep(20);
                            if (++spins > (1u << 22)) {  // the group never became co-resident: report, do not hang
                                atomicExch(a.counters + kWsErrorWord, 1u);
                                ok = 0;
                                break;
                            }
                        }
                    } while (seen < expected);
                    // acquire side: one acquire load of the counter (lighter than a full fence: nothing of this thread's
                    // own is outstanding); the states are read at L2 (ld.global.cg) behind the barrier below
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(cnt) : "memory");
                    // this CTA is past the wait: count it out now, the round trip hides behind the merge
                    done_before = atomicAdd(cnt + 1, 1u);
                    xl[0] = __int_as_float(ok);
                }
                named_bar_sync(9, 512);
                if (__float_as_int(xl[0]))
                    merge_rows(pl, a, dbg_rows, wk, wk.rows * wk.chunk / wk.n_chunks, wk.rows * (wk.chunk + 1) / wk.n_chunks,
                               warp, lane);
                if (warp == 0 && lane == 0) {
                    if (done_before == expected - 1) {  // last CTA out: everybody is past the wait
                        cnt[0] = 0;
                        cnt[1] = 0;
                    }
                }
            }
        }
      }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 18) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(kTmemCols) : "memory");
    }
    // no CTA leaves while its peer may still signal its barriers (every thread of the pair arrived after its last
    // remote operation; by now the peer's arrivals are an epilogue old)
    if (pair) asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}

// ---- host side ----------------------------------------------------------------------------------
}  // namespace

bool attn_stream_supported(const AttnPlan& pl) {
    // contiguous or 16-key-paged KV, rows of one query tile must be whole tree nodes (128 % G == 0),
    // and the tensor-map extents must fit.
    return (pl.page_size == 0 || pl.page_size == 16) && pl.d == kD && pl.G <= 128 && (128 % pl.G) == 0 &&
           (int64_t)pl.B * pl.T_cap < (1ll << 31) && pl.kv_rows < (1ll << 31);
}

int32_t launch_attn_stream(const AttnPlan& pl, const AttnArgs& a, int mode, float* dbg_rows, cudaStream_t s) {
    static unsigned long long attr_done = 0;
    if (first_use_on_device(attr_done))
        D2SD_CHECK_CUDA(cudaFuncSetAttribute(attn_stream_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
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
    cfg.gridDim = dim3((pl.n_mt >> 1) * 2 * pl.chunks_a + (pl.n_mt & 1) * ((pl.chunks_b + 1) & ~1), pl.Hkv, pl.B);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = kSmemBytes;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;  // PDL: see the file header
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    D2SD_CHECK_CUDA(cudaLaunchKernelEx(&cfg, attn_stream_kernel, tm_q, tm_k, tm_v, tm_tk, tm_tv, pl, a, mode, dbg_rows));
    D2SD_CHECK_LAUNCH("attn_stream_kernel");
    return D2SD_OK;
}


}  // namespace d2sd
