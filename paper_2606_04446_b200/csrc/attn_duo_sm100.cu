// Stage (c), fused: cascade tree-verify attention, TWO query tiles per CTA (tcgen05 / TMEM / TMA, sm_100a).
// PAPER.md:52, :124, :154.  Sibling of attn_stream_sm100.cu (one query tile per CTA); api.cu picks this one
// where the bytes delivered from L2 to the SMs bound the launch (long contexts, wide trees, several waves).
//
// Every M-tile CTA needs the whole K and V tile in its own shared memory, and the fabric between L2 and the
// SMs delivers ~6.5 TB/s in total whatever the L2 hit rate (multicast inside a cluster reads L2 once but
// still delivers twice).  A CTA of this kernel serves (request, kv head, ITEM, context chunk), an item being
// the M tiles (2i, 2i+1) -- 256 query rows per delivered KV byte -- or an odd last M tile on its own.
//
// A 128-key tile is processed as 64-key SUB-UNITS, always two halves per (key tile, M tile) (a ragged tile's
// empty half is a no-op that keeps the rotation static): duo item  n -> (h0,m0) (h0,m1) (h1,m0) (h1,m1),
// solo item n -> (h0) (h1).  Sub-unit n uses TMEM buffer n & 3 and softmax team n & 3 (four warps, one thread
// per query row, 64 scores each).  TMEM (512 columns): O_0, O_1 (128 fp32 columns each), four S/P buffers
// (64 columns each); P (bf16 pairs, 32 columns) is written over the S it was computed from, so a buffer's
// chain is  Q.K^T -> softmax -> P.V -> next Q.K^T  and four chains are in flight:
//
//   S[128 x 64]   = Q_m[128 x 128] . K^T         tcgen05.mma, A/B from 128B-swizzled SMEM (TMA)
//   P             = exp2(c*(S - m_ref))          softmax thread per row (TMEM lane), P -> TMEM over S
//   O_m[128x128] += P[128 x 64] . V              tcgen05.mma, A = P from TMEM, B = V (MN-major SMEM)
//
// Warp roles (640 threads): warps 0..15 = four softmax teams; warp 16 = K producer (+ Q tiles), warp 17 = V
// producer (also zeroes the V rows behind a ragged tile end), warp 18 = Q.K^T issuer (owns the TMEM
// allocation), warp 19 = P.V issuer.  The sub-units of one M tile alternate between two teams (duo) or
// rotate over all four (solo), and that M tile has ONE accumulator: the row's reference maximum travels with
// the M tile's sub-unit sequence through shared memory (an mbarrier per (team, warp)); the owner of a
// sub-unit raises it only when the tile maximum exceeds it by more than 2^8 (lazy rescale) and then -- after
// P.V of the M tile's previous sub-unit has completed, before it releases its own P -- rescales its O row.
// Each thread keeps its own row sum relative to the last reference it saw; the sums meet in the epilogue.
//
// Cascade merge in the same launch as in attn_stream_sm100.cu: single-chunk groups write `out` directly;
// otherwise the CTA writes its normalised state (O rows in bf16, LSE fp32), and either (one wave) waits for
// its group and merges its share of the rows, or (several waves) leaves, the last arriver merging the group.
#include "tc_ptx.cuh"

namespace d2sd {
namespace {

constexpr int kRingK = 2, kRingV = 3;   // K tiles / V tiles in flight or in use (half-tile slots measured slower: the
                                        // 16 KiB boxes double the TMA operations, configs 3/4/5: 83 / 64 / 386 us vs 68 / 55 / 314)
constexpr int kThreads = 640;      // 16 softmax warps (4 teams) + 4 control warps
constexpr int kTeams = 4;
constexpr int kSubN = 64;          // keys per sub-unit
constexpr int kItemRows = 2 * kTileM;  // partial-state rows per (chunk, item)
constexpr uint32_t kOffQ = 0;                               // two query tiles
constexpr uint32_t kOffK = 2 * kQTileBytes;
constexpr uint32_t kOffV = kOffK + kRingK * kKvTileBytes;
constexpr uint32_t kOffBar = kOffV + kRingV * kKvTileBytes;
constexpr uint32_t kOffX = kOffBar + 512;                   // reference-maximum hand-off: fp32 [4 teams][128 rows]
constexpr uint32_t kSmemUsed = kOffX + kTeams * kTileM * 4;
constexpr uint32_t kSmemBytes = 232448;                     // the whole 227 KiB: kSmemUsed + alignment slack
constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kTmemBuf = 256;  // four S/P buffers behind O_0, O_1
constexpr float kRescaleThreshold = 8.0f;  // log2 units
constexpr uint32_t kRegsControl = 64, kRegsSoftmax = 104;  // setmaxnreg targets: 512 x 104 + 128 x 64 = the launch allocation

enum : uint32_t {
    kBarQFull = 0,                       // [2]
    kBarKFull = 2,                       // [kRingK]
    kBarKEmpty = kBarKFull + kRingK,     // [kRingK]
    kBarVFull = kBarKEmpty + kRingK,     // [kRingV]
    kBarVEmpty = kBarVFull + kRingV,     // [kRingV]
    kBarSFull = kBarVEmpty + kRingV,     // [4] Q.K^T of a sub-unit has completed
    kBarPFull = kBarSFull + kTeams,      // [4] the owning team has written P over S
    kBarPFree = kBarPFull + kTeams,      // [4] P.V of a sub-unit has completed (buffer reusable, O current)
    kBarRef = kBarPFree + kTeams,        // [4 teams][4 warps] the team's warp has published its rows' reference maxima
    kBarVFix = kBarRef + 4 * kTeams,     // [2] V rows behind a ragged tile end are zero (<= 2 ragged tiles per CTA)
    kBarAllDone = kBarVFix + 2,
    kNumBars = kBarAllDone + 1,
    kTmemSlot = kNumBars  // uint32 written by tcgen05.alloc
};
static_assert((kNumBars + 1) * 8 <= 512, "barrier area");
static_assert(kSmemUsed + 512 <= kSmemBytes, "shared memory budget");  // the kernel checks the actual alignment slack

struct Work {
    int b, g, item, chunk;
    int n_m;           // M tiles this CTA really holds (2: duo, 1: solo or a duo whose second tile has no rows)
    int row_base;      // first query row (t*G + hh) of the item
    int rows0, rows1;  // valid query rows of the two M tiles
    int np, nt;        // prefix / tree key tiles of the request (after the mode bits)
    int j_begin, n_tiles;
    int n_chunks;      // non-empty chunks of the group = CTAs that arrive at the group counter
    int group;         // (b*Hkv + g)*n_items + item
    int T, L;
    __device__ __forceinline__ int rows(int m) const { return m ? rows1 : rows0; }
    __device__ __forceinline__ int rows_item() const { return rows0 + rows1; }
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
__device__ __forceinline__ float bf_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf_hi(uint32_t w) { return __uint_as_float(w & 0xFFFF0000u); }

// -------------------------------------------------------------------------------------------------
// Cascade merge of one group's rows (log-sum-exp state merge):
//   LSE = log sum_p e^{LSE_p};  O = sum_p e^{LSE_p - LSE} O_p   over the group's chunk states.
// CTA `chunk` of the group's n_chunks CTAs takes a contiguous range of the item's rows.  One THREAD takes 8
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
    const int nrows = r1 - r0;  // <= 256
    const int g_shift = __ffs(G) - 1;  // G divides 128 (attn_duo_supported): a power of two
    constexpr int kSB = 8;      // states per batch
    for (int idx = warp * 32 + lane; idx < nrows * 16; idx += 512) {
        const int r = r0 + (idx >> 4), cg = idx & 15;
        const float* lp = a.part_lse + grp0 + r;
        const __nv_bfloat16* op = a.part_o16 + (grp0 + r) * kD + cg * 8;
        float lv[kSB];
        uint4 v[kSB];
#pragma unroll
        for (int i = 0; i < kSB; ++i) lv[i] = i < nc ? ld_cg_f32(lp + (size_t)i * kItemRows) : -INFINITY;
#pragma unroll
        for (int i = 0; i < kSB; ++i)
            if (i < nc) v[i] = ld_cg_u4(op + (size_t)i * kItemRows * kD);
        float m = lv[0];
#pragma unroll
        for (int i = 1; i < kSB; ++i) m = fmaxf(m, lv[i]);
#pragma unroll 1
        for (int i = kSB; i < nc; ++i) m = fmaxf(m, ld_cg_f32(lp + (size_t)i * kItemRows));  // more than eight chunks
        float ws = 0.f, wv[kSB];
#pragma unroll
        for (int i = 0; i < kSB; ++i) {
            wv[i] = lv[i] == -INFINITY ? 0.f : __expf(lv[i] - m);
            ws += wv[i];
        }
#pragma unroll 1
        for (int i = kSB; i < nc; ++i) {
            const float l = ld_cg_f32(lp + (size_t)i * kItemRows);
            ws += l == -INFINITY ? 0.f : __expf(l - m);
        }
        const float inv = ws > 0.f ? __fdividef(1.f, ws) : 0.f;  // no key at all (L = 0, prefix-only mode): O = 0, LSE = -inf
        const float lse = ws > 0.f ? m + __logf(ws) : -INFINITY;  // (1 <= ws <= 64: lg2.approx is accurate to ~1e-7 here)
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
            const float l = ld_cg_f32(lp + (size_t)i * kItemRows);
            const float w1 = l == -INFINITY ? 0.f : __expf(l - m) * inv;
            const uint4 x = ld_cg_u4(op + (size_t)i * kItemRows * kD);
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
__global__ void __launch_bounds__(kThreads, 1)
attn_duo_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
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

    // ---- prologue that touches no global memory (overlaps the preceding kernel's tail under PDL) ----
    if (warp == 16 && lane == 0) {
        mbar_init(bar(kBarQFull + 0), 1);
        mbar_init(bar(kBarQFull + 1), 1);
        for (int i = 0; i < kRingK; ++i) {
            mbar_init(bar(kBarKFull + i), 1);
            mbar_init(bar(kBarKEmpty + i), 1);
        }
        for (int i = 0; i < kRingV; ++i) {
            mbar_init(bar(kBarVFull + i), 1);
            mbar_init(bar(kBarVEmpty + i), 1);
        }
        for (int t = 0; t < kTeams; ++t) {
            mbar_init(bar(kBarSFull + t), 1);
            mbar_init(bar(kBarPFull + t), 4);  // one elected arrival per warp of the owning team
            mbar_init(bar(kBarPFree + t), 1);
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
    pdl_launch_dependents();  // the next kernel may begin its own prologue as SMs free up
    pdl_wait();               // everything before this kernel in the stream is complete and visible

    // ---- this CTA's work ----
    Work wk;
    {
        const int G = pl.G;
        wk.g = blockIdx.y;
        wk.b = blockIdx.z;
        if (pl.last_merges && pl.B <= 32) {
            // Several waves: blocks are handed out in grid order, so the requests are taken longest first (slice z of
            // the grid serves the request of rank z by context length, ties by index) and the last, partly filled
            // wave is made of short CTAs.  Every warp computes the same permutation.
            const int Lz = lane < pl.B ? a.ctx_len[lane] : -1;
            int rank = 0;
            for (int j = 0; j < pl.B; ++j) {
                const int Lj = __shfl_sync(0xffffffffu, Lz, j);
                rank += (Lj > Lz || (Lj == Lz && j < lane)) ? 1 : 0;
            }
            const unsigned hit = __ballot_sync(0xffffffffu, lane < pl.B && rank == (int)blockIdx.z);
            wk.b = __ffs(hit) - 1;
        }
        int x = blockIdx.x, n_static;
        bool duo;
        if (x < pl.n_pair * pl.chunks_a) {
            wk.item = x / pl.chunks_a; wk.chunk = x - wk.item * pl.chunks_a; n_static = pl.chunks_a; duo = true;
        } else {
            x -= pl.n_pair * pl.chunks_a;
            wk.item = pl.n_pair; wk.chunk = x; n_static = pl.chunks_b; duo = false;
        }
        wk.T = a.tree_len[wk.b];
        wk.L = a.ctx_len[wk.b];
        const int rows_valid = wk.T * G;
        wk.row_base = wk.item * kItemRows;
        wk.rows0 = max(0, min(kTileM, rows_valid - wk.row_base));
        wk.rows1 = duo ? max(0, min(kTileM, rows_valid - wk.row_base - kTileM)) : 0;
        wk.n_m = wk.rows1 > 0 ? 2 : 1;
        wk.group = (wk.b * pl.Hkv + wk.g) * (pl.n_pair + pl.n_single) + wk.item;
        wk.np = (mode & 1) ? (wk.L + kTileN - 1) / kTileN : 0;
        wk.nt = (mode & 2) ? (wk.T + kTileN - 1) / kTileN : 0;
        const int nk = wk.np + wk.nt;
        const int tps = max(max(1, pl.tps_min), (nk + n_static - 1) / n_static);
        wk.n_chunks = max(1, (nk + tps - 1) / tps);  // chunk 0 always takes part (nk = 0: state (0, -inf))
        wk.j_begin = wk.chunk * tps;
        wk.n_tiles = max(0, min(nk, wk.j_begin + tps) - wk.j_begin);
    }
    // items past the tree's rows, and chunks past the request's key tiles, leave at once: nobody waits for them
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
    const int N = wk.n_tiles;
    const int n_m = wk.n_m;
    const int n_sub = N * 2 * n_m;  // sub-units of this CTA: two halves per (key tile, M tile)

    if (warp >= 16) {
      asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsControl));
      if (idle) {
        // fall through to the TMEM release
      } else if (warp == 16 || warp == 17) {
        // ===== K producer (warp 16, also loads the query tiles) and V producer (warp 17).  Contiguous KV: lane 0
        // issues one 32 KiB box per tile.  Paged KV (page = 16 keys): a 128-key tile is 8 pages; lane 2p+hi
        // issues the 2 KiB box (page p, d half hi), so a tile is 16 loads in flight at once; only the
        // ceil(valid/16) pages that exist are loaded (the MMAs never read past ceil16(valid) keys); the page ids
        // of the next tile are fetched one tile ahead.  The V producer also zeroes the V rows behind a ragged
        // tile end: the P.V MMA runs over ceil16(valid) keys, rows valid..ceil16(valid)-1 belong to nobody (next
        // request, tree padding), are multiplied by P = 0 exactly and must not hold NaN/Inf.  A row is 2 x 128 B
        // (d halves); the 128B swizzle permutes 16-byte chunks inside a row's 128 B only. =====
        const bool is_v = warp == 17;
        const bool paged = pl.page_size > 0;
        const int ring = is_v ? kRingV : kRingK;
        const uint32_t ring_off = is_v ? kOffV : kOffK;
        const uint32_t bar_full = is_v ? kBarVFull : kBarKFull, bar_empty = is_v ? kBarVEmpty : kBarKEmpty;
        auto page_of = [&](int jj) {
            int pg = 0;
            if (paged && jj < N) {
                const TileInfo t2 = tile_info(jj);
                const int p = lane >> 1;
                if (!t2.tree && lane < 16 && p * 16 < t2.valid) pg = __ldg(a.kv_indices + kv_row0 + t2.j * 8 + p);
            }
            return pg;
        };
        if (!is_v && lane == 0) {  // one box = a 128-row query tile of this kv head
            for (int m = 0; m < n_m; ++m) {
                const int t0 = wk.b * pl.T_cap + (wk.row_base + m * kTileM) / pl.G;
                mbar_expect_tx(bar(kBarQFull + m), kQTileBytes);
                tma_load_5d(smem + kOffQ + m * kQTileBytes, &tm_q, bar(kBarQFull + m), 0, 0, t0, 0, wk.g, kEvictLast);
            }
        }
        int page_cur = page_of(0);
        int n_ragged = 0;
        for (int jj = 0; jj < N; ++jj) {
            const TileInfo ti = tile_info(jj);
            const int page_next = page_of(jj + 1);
            const int i = jj % ring;
            const uint32_t dst = smem + ring_off + i * kKvTileBytes;
            const uint32_t fb = bar(bar_full + i);
            const bool by_page = paged && !ti.tree;
            const int n_pages = (ti.valid + 15) >> 4;
            if (lane == 0) {
                mbar_wait(bar(bar_empty + i), ((jj / ring) & 1) ^ 1);
                mbar_expect_tx(fb, by_page ? (uint32_t)n_pages * 4096u : kKvTileBytes);
            }
            __syncwarp();
            if (by_page) {
                if (lane < 2 * n_pages)
                    tma_load_5d(dst + (uint32_t)(lane & 1) * (kKvTileBytes / 2) + (uint32_t)(lane >> 1) * 2048u,
                                is_v ? &tm_v : &tm_k, fb, 0, 0, lane & 1, wk.g, page_cur, kEvictNormal);
            } else if (lane == 0) {
                const CUtensorMap* tm = ti.tree ? (is_v ? &tm_tv : &tm_tk) : (is_v ? &tm_v : &tm_k);
                tma_load_4d(dst, tm, fb, 0, ti.row, 0, wk.g, ti.tree ? kEvictLast : kEvictNormal);
            }
            if (is_v && (ti.valid & 15) != 0) {
                mbar_wait(fb, (jj / ring) & 1);  // this fill has landed (every lane observes it)
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
        }
      } else {
        // ===== MMA issuers (warp 18: Q.K^T stream, warp 19: P.V stream), one elected thread each.  Sub-unit n =
        // (key tile n / (2 n_m), M tile, half); buffer n & 3.  Q.K^T of sub-unit n needs the buffer back from
        // P.V of sub-unit n-4 (P lies over S); P.V of sub-unit n needs the owning team's P.  A ring slot is
        // released by the commit behind its last reader. =====
        if (elect_one()) {
            const int per = 2 * n_m;  // sub-units per key tile: n -> (key tile n / per, half (n % per) / n_m, M tile n % n_m)
            // (per is 2 or 4: shifts; every key tile is whole except the request's last prefix and last tree tile:
            // the issuer threads pace the kernel, see attn_stream_sm100.cu)
            const int jr0 = wk.np - 1 - wk.j_begin, jr1 = wk.np + wk.nt - 1 - wk.j_begin;
            const int v0 = wk.L - (wk.np - 1) * kTileN, v1 = wk.T - (wk.nt - 1) * kTileN;
            auto valid_of = [&](int jj) { return jj == jr0 ? v0 : (jj == jr1 ? v1 : kTileN); };
            if (warp == 18) {
                for (int m = 0; m < n_m; ++m) mbar_wait(bar(kBarQFull + m), 0);  // (also with N = 0: no load left in flight)
                uint32_t n = 0, ki = 0, kph = 0;
                for (int jj = 0; jj < N; ++jj) {
                    const int valid = valid_of(jj);
                    // the tile's K barrier and the buffers of its first two sub-units, probed together
                    uint32_t ok_k, ok_0, ok_1;
                    mbar_probe3(bar(kBarKFull + ki), kph, n >= kTeams ? bar(kBarPFree + (n & 3)) : bar(kBarQFull),
                                n >= kTeams ? (((n >> 2) & 1) ^ 1) : 0u,
                                n + 1 >= kTeams ? bar(kBarPFree + ((n + 1) & 3)) : bar(kBarQFull),
                                n + 1 >= kTeams ? ((((n + 1) >> 2) & 1) ^ 1) : 0u, ok_k, ok_0, ok_1);
                    if (!ok_k) mbar_wait(bar(kBarKFull + ki), kph);
                    const uint64_t kd0 = smem_desc(smem + kOffK + ki * kKvTileBytes, 16, 1024);
#pragma unroll 1
                    for (int r = 0; r < per; ++r, ++n) {
                        const int hf = r >> (n_m - 1), m = r & (n_m - 1);
                        const uint32_t t = n & 3;
                        // P.V of n-4 has consumed the buffer
                        if (n >= kTeams && !(r == 0 ? ok_0 : (r == 1 ? ok_1 : 0u)))
                            mbar_wait(bar(kBarPFree + t), ((n >> 2) & 1) ^ 1);
                        int n_cols = (max(0, min(kSubN, valid - hf * kSubN)) + 15) & ~15;  // MMA N (multiple of 16); an empty
                        if (n_cols == 0) n_cols = 16;  // half still produces 16 columns that are all masked
                        const uint64_t qd = smem_desc(smem + kOffQ + m * kQTileBytes, 16, 1024);
                        const uint64_t kd = kd0 + (uint64_t)((hf * (kSubN * 128u)) >> 4);
                        const uint32_t id_qk = idesc(kTileM, (uint32_t)n_cols, 0);
                        const uint32_t sd = tmem + kTmemBuf + t * kSubN;
                        tc_fence_after();
#pragma unroll
                        for (int kk = 0; kk < kD / 16; ++kk) {
                            const uint64_t off = (uint64_t)(((kk >> 2) * (kQTileBytes / 2) + (kk & 3) * 32) >> 4);
                            umma_ss(sd, qd + off, kd + off, id_qk, kk > 0);
                        }
                        tc_commit(bar(kBarSFull + t));
                    }
                    tc_commit(bar(kBarKEmpty + ki));  // K is free once the tile's last Q.K^T has completed
                    if (++ki == (uint32_t)kRingK) { ki = 0; kph ^= 1u; }
                }
            } else {
                uint32_t n_ragged = 0, started = 0;  // started: bit m set once O_m holds a product
                uint32_t n = 0, vi = 0, vph = 0;
                for (int jj = 0; jj < N; ++jj) {
                    const int valid = valid_of(jj);
                    uint32_t ok_v, ok_p, ok_x;
                    mbar_probe3(bar(kBarVFull + vi), vph, bar(kBarPFull + (n & 3)), (n >> 2) & 1, bar(kBarQFull), 0u, ok_v,
                                ok_p, ok_x);
                    if (!ok_v) mbar_wait(bar(kBarVFull + vi), vph);
                    if (valid & 15) mbar_wait(bar(kBarVFix + n_ragged++), 0);
                    const uint64_t vd = smem_desc(smem + kOffV + vi * kKvTileBytes, kKvTileBytes / 2, 1024);
#pragma unroll 1
                    for (int r = 0; r < per; ++r, ++n) {
                        const int hf = r >> (n_m - 1), m = r & (n_m - 1);
                        const uint32_t t = n & 3;
                        const int keys = max(0, min(kSubN, valid - hf * kSubN));
                        const int ksteps = ((keys + 15) & ~15) >> 4;  // K extent of this P.V in 16-key steps
                        const uint32_t pd = tmem + kTmemBuf + t * kSubN;
                        const uint32_t od = tmem + m * kD;
                        if (!(r == 0 && ok_p)) mbar_wait(bar(kBarPFull + t), (n >> 2) & 1);
                        tc_fence_after();
#pragma unroll
                        for (int ks = 0; ks < kSubN / 16; ++ks)
                            if (ks < ksteps)
                                umma_ts(od, pd + ks * 8, vd + (uint64_t)((hf * (kSubN / 16) + ks) * (2048 >> 4)), kIdescPV,
                                        ((started >> m) & 1u) | ks);
                        if (ksteps > 0) started |= 1u << m;
                        tc_commit(bar(kBarPFree + t));
                    }
                    tc_commit(bar(kBarVEmpty + vi));  // V is free once the tile's last P.V has completed
                    if (++vi == (uint32_t)kRingV) { vi = 0; vph ^= 1u; }
                }
                tc_commit(bar(kBarAllDone));
            }
        }
      }
    } else {
      asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegsSoftmax));
      if (!idle) {
        // ===== softmax: team t owns the sub-units n = t (mod 4): in a duo item M tile t >> 1, half t & 1 of every
        // key tile; in a solo item the halves of the key tiles in rotation.  Thread (w, lane) owns query row
        // w*32 + lane of its M tile (TMEM lane) and the sub-unit's 64 scores. =====
        const int t = warp >> 2;       // team
        const int w = warp & 3;
        const int rl = w * 32 + lane;  // row within the M tile
        const uint32_t lane_addr = (uint32_t)(w * 32) << 16;
        const float c2 = pl.sm_scale * kLog2e;
        const float thr = kRescaleThreshold / c2;  // in raw score units
        float* xm = reinterpret_cast<float*>(smem_gen + kOffX);  // [team][row]: reference maximum after the team's last sub-unit
        const int per = 2 * n_m;
        const int m = n_m == 2 ? (t & 1) : 0;                // this team's M tile
        const int tp = (t + kTeams - n_m) & 3;               // the team that owns the M tile's previous sub-unit (n - n_m)
        const bool warp_active = w * 32 < wk.rows(m);
        float m_mine = -INFINITY;  // the reference this thread's row sum is relative to
        float l_mine = 0.f;
        const int t_node = min((wk.row_base + m * kTileM + rl) / pl.G, wk.T - 1);
        const uint32_t* mrow = a.mask + ((size_t)wk.b * pl.T_cap + t_node) * pl.W;
        const uint32_t sbuf = tmem + kTmemBuf + t * kSubN + lane_addr;
        const uint32_t o_addr = tmem + m * kD + lane_addr;
        const int s_jr0 = wk.np - 1 - wk.j_begin, s_jr1 = wk.np + wk.nt - 1 - wk.j_begin, s_jtree = wk.np - wk.j_begin;
        const int s_v0 = wk.L - (wk.np - 1) * kTileN, s_v1 = wk.T - (wk.nt - 1) * kTileN;
        for (int n = t; n < n_sub; n += kTeams) {
            const int jj = n >> n_m, r = n & (per - 1), hf = r >> (n_m - 1);
            const int par = (n >> 2) & 1;
            struct { int valid; bool tree; int tt; } ti;  // (no per-tile decode: see the issuers)
            ti.valid = jj == s_jr0 ? s_v0 : (jj == s_jr1 ? s_v1 : kTileN);
            ti.tree = jj >= s_jtree;
            ti.tt = jj - s_jtree;
            const int keys = max(0, min(kSubN, ti.valid - hf * kSubN));
            // the M tile's previous sub-unit is n - n_m (the sequence is (h0: m0 [m1]) (h1: m0 [m1]) per key tile)
            const int n_prev = n - n_m;
            const bool has_prev = n_prev >= 0;
            const bool has_next = n + n_m < n_sub;
            mbar_wait(bar(kBarSFull + t), par);
            if (!warp_active) {  // a warp without rows only keeps the barrier phases in step
                if (lane == 0) mbar_arrive(bar(kBarPFull + t));
                __syncwarp();
                continue;
            }
            uint32_t sv[kSubN];
            tc_fence_after();
            D2SD_TMEM_LD32(sbuf, sv, 0);
            D2SD_TMEM_LD32(sbuf + 32, sv, 32);
            tmem_wait_ld();
            if (ti.tree || keys < kSubN) {
                // keys past the tile's end, and (tree tiles) keys that are not ancestors-or-self of this row's
                // node: the sub-unit's 64 mask bits -> -inf
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
            // reference hand-off along the M tile's sub-unit sequence, lazy raise
            float m_prev = -INFINITY;
            if (has_prev) {
                mbar_wait(bar(kBarRef + 4 * tp + w), (n_prev >> 2) & 1);
                m_prev = xm[tp * kTileM + rl];
            }
            const bool need = has_prev && mx > m_prev + thr;
            const float m_new = !has_prev ? mx : (need ? mx : m_prev);
            if (has_next) {
                xm[t * kTileM + rl] = m_new;
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(kBarRef + 4 * t + w));
            }
            if (m_new != m_mine) {  // this thread's own row sum follows the reference
                l_mine *= m_mine == -INFINITY ? 0.f : ex2((m_mine - m_new) * c2);
                m_mine = m_new;
            }
            if (__any_sync(0xffffffffu, need)) {
                // O_m holds the M tile's earlier sub-units relative to m_prev: wait for P.V of the previous one,
                // rescale this row.  (Sound as a single parity wait: this sub-unit's S needed P.V of n-4 complete,
                // hence P.V of n_prev-4, so that barrier is at most one phase behind.)  P.V of this sub-unit
                // cannot start before this thread releases P below.
                mbar_wait(bar(kBarPFree + (n_prev & 3)), (n_prev >> 2) & 1);
                tc_fence_after();
                const float alpha = need ? (m_prev == -INFINITY ? 0.f : ex2((m_prev - m_new) * c2)) : 1.f;
#pragma unroll 1
                for (int c0 = 0; c0 < kD; c0 += 16) {
                    uint32_t o[16];
                    asm volatile(
                        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                        : "=r"(o[0]), "=r"(o[1]), "=r"(o[2]), "=r"(o[3]), "=r"(o[4]), "=r"(o[5]), "=r"(o[6]), "=r"(o[7]),
                          "=r"(o[8]), "=r"(o[9]), "=r"(o[10]), "=r"(o[11]), "=r"(o[12]), "=r"(o[13]), "=r"(o[14]), "=r"(o[15])
                        : "r"(o_addr + c0));
                    tmem_wait_ld();
#pragma unroll
                    for (int c = 0; c < 16; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * alpha);
                    D2SD_TMEM_ST16(o_addr + c0, o);
                }
                tmem_wait_st();
                tc_fence_before();
            }
            // a row with every key so far masked has m_ref = -inf: exp2(-inf - 0) = 0, not NaN
            const float ms = m_new == -INFINITY ? 0.f : m_new * c2;
            float sum0 = 0.f, sum1 = 0.f;
            // P[128 x 64] bf16 = 32 TMEM columns written over the first half of S (this thread has its whole S row
            // in registers; other rows are other TMEM lanes)
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
                D2SD_TMEM_ST16(sbuf + q * 16, p);
            }
            l_mine += sum0 + sum1;
            tmem_wait_st();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(kBarPFull + t));
        }
        // ---- epilogue: the row sums of the teams that share an M tile meet at the final reference; the normalised
        // state leaves the CTA straight from registers through a per-warp transpose in shared memory (the rings
        // are free): a thread holds 64 (duo) or 32 (solo) columns of its row, 32 at a time. ----
        const int t_last = n_m == 2 ? m + 2 : (n_sub - 1) & 3;  // the team that owns the M tile's last sub-unit
        if (warp_active && n_sub > 0 && t_last == t) xm[t * kTileM + rl] = m_mine;
        mbar_wait(bar(kBarAllDone), 0);  // every MMA done: O is final, the rings are free
        named_bar_sync(9, 512);
        const float m_fin = n_sub > 0 ? xm[t_last * kTileM + rl] : -INFINITY;
        if (m_fin != m_mine) l_mine *= m_mine == -INFINITY ? 0.f : ex2((m_mine - m_fin) * c2);
        float* xl = reinterpret_cast<float*>(smem_gen + kOffV);  // [team][row]
        xl[t * kTileM + rl] = l_mine;
        named_bar_sync(10, 512);
        const float l_tot = n_m == 2 ? xl[m * kTileM + rl] + xl[(m + 2) * kTileM + rl]
                                     : (xl[rl] + xl[kTileM + rl]) + (xl[2 * kTileM + rl] + xl[3 * kTileM + rl]);
        const float inv = l_tot > 0.f ? 1.f / l_tot : 0.f;  // l = 0: every key of the chunk masked, or no key at all
        const float lse_v = l_tot > 0.f ? m_fin * pl.sm_scale + logf(l_tot) : -INFINITY;
        const bool direct = wk.n_chunks == 1;
        const int rows_m = wk.rows(m);
        const size_t prow0 = (size_t)wk.group * pl.grp_rows + (size_t)wk.chunk * kItemRows + (size_t)m * kTileM;
        if (warp_active) {
            // per-warp staging: [32 rows][128 B] of fp32 (direct output) or [32 rows][64 B] of bf16 pairs (partial
            // state), 16-byte chunks XOR-swizzled by the row
            const uint32_t region = smem + kOffK + (uint32_t)warp * 4096u;
            const int G = pl.G;
            const int col_base = n_m == 2 ? (t >> 1) * 64 : t * 32, n_piece = n_m == 2 ? 2 : 1;
#pragma unroll 1
            for (int pc = 0; pc < n_piece; ++pc) {
                const int col0 = col_base + 32 * pc;
                uint32_t ov[32];
                tc_fence_after();
                if (n_sub > 0) {
                    D2SD_TMEM_LD32(o_addr + col0, ov, 0);
                    tmem_wait_ld();
                }
#pragma unroll
                for (int c = 0; c < 32; ++c) ov[c] = n_sub > 0 ? __float_as_uint(__uint_as_float(ov[c]) * inv) : 0u;
                __syncwarp();  // the previous piece has been read out of the staging region
                if (direct) {
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
                        const int r = w * 32 + row;  // row of the M tile
                        if (r >= rows_m) continue;
                        const int col = col0 + ck * 4;
                        const int ra = wk.row_base + m * kTileM + r, tn = ra / G;
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
                } else {
#pragma unroll
                    for (int c = 0; c < 32; c += 8) {  // 8 columns = one 16-byte chunk of bf16
                        const uint32_t chunk = (uint32_t)(c >> 3) ^ ((uint32_t)(lane >> 1) & 3u);
                        uint32_t pk[4];
#pragma unroll
                        for (int e = 0; e < 4; ++e) pk[e] = pack2_bf16(__uint_as_float(ov[c + 2 * e]), __uint_as_float(ov[c + 2 * e + 1]));
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
                        const int r = w * 32 + row;  // row of the M tile
                        if (r < rows_m) *reinterpret_cast<uint4*>(a.part_o16 + (prow0 + r) * kD + col0 + ck * 8) = v;
                    }
                }
            }
            const bool lse_writer = n_m == 2 ? (t >> 1) == 0 : t == 0;
            if (lse_writer && rl < rows_m) {
                if (!direct) {
                    a.part_lse[prow0 + rl] = lse_v;
                } else {
                    const int ra = wk.row_base + m * kTileM + rl, tn = ra / G;
                    const size_t orow = ((size_t)wk.b * pl.T_cap + tn) * pl.Hq + wk.g * G + (ra - tn * G);
                    if (dbg_rows) dbg_rows[orow * (kD + 1) + kD] = lse_v;
                    else if (a.lse) a.lse[orow] = lse_v;
                }
            }
        }
        if (!direct) {
            // ---- publish this CTA's partial state and merge (see attn_stream_sm100.cu): one wave -> wait for the
            // group, merge this CTA's share of the item's rows; several waves -> the last arriver merges them all ----
            const unsigned expected = (unsigned)wk.n_chunks;
            unsigned* cnt = a.counters + 2 * wk.group;  // [0] arrivals, [1] done
            const int rows_item = wk.rows_item();
            named_bar_sync(9, 512);  // every thread's partial-state writes happen before the leader's (cumulative) release
            unsigned done_before = 0;
            if (pl.last_merges) {
                if (warp == 0 && lane == 0) {
                    __threadfence();
                    const unsigned before = atomicAdd(cnt, 1u);
                    __threadfence();  // acquire side for the last arriver
                    if (before == expected - 1) cnt[0] = 0;  // the counter is ready for the next launch
                    xl[0] = __int_as_float(before == expected - 1);
                }
                named_bar_sync(10, 512);
                if (__float_as_int(xl[0])) merge_rows(pl, a, dbg_rows, wk, 0, rows_item, warp, lane);
            } else {
                int ok = 1;
                if (warp == 0 && lane == 0) {
                    __threadfence();
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
                    // acquire side: one acquire load of the counter; the states are read at L2 (ld.global.cg) behind
                    // the barrier below
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(cnt) : "memory");
                    done_before = atomicAdd(cnt + 1, 1u);
                    xl[0] = __int_as_float(ok);
                }
                named_bar_sync(10, 512);
                if (__float_as_int(xl[0]))
                    merge_rows(pl, a, dbg_rows, wk, rows_item * wk.chunk / wk.n_chunks, rows_item * (wk.chunk + 1) / wk.n_chunks,
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
}

// ---- host side ----------------------------------------------------------------------------------
}  // namespace

bool attn_duo_supported(const AttnPlan& pl) {
    // contiguous or 16-key-paged KV, rows of one query tile must be whole tree nodes (128 % G == 0),
    // and the tensor-map extents must fit.
    return (pl.page_size == 0 || pl.page_size == 16) && pl.d == kD && pl.G <= 128 && (128 % pl.G) == 0 &&
           (int64_t)pl.B * pl.T_cap < (1ll << 31) && pl.kv_rows < (1ll << 31);
}

int32_t launch_attn_duo(const AttnPlan& pl, const AttnArgs& a, int mode, float* dbg_rows, cudaStream_t s) {
    static unsigned long long attr_done = 0;
    if (first_use_on_device(attr_done))
        D2SD_CHECK_CUDA(cudaFuncSetAttribute(attn_duo_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
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
    D2SD_CHECK_CUDA(cudaLaunchKernelEx(&cfg, attn_duo_kernel, tm_q, tm_k, tm_v, tm_tk, tm_tv, pl, a, mode, dbg_rows));
    D2SD_CHECK_LAUNCH("attn_duo_kernel");
    return D2SD_OK;
}


}  // namespace d2sd
