// extern "C" entry points of libd2sd (declared and documented in include/d2sd.h): argument checks,
// launch planning, kernel enqueue.  No allocation, no synchronisation, no host reads of device data.
#include <cmath>
#include <cstring>

#include "common.cuh"

namespace d2sd {

static thread_local char g_err[512] = "";

int32_t set_error(int32_t status, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return status;
}
void clear_error() { g_err[0] = '\0'; }

int sm_count() {
    // per device (a process may drive several GPUs); a benign race at worst writes the same value twice
    static int cache[64] = {0};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 148;  // B200
    if (dev < 0 || dev >= 64) dev = 0;
    int n = cache[dev];
    if (n == 0) {
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
        cache[dev] = n;
    }
    return n;
}

static int32_t check_block(int32_t B, int32_t gamma, int32_t K) {
    D2SD_CHECK_ARG(B >= 0, "B = %d must be >= 0", B);
    D2SD_CHECK_ARG(gamma >= 2 && gamma <= 64, "gamma = %d outside [2,64]", gamma);
    D2SD_CHECK_ARG(K >= 0 && K <= gamma - 1, "K = %d outside [0,gamma-1] (gamma = %d)", K, gamma);
    return D2SD_OK;
}

// Split-KV plan.  chunk_keys is a multiple of 64 (the key-tile size of both prefix kernels).
static int32_t make_plan(const d2sd_attn_params* p, AttnPlan* out) {
    D2SD_CHECK_ARG(p != nullptr, "params is NULL");
    D2SD_CHECK_ARG(p->B >= 0 && p->T_cap >= 1, "B = %d, T_cap = %d", p->B, p->T_cap);
    D2SD_CHECK_ARG(p->Hq >= 1 && p->Hkv >= 1 && p->Hq % p->Hkv == 0, "Hq = %d not a multiple of Hkv = %d",
                   p->Hq, p->Hkv);
    D2SD_CHECK_ARG(p->max_ctx_len >= 0 && p->kv_rows >= 0, "max_ctx_len = %d, kv_rows = %lld",
                   p->max_ctx_len, (long long)p->kv_rows);
    D2SD_CHECK_ARG(p->num_splits >= 0 && p->impl >= 0 && p->impl <= 3, "num_splits = %d, impl = %d",
                   p->num_splits, p->impl);
    D2SD_CHECK_ARG(p->phases >= 0 && p->phases <= 7, "phases = %d outside [0,7]", p->phases);
    D2SD_CHECK_SUPPORTED(p->d == 128, "head dim %d: only 128 is built", p->d);
    D2SD_CHECK_SUPPORTED(p->page_size == 0 || p->page_size == 16, "page_size %d: only 0 (contiguous) or 16",
                         p->page_size);
    D2SD_CHECK_SUPPORTED(p->T_cap <= 1024, "T_cap = %d > 1024", p->T_cap);
    D2SD_CHECK_SUPPORTED((int64_t)p->B * p->Hkv <= 65535, "B*Hkv = %lld > 65535", (long long)p->B * p->Hkv);
    AttnPlan pl{};
    pl.B = p->B; pl.T_cap = p->T_cap; pl.W = (p->T_cap + 31) / 32;
    pl.Hq = p->Hq; pl.Hkv = p->Hkv; pl.G = p->Hq / p->Hkv; pl.d = p->d;
    pl.sm_scale = p->sm_scale > 0.f ? p->sm_scale : 1.0f / sqrtf((float)p->d);
    pl.page_size = p->page_size;
    pl.max_ctx_len = p->max_ctx_len;
    pl.kv_rows = p->kv_rows;
    pl.use_stream = false;
    pl.use_duo = false;
    // auto: the one-tile-per-CTA kernel, except for paged KV with more (request, kv head) pairs than one wave holds:
    // there the two-tiles-per-CTA kernel amortises the 2 KiB page boxes over twice the query rows (config 5:
    // 314 vs 416 us)
    const bool paged_multiwave = p->page_size > 0 && (int64_t)p->B * p->Hkv * 4 > sm_count();
    if (p->impl == 2 || (p->impl == 0 && paged_multiwave)) {
        pl.use_duo = attn_duo_supported(pl);
        D2SD_CHECK_SUPPORTED(pl.use_duo || p->impl != 2, "impl = 2 (two-tiles-per-CTA tcgen05 kernel) does not cover this shape");
    }
    if (!pl.use_duo && (p->impl == 3 || p->impl == 0)) {
        pl.use_stream = attn_stream_supported(pl);
        D2SD_CHECK_SUPPORTED(pl.use_stream || p->impl != 3, "impl = 3 (one-tile-per-CTA tcgen05 kernel) does not cover this shape");
    }
    const int rows = pl.T_cap * pl.G;
    const int max_ctx = p->max_ctx_len > 0 ? p->max_ctx_len : 1;
    int splits = p->num_splits;
    if (pl.use_duo) {
        // One CTA = (request, kv head, item, context chunk); an item is the M tiles (2i, 2i+1) or an odd last tile.
        // A duo item costs two softmax sub-unit rounds per key tile, a solo item one: its chunks are about half
        // as many.  One wave: chunk counts from the cost model; otherwise fixed chunks of 32 key tiles.
        const int n_mt = ceil_div(rows, 128);
        const int n_duo = n_mt / 2, odd = n_mt & 1;
        const int max_tiles = ceil_div(p->max_ctx_len, 128) + ceil_div(pl.T_cap, 128);
        const int64_t heads = (int64_t)pl.B * pl.Hkv;
        const int budget = (int)(sm_count() / (heads > 0 ? heads : 1));
        int ca = 1, cb = 1;
        pl.tps_min = 1;
        if (splits > 0) {
            ca = splits;
            cb = (splits + 1) / 2;
        } else if (budget >= n_duo + odd) {
            const double ua = 3600.0, ub = 1800.0, xa = 8000.0, xb = 5000.0;
            auto cost = [&](int c, double u, double x) { return ceil_div(max_tiles, c) * u + (c > 1 ? x : 0.0); };
            double best = 1e30;
            const int ca_max = n_duo ? (budget - odd) / n_duo : 1;
            for (int a2 = 1; a2 <= (n_duo ? ca_max : 1) && a2 <= 64; ++a2) {
                int b_room = odd ? budget - n_duo * a2 : 0;
                if (b_room > 64) b_room = 64;
                double tb = 0.0;
                int b_best = 1;
                if (odd) {
                    tb = 1e30;
                    for (int b2 = 1; b2 <= b_room; ++b2) {
                        const double t = cost(b2, ub, xb);
                        if (t < tb) { tb = t; b_best = b2; }
                    }
                }
                const double ta = n_duo ? cost(a2, ua, xa) : 0.0;
                const double t = ta > tb ? ta : tb;
                if (t < best) { best = t; ca = a2; cb = b_best; }
            }
        } else {
            ca = ceil_div(max_tiles, 32);
            cb = ceil_div(max_tiles, 64);
            pl.tps_min = -1;  // fixed below
        }
        if (ca > 64) ca = 64;
        if (cb > 64) cb = 64;
        if (ca > max_tiles) ca = max_tiles;  // never an always-empty chunk
        if (cb > max_tiles) cb = max_tiles;
        if (ca < 1) ca = 1;
        if (cb < 1) cb = 1;
        pl.last_merges = pl.tps_min < 0 && splits == 0;
        if (pl.tps_min < 0) pl.tps_min = ceil_div(max_tiles, n_duo ? ca : cb);
        pl.n_mt = n_mt;
        pl.n_pair = n_duo; pl.n_single = odd;
        pl.chunks_a = ca;
        pl.chunks_b = cb;
        pl.chunk_keys = 0;
        pl.num_splits = n_duo ? ca : cb;
        pl.NS = 0;
        pl.grp_rows = 256 * (ca > cb ? ca : cb);
        const size_t n_groups = (size_t)pl.B * pl.Hkv * (n_duo + odd);
        const size_t slot_rows = n_groups * pl.grp_rows;
        D2SD_CHECK_SUPPORTED(n_groups * 2 * sizeof(unsigned) <= kWsHeaderBytes - 16, "B*Hkv*items = %zu groups > %zu",
                             n_groups, (kWsHeaderBytes - 16) / (2 * sizeof(unsigned)));
        pl.off_cnt = 0;
        pl.cnt_bytes = kWsHeaderBytes;
        pl.off_o = pl.cnt_bytes;
        pl.off_lse = pl.off_o + align_up(slot_rows * pl.d * sizeof(float), 256);
        pl.bytes = pl.off_lse + align_up(slot_rows * sizeof(float), 256);
    } else if (pl.use_stream) {
        // One CTA = (request, kv head, M tile, context chunk).  M tiles (2p, 2p+1) over the same chunk form a
        // 2-CTA cluster that shares its key tiles; an odd last tile's chunks are paired without sharing.
        // One wave (enough SMs for every M tile of every (request, kv head)): the chunk counts are chosen
        // from a cost model (cycles per unit, fixed cost of the partial-state exchange) so that paired tiles
        // and the usually short last tile finish together; every request cuts its own key tiles evenly
        // (tps_min = 1).  Otherwise: fixed chunks of 32 key tiles, several waves.
        const int n_mt = ceil_div(rows, 128);
        const int n_pairs = n_mt / 2, odd = n_mt & 1;
        const int max_tiles = ceil_div(p->max_ctx_len, 128) + ceil_div(pl.T_cap, 128);
        const int64_t heads = (int64_t)pl.B * pl.Hkv;
        const int budget = (int)((sm_count() & ~1) / (heads > 0 ? heads : 1));
        int ca = 1, cb = 1;
        pl.tps_min = 1;
        if (splits >= 256) {  // test knob: (chunks_b << 8) | chunks_a
            ca = splits & 255;
            cb = splits >> 8;
        } else if (splits > 0) {
            ca = cb = splits;
        } else if (budget >= 2 * n_pairs + 2 * odd) {
            const int rows_last = rows - (n_mt - 1) * 128;
            const double ua = 1250.0, ub = (odd && rows_last <= 32) ? 1050.0 : 1250.0;
            const double xa = 3000.0, xb = 500.0 + 3000.0 * (odd ? rows_last : 128) / 128.0;
            auto cost = [&](int c, double u, double x) { return ceil_div(max_tiles, c) * u + (c > 1 ? x : 0.0); };
            double best = 1e30;
            const int ca_max = n_pairs ? (budget - 2 * odd) / (2 * n_pairs) : 1;
            for (int a2 = 1; a2 <= (n_pairs ? ca_max : 1) && a2 <= 64; ++a2) {
                int b_room = odd ? ((budget - 2 * n_pairs * a2) & ~1) : 0;
                if (b_room > 64) b_room = 64;
                double tb = 0.0;
                int b_best = 1;
                if (odd) {
                    tb = 1e30;
                    for (int b2 = 1; b2 <= b_room; ++b2) {
                        const double t = cost(b2, ub, xb);
                        if (t < tb) { tb = t; b_best = b2; }
                    }
                }
                const double ta = n_pairs ? cost(a2, ua, xa) : 0.0;
                const double t = ta > tb ? ta : tb;
                if (t < best) { best = t; ca = a2; cb = b_best; }
            }
        } else {
            ca = cb = ceil_div(max_tiles, 32);  // measured on config 5: 20 -> 497, 32 -> 486, 64 -> 500, 129 -> 572 us per step
            pl.tps_min = -1;  // fixed below
        }
        if (ca > 64) ca = 64;  // a group's CTAs wait for each other
        if (cb > 64) cb = 64;
        if (ca > max_tiles) ca = max_tiles;  // never an always-empty chunk
        if (cb > max_tiles) cb = max_tiles;
        if (ca < 1) ca = 1;
        if (cb < 1) cb = 1;
        pl.last_merges = pl.tps_min < 0 && splits == 0;
        if (pl.tps_min < 0) pl.tps_min = ceil_div(max_tiles, ca);
        pl.n_mt = n_mt;
        pl.n_pair = n_pairs; pl.n_single = odd;
        pl.chunks_a = ca;
        pl.chunks_b = cb;
        pl.chunk_keys = 0;
        pl.num_splits = n_pairs ? ca : cb;
        pl.NS = 0;
        pl.grp_rows = 128 * (ca > cb ? ca : cb);
        const size_t n_groups = (size_t)pl.B * pl.Hkv * n_mt;
        const size_t slot_rows = n_groups * pl.grp_rows;
        D2SD_CHECK_SUPPORTED(n_groups * 2 * sizeof(unsigned) <= kWsHeaderBytes - 16, "B*Hkv*tiles = %zu groups > %zu",
                             n_groups, (kWsHeaderBytes - 16) / (2 * sizeof(unsigned)));
        pl.off_cnt = 0;
        pl.cnt_bytes = kWsHeaderBytes;
        pl.off_o = pl.cnt_bytes;
        pl.off_lse = pl.off_o + align_up(slot_rows * pl.d * sizeof(float), 256);
        pl.bytes = pl.off_lse + align_up(slot_rows * sizeof(float), 256);
    } else {
        if (splits == 0) {
            // ~3 CTAs/SM of 64-row M blocks
            const int64_t per_split = (int64_t)pl.B * pl.Hkv * ceil_div(rows, 64);
            splits = (int)(3 * sm_count() / (per_split > 0 ? per_split : 1));
            if (splits < 1) splits = 1;
            // never cut below 128 keys per chunk: the partial state would outweigh the KV it covers
            const int max_splits = (max_ctx + 127) / 128;
            if (splits > max_splits) splits = max_splits;
            if (splits > 64) splits = 64;
        }
        pl.chunk_keys = (ceil_div(max_ctx, splits) + 63) / 64 * 64;
        pl.num_splits = ceil_div(max_ctx, pl.chunk_keys);
        pl.NS = pl.num_splits + 1;
        const size_t rows_all = (size_t)pl.B * pl.NS * pl.T_cap * pl.Hq;
        pl.off_cnt = 0;
        pl.cnt_bytes = kWsHeaderBytes;  // unused by these kernels, but never overwritten either
        pl.off_o = pl.cnt_bytes;
        pl.off_lse = pl.off_o + align_up(rows_all * pl.d * sizeof(float), 256);
        pl.bytes = pl.off_lse + align_up(rows_all * sizeof(float), 256);
    }
    *out = pl;
    return D2SD_OK;
}

}  // namespace d2sd

using namespace d2sd;

extern "C" {

const char* d2sd_last_error(void) { return g_err; }
const char* d2sd_version(void) { return "d2sd 0.1 sm_100a"; }

int32_t d2sd_select_prefixes(const float* conf, int32_t B, int32_t gamma, int32_t K, int32_t* prefix_len,
                             double* r_out, void* stream) {
    clear_error();
    if (int32_t st = check_block(B, gamma, K)) return st;
    D2SD_CHECK_ARG(B == 0 || conf != nullptr, "conf is NULL");
    D2SD_CHECK_ARG(B == 0 || K == 0 || prefix_len != nullptr, "prefix_len is NULL");
    return launch_select(conf, B, gamma, K, prefix_len, r_out, static_cast<cudaStream_t>(stream));
}

int32_t d2sd_build_tree(const int32_t* draft1, const int32_t* draft2, const int32_t* prefix_len,
                        const int32_t* ctx_len, int32_t B, int32_t gamma, int32_t K, int32_t T_cap,
                        int32_t* tokens, int32_t* parent, int32_t* depth, int32_t* pos_id,
                        int32_t* branch_off, uint32_t* mask, int32_t* tree_len, void* stream) {
    clear_error();
    if (int32_t st = check_block(B, gamma, K)) return st;
    const int need = gamma + K * (gamma - 1) - K * (K - 1) / 2;
    D2SD_CHECK_ARG(T_cap >= need, "T_cap = %d < largest tree %d for gamma = %d, K = %d", T_cap, need, gamma, K);
    D2SD_CHECK_SUPPORTED(T_cap <= 1024, "T_cap = %d > 1024", T_cap);
    if (B == 0) return D2SD_OK;
    D2SD_CHECK_ARG(draft1 && ctx_len && tokens && parent && depth && pos_id && branch_off && mask && tree_len,
                   "a required buffer is NULL");
    D2SD_CHECK_ARG(K == 0 || (draft2 && prefix_len), "draft2 / prefix_len is NULL with K = %d", K);
    return launch_build_tree(draft1, draft2, prefix_len, ctx_len, B, gamma, K, T_cap, tokens, parent, depth,
                             pos_id, branch_off, mask, tree_len, static_cast<cudaStream_t>(stream));
}

size_t d2sd_cascade_workspace_bytes(const d2sd_attn_params* p) {
    clear_error();
    AttnPlan pl;
    if (make_plan(p, &pl) != D2SD_OK) return 0;
    return pl.bytes;
}

int32_t d2sd_cascade_verify_attn(const d2sd_attn_params* p, const void* q, const void* k_cache,
                                 const void* v_cache, const int32_t* kv_indptr, const int32_t* kv_indices,
                                 const int32_t* ctx_len, const void* tree_k, const void* tree_v,
                                 const uint32_t* mask, const int32_t* tree_len, void* out, float* lse,
                                 float* dbg_state, void* workspace, size_t workspace_bytes, void* stream) {
    clear_error();
    AttnPlan pl;
    if (int32_t st = make_plan(p, &pl)) return st;
    if (pl.B == 0) return D2SD_OK;
    D2SD_CHECK_ARG(q && ctx_len && tree_k && tree_v && mask && tree_len && out, "a required buffer is NULL");
    D2SD_CHECK_ARG(p->max_ctx_len == 0 || (k_cache && v_cache), "k_cache / v_cache is NULL");
    D2SD_CHECK_ARG(p->max_ctx_len == 0 || p->kv_rows > 0, "max_ctx_len = %d but kv_rows = 0", p->max_ctx_len);
    D2SD_CHECK_ARG(p->page_size == 0 || p->kv_rows % p->page_size == 0, "kv_rows = %lld is not a whole number of pages",
                   (long long)p->kv_rows);
    D2SD_CHECK_ARG(kv_indptr != nullptr || (pl.B == 1 && pl.page_size == 0),
                   "kv_indptr may be NULL only for B == 1 contiguous KV");
    D2SD_CHECK_ARG((pl.page_size > 0) == (kv_indices != nullptr),
                   "kv_indices must be given exactly when page_size > 0");
    const uintptr_t al = reinterpret_cast<uintptr_t>(q) | reinterpret_cast<uintptr_t>(k_cache) |
                         reinterpret_cast<uintptr_t>(v_cache) | reinterpret_cast<uintptr_t>(tree_k) |
                         reinterpret_cast<uintptr_t>(tree_v) | reinterpret_cast<uintptr_t>(out);
    D2SD_CHECK_ARG((al & 15) == 0, "q/k_cache/v_cache/tree_k/tree_v/out must be 16-byte aligned");
    if (workspace == nullptr || workspace_bytes < pl.bytes || (reinterpret_cast<uintptr_t>(workspace) & 255))
        return set_error(D2SD_ERR_WORKSPACE, "workspace %p with %zu bytes; need %zu bytes, 256-byte aligned",
                         workspace, workspace_bytes, pl.bytes);
    AttnArgs a{};
    a.q = static_cast<const __nv_bfloat16*>(q);
    a.k_cache = static_cast<const __nv_bfloat16*>(k_cache);
    a.v_cache = static_cast<const __nv_bfloat16*>(v_cache);
    a.tree_k = static_cast<const __nv_bfloat16*>(tree_k);
    a.tree_v = static_cast<const __nv_bfloat16*>(tree_v);
    a.kv_indptr = kv_indptr; a.kv_indices = kv_indices; a.ctx_len = ctx_len; a.tree_len = tree_len;
    a.mask = mask;
    a.out = static_cast<__nv_bfloat16*>(out);
    a.lse = lse; a.dbg_state = dbg_state;
    a.part_o = reinterpret_cast<float*>(static_cast<char*>(workspace) + pl.off_o);
    a.part_lse = reinterpret_cast<float*>(static_cast<char*>(workspace) + pl.off_lse);
    a.part_o16 = reinterpret_cast<__nv_bfloat16*>(static_cast<char*>(workspace) + pl.off_o);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int phases = p->phases ? p->phases : 7;
    const bool do_prefix = phases & 1, do_tree = phases & 2, do_merge = phases & 4;
    if (pl.use_stream || pl.use_duo) {
        auto launch_attn_stream = [&](const AttnPlan& pl_, const AttnArgs& a_, int mode_, float* dbg_, cudaStream_t s_) {
            return pl_.use_duo ? launch_attn_duo(pl_, a_, mode_, dbg_, s_) : d2sd::launch_attn_stream(pl_, a_, mode_, dbg_, s_);
        };
        a.counters = reinterpret_cast<unsigned*>(static_cast<char*>(workspace) + pl.off_cnt);
        if (dbg_state) {
            const size_t half = (size_t)pl.B * pl.T_cap * pl.Hq * (pl.d + 1);
            if (int32_t st = launch_attn_stream(pl, a, 1, dbg_state, s)) return st;
            if (int32_t st = launch_attn_stream(pl, a, 2, dbg_state + half, s)) return st;
        }
        const int mode = phases & 3;
        if (mode == 0) return D2SD_OK;
        return launch_attn_stream(pl, a, mode, nullptr, s);
    }
    if (do_prefix || do_tree)
        if (int32_t st = launch_attn_mma(pl, a, do_prefix, do_tree, s)) return st;
    if (do_merge) return launch_attn_merge(pl, a, s);
    return D2SD_OK;
}

int32_t d2sd_cascade_workspace_init(const d2sd_attn_params* p, void* workspace, size_t workspace_bytes,
                                    void* stream) {
    clear_error();
    AttnPlan pl;
    if (int32_t st = make_plan(p, &pl)) return st;
    if (workspace == nullptr || workspace_bytes < pl.bytes || (reinterpret_cast<uintptr_t>(workspace) & 255))
        return set_error(D2SD_ERR_WORKSPACE, "workspace %p with %zu bytes; need %zu bytes, 256-byte aligned",
                         workspace, workspace_bytes, pl.bytes);
    if (pl.cnt_bytes)
        D2SD_CHECK_CUDA(cudaMemsetAsync(static_cast<char*>(workspace) + pl.off_cnt, 0, pl.cnt_bytes,
                                        static_cast<cudaStream_t>(stream)));
    return D2SD_OK;
}

size_t d2sd_accept_workspace_bytes(int32_t B, int32_t T_cap, int32_t V) {
    if (B < 0 || T_cap < 1 || V < 1) return 0;
    return align_up((size_t)B * T_cap * ceil_div(V, kScanChunk) * kScanPartBytes, 256) + 256;
}

int32_t d2sd_accept(const void* logits, int64_t row_stride, int32_t V, const int32_t* tokens,
                    const int32_t* parent, const int32_t* depth, const int32_t* tree_len, int32_t B,
                    int32_t gamma, int32_t T_cap, int32_t* argmax_out, int32_t* accept_len, int32_t* path,
                    int32_t* bonus, int32_t* best_node, void* workspace, size_t workspace_bytes,
                    void* stream) {
    clear_error();
    D2SD_CHECK_ARG(B >= 0 && V >= 1 && row_stride >= V, "B = %d, V = %d, row_stride = %lld", B, V,
                   (long long)row_stride);
    D2SD_CHECK_ARG(gamma >= 2 && gamma <= 64, "gamma = %d outside [2,64]", gamma);
    D2SD_CHECK_ARG(T_cap >= 1, "T_cap = %d", T_cap);
    D2SD_CHECK_SUPPORTED(T_cap <= 1024, "T_cap = %d > 1024", T_cap);
    D2SD_CHECK_SUPPORTED(ceil_div(V, kScanChunk) <= 65535, "V = %d too large", V);
    if (B == 0) return D2SD_OK;
    D2SD_CHECK_ARG(logits && tokens && parent && depth && tree_len && argmax_out && accept_len && path &&
                       bonus && best_node,
                   "a required buffer is NULL");
    if (workspace == nullptr || workspace_bytes < d2sd_accept_workspace_bytes(B, T_cap, V) ||
        (reinterpret_cast<uintptr_t>(workspace) & 15))
        return set_error(D2SD_ERR_WORKSPACE, "accept workspace %p with %zu bytes; need %zu, 16-byte aligned",
                         workspace, workspace_bytes, d2sd_accept_workspace_bytes(B, T_cap, V));
    return launch_accept(static_cast<const __nv_bfloat16*>(logits), row_stride, V, tokens, parent, depth,
                         tree_len, B, gamma, T_cap, argmax_out, accept_len, path, bonus, best_node, workspace,
                         static_cast<cudaStream_t>(stream));
}

size_t d2sd_confidence_workspace_bytes(int32_t B, int32_t gamma, int32_t V) {
    if (B < 0 || gamma < 2 || V < 1) return 0;
    return align_up((size_t)B * (gamma - 1) * ceil_div(V, kScanChunk) * kScanPartBytes, 256) + 256;
}

int32_t d2sd_draft_confidence(const void* logits, int64_t row_stride, int32_t V, const int32_t* anchor,
                              int32_t B, int32_t gamma, int32_t* draft, float* conf, void* workspace,
                              size_t workspace_bytes, void* stream) {
    clear_error();
    D2SD_CHECK_ARG(B >= 0 && V >= 1 && row_stride >= V, "B = %d, V = %d, row_stride = %lld", B, V,
                   (long long)row_stride);
    D2SD_CHECK_ARG(gamma >= 2 && gamma <= 64, "gamma = %d outside [2,64]", gamma);
    D2SD_CHECK_SUPPORTED(ceil_div(V, kScanChunk) <= 65535, "V = %d too large", V);
    if (B == 0) return D2SD_OK;
    D2SD_CHECK_ARG(logits && anchor && draft && conf, "a required buffer is NULL");
    if (workspace == nullptr || workspace_bytes < d2sd_confidence_workspace_bytes(B, gamma, V) ||
        (reinterpret_cast<uintptr_t>(workspace) & 15))
        return set_error(D2SD_ERR_WORKSPACE, "confidence workspace %p with %zu bytes; need %zu, 16-byte aligned",
                         workspace, workspace_bytes, d2sd_confidence_workspace_bytes(B, gamma, V));
    return launch_confidence(static_cast<const __nv_bfloat16*>(logits), row_stride, V, anchor, B, gamma, draft, conf,
                             workspace, static_cast<cudaStream_t>(stream));
}

size_t d2sd_commit_workspace_bytes(int32_t B) {
    if (B < 0) return 0;
    return align_up((size_t)(B + 1) * sizeof(int32_t), 256);
}

int32_t d2sd_commit_kv(const d2sd_commit_params* p, const void* tree_k, const void* tree_v, const int32_t* path,
                       const int32_t* accept_len, const int32_t* ctx_len, void* k_cache, void* v_cache,
                       const int32_t* kv_indptr, int32_t* kv_indices, const int32_t* free_pages, int32_t n_free,
                       int32_t* free_head, int32_t* ctx_len_out, int32_t* dropped, const void* feat, void* feat_out,
                       void* workspace, size_t workspace_bytes, void* stream) {
    clear_error();
    D2SD_CHECK_ARG(p != nullptr, "params is NULL");
    D2SD_CHECK_ARG(p->B >= 0 && p->T_cap >= 1 && p->Hkv >= 1 && p->d >= 1 && p->n_layers >= 0,
                   "B = %d, T_cap = %d, Hkv = %d, d = %d, n_layers = %d", p->B, p->T_cap, p->Hkv, p->d, p->n_layers);
    D2SD_CHECK_ARG(p->gamma >= 2 && p->gamma <= 64, "gamma = %d outside [2,64]", p->gamma);
    D2SD_CHECK_ARG(p->page_size >= 0 && p->kv_rows >= 0 && p->F >= 0, "page_size = %d, kv_rows = %lld, F = %d",
                   p->page_size, (long long)p->kv_rows, p->F);
    D2SD_CHECK_SUPPORTED(p->B <= 65535 && p->n_layers <= 65535, "B = %d / n_layers = %d > 65535", p->B, p->n_layers);
    const int64_t row_elems = (int64_t)p->Hkv * p->d;
    D2SD_CHECK_SUPPORTED(row_elems % 8 == 0 && p->F % 8 == 0, "Hkv*d = %lld and F = %d must be multiples of 8",
                         (long long)row_elems, p->F);
    D2SD_CHECK_ARG(p->tree_layer_stride >= (int64_t)p->B * p->T_cap * row_elems && p->tree_layer_stride % 8 == 0,
                   "tree_layer_stride = %lld", (long long)p->tree_layer_stride);
    D2SD_CHECK_ARG(p->cache_layer_stride >= p->kv_rows * row_elems && p->cache_layer_stride % 8 == 0,
                   "cache_layer_stride = %lld", (long long)p->cache_layer_stride);
    if (p->B == 0 || p->n_layers == 0) return D2SD_OK;
    D2SD_CHECK_ARG(tree_k && tree_v && path && accept_len && ctx_len && k_cache && v_cache && ctx_len_out && dropped,
                   "a required buffer is NULL");
    D2SD_CHECK_ARG(kv_indptr != nullptr || (p->B == 1 && p->page_size == 0),
                   "kv_indptr may be NULL only for B == 1 contiguous KV");
    D2SD_CHECK_ARG((p->page_size > 0) == (kv_indices != nullptr), "kv_indices must be given exactly when page_size > 0");
    D2SD_CHECK_ARG((free_pages != nullptr) == (free_head != nullptr) && n_free >= 0 && (free_pages || n_free == 0),
                   "free_pages / free_head must be given together (n_free = %d)", n_free);
    D2SD_CHECK_ARG(free_pages == nullptr || p->page_size > 0, "a free list needs paged KV");
    D2SD_CHECK_ARG((feat != nullptr) == (feat_out != nullptr) && ((feat != nullptr) == (p->F > 0)),
                   "feat / feat_out / F must be given together");
    const uintptr_t al = reinterpret_cast<uintptr_t>(tree_k) | reinterpret_cast<uintptr_t>(tree_v) |
                         reinterpret_cast<uintptr_t>(k_cache) | reinterpret_cast<uintptr_t>(v_cache) |
                         reinterpret_cast<uintptr_t>(feat) | reinterpret_cast<uintptr_t>(feat_out);
    D2SD_CHECK_ARG((al & 15) == 0, "tree_k/tree_v/k_cache/v_cache/feat/feat_out must be 16-byte aligned");
    if (workspace == nullptr || workspace_bytes < d2sd_commit_workspace_bytes(p->B) ||
        (reinterpret_cast<uintptr_t>(workspace) & 15))
        return set_error(D2SD_ERR_WORKSPACE, "commit workspace %p with %zu bytes; need %zu, 16-byte aligned", workspace,
                         workspace_bytes, d2sd_commit_workspace_bytes(p->B));
    CommitArgs a{};
    a.tree_k = static_cast<const __nv_bfloat16*>(tree_k);
    a.tree_v = static_cast<const __nv_bfloat16*>(tree_v);
    a.tree_layer_stride = p->tree_layer_stride;
    a.path = path; a.accept_len = accept_len; a.ctx_len = ctx_len;
    a.k_cache = static_cast<__nv_bfloat16*>(k_cache);
    a.v_cache = static_cast<__nv_bfloat16*>(v_cache);
    a.cache_layer_stride = p->cache_layer_stride; a.kv_rows = p->kv_rows;
    a.kv_indptr = kv_indptr; a.kv_indices = kv_indices; a.page_size = p->page_size;
    a.free_pages = free_pages; a.n_free = n_free; a.free_head = free_head;
    a.B = p->B; a.gamma = p->gamma; a.T_cap = p->T_cap; a.Hkv = p->Hkv; a.d = p->d; a.n_layers = p->n_layers;
    a.ctx_len_out = ctx_len_out; a.dropped = dropped;
    a.feat = static_cast<const __nv_bfloat16*>(feat);
    a.feat_out = static_cast<__nv_bfloat16*>(feat_out);
    a.F = p->F;
    a.n_fit = static_cast<int32_t*>(workspace);
    return launch_commit_kv(a, static_cast<cudaStream_t>(stream));
}

int32_t d2sd_select_third(const float* conf2, const int32_t* prefix_len, int32_t B, int32_t gamma, int32_t K,
                          int32_t* third_len, double* r3_out, void* stream) {
    clear_error();
    if (int32_t st = check_block(B, gamma, K)) return st;
    if (B == 0 || K == 0) return D2SD_OK;
    D2SD_CHECK_ARG(conf2 && prefix_len && third_len, "a required buffer is NULL");
    return launch_select_third(conf2, prefix_len, B, gamma, K, third_len, r3_out, static_cast<cudaStream_t>(stream));
}

int32_t d2sd_build_tree3(const int32_t* draft1, const int32_t* draft2, const int32_t* draft3,
                         const int32_t* prefix_len, const int32_t* third_len, const int32_t* ctx_len, int32_t B,
                         int32_t gamma, int32_t K, int32_t T_cap, int32_t* tokens, int32_t* parent, int32_t* depth,
                         int32_t* pos_id, int32_t* branch_off, uint32_t* mask, int32_t* tree_len, void* stream) {
    clear_error();
    if (int32_t st = check_block(B, gamma, K)) return st;
    const int need = gamma + K * (gamma - 1) - K * (K - 1) / 2 + K * (gamma - 2) - K * (K - 1) / 2;
    D2SD_CHECK_ARG(T_cap >= need, "T_cap = %d < largest depth-3 tree %d for gamma = %d, K = %d", T_cap, need, gamma, K);
    D2SD_CHECK_SUPPORTED(T_cap <= 1024, "T_cap = %d > 1024", T_cap);
    if (B == 0) return D2SD_OK;
    D2SD_CHECK_ARG(draft1 && ctx_len && tokens && parent && depth && pos_id && branch_off && mask && tree_len,
                   "a required buffer is NULL");
    D2SD_CHECK_ARG(K == 0 || (draft2 && draft3 && prefix_len && third_len), "draft2 / draft3 / prefix_len / third_len is NULL with K = %d", K);
    return launch_build_tree3(draft1, draft2, draft3, prefix_len, third_len, ctx_len, B, gamma, K, T_cap, tokens, parent,
                              depth, pos_id, branch_off, mask, tree_len, static_cast<cudaStream_t>(stream));
}

}  // extern "C"
