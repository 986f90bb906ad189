// Shared host/device helpers of libd2sd (CUDA side only; the CPU oracle shares nothing with this).
#pragma once

#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdint>
#include <cstdio>

#include "d2sd.h"

namespace d2sd {

// Thread-local last-error text behind d2sd_last_error().
int32_t set_error(int32_t status, const char* fmt, ...);
void clear_error();

#define D2SD_CHECK_ARG(cond, ...)                                         \
    do {                                                                  \
        if (!(cond)) return ::d2sd::set_error(D2SD_ERR_INVALID_ARG, __VA_ARGS__); \
    } while (0)

#define D2SD_CHECK_SUPPORTED(cond, ...)                                   \
    do {                                                                  \
        if (!(cond)) return ::d2sd::set_error(D2SD_ERR_UNSUPPORTED, __VA_ARGS__); \
    } while (0)

#define D2SD_CHECK_CUDA(expr)                                                                  \
    do {                                                                                       \
        cudaError_t _e = (expr);                                                               \
        if (_e != cudaSuccess)                                                                 \
            return ::d2sd::set_error(D2SD_ERR_CUDA, "%s failed: %s", #expr, cudaGetErrorString(_e)); \
    } while (0)

// Launch check that is legal during stream capture (no synchronisation).
#define D2SD_CHECK_LAUNCH(name)                                                                \
    do {                                                                                       \
        cudaError_t _e = cudaPeekAtLastError();                                                \
        if (_e != cudaSuccess) {                                                               \
            (void)cudaGetLastError();                                                          \
            return ::d2sd::set_error(D2SD_ERR_CUDA, "launch of %s failed: %s", name,           \
                                     cudaGetErrorString(_e));                                  \
        }                                                                                      \
    } while (0)

inline int ceil_div(int a, int b) { return (a + b - 1) / b; }
inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

int sm_count();  // multiprocessor count of the current device (cached per device)
// True exactly once per device and call site (per-device function attributes such as the dynamic shared
// memory opt-in); a race between two first callers only repeats an idempotent call.
inline bool first_use_on_device(unsigned long long& done_mask) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return true;
    if ((done_mask >> dev) & 1ull) return false;
    done_mask |= 1ull << dev;
    return true;
}
constexpr size_t kWsHeaderBytes = 1u << 20;  // fixed-size head of the attention workspace (group counters)
constexpr unsigned kWsErrorWord = (1u << 20) / 4 - 2;  // uint32 index in the header: set when a group wait gave up

// ---- stage launchers (defined in the per-stage .cu files) -------------------------------------
int32_t launch_select(const float* conf, int B, int gamma, int K, int32_t* prefix_len, double* r_out,
                      cudaStream_t s);
int32_t launch_build_tree(const int32_t* draft1, const int32_t* draft2, const int32_t* prefix_len,
                          const int32_t* ctx_len, int B, int gamma, int K, int T_cap, int32_t* tokens,
                          int32_t* parent, int32_t* depth, int32_t* pos_id, int32_t* branch_off,
                          uint32_t* mask, int32_t* tree_len, cudaStream_t s);

constexpr int kScanChunk = 16384;  // vocabulary elements scanned per CTA (accept.cu)
constexpr size_t kScanPartBytes = 16;
int32_t launch_accept(const __nv_bfloat16* logits, int64_t row_stride, int V, const int32_t* tokens,
                      const int32_t* parent, const int32_t* depth, const int32_t* tree_len, int B,
                      int gamma, int T_cap, int32_t* argmax_out, int32_t* accept_len, int32_t* path,
                      int32_t* bonus, int32_t* best_node, void* workspace, cudaStream_t s);
int32_t launch_confidence(const __nv_bfloat16* logits, int64_t row_stride, int V, const int32_t* anchor, int B,
                          int gamma, int32_t* draft, float* conf, void* workspace, cudaStream_t s);
int32_t launch_select_third(const float* conf2, const int32_t* prefix_len, int B, int gamma, int K,
                            int32_t* third_len, double* r3_out, cudaStream_t s);
int32_t launch_build_tree3(const int32_t* draft1, const int32_t* draft2, const int32_t* draft3,
                           const int32_t* prefix_len, const int32_t* third_len, const int32_t* ctx_len, int B,
                           int gamma, int K, int T_cap, int32_t* tokens, int32_t* parent, int32_t* depth,
                           int32_t* pos_id, int32_t* branch_off, uint32_t* mask, int32_t* tree_len, cudaStream_t s);
struct CommitArgs {
    const __nv_bfloat16 *tree_k, *tree_v;
    int64_t tree_layer_stride;  // elements
    const int32_t *path, *accept_len, *ctx_len;
    __nv_bfloat16 *k_cache, *v_cache;
    int64_t cache_layer_stride, kv_rows;
    const int32_t* kv_indptr;
    int32_t* kv_indices;
    int page_size;
    const int32_t* free_pages;
    int n_free;
    int32_t* free_head;
    int B, gamma, T_cap, Hkv, d, n_layers;
    int32_t *ctx_len_out, *dropped;
    const __nv_bfloat16* feat;  // optional [B,T_cap,F]
    __nv_bfloat16* feat_out;    // optional [B,gamma,F]
    int F;
    int32_t* n_fit;             // workspace [B]
};
int32_t launch_commit_kv(const CommitArgs& a, cudaStream_t s);

// Partial softmax states in the workspace.
//  mma.sync path ("row layout"): O fp32 [B][NS][T_cap][Hq][d], LSE fp32 [B][NS][T_cap][Hq]; slots
//    0..num_splits-1 are the prefix chunks, slot num_splits is the tree pass.
//  tcgen05 kernels (attn_stream_sm100.cu, attn_duo_sm100.cu): a fixed 1 MiB header of self-resetting group
//    counters (zero between calls) and the error word, then partials per group (request, kv head, M tile or
//    item): O bf16 [group][grp_rows][d] and one fp32 [group][grp_rows]; chunk c of a group holds its rows at
//    c*128.. (one tile per CTA) or c*256.. (two tiles per CTA); the tree keys are key tiles of the same kernel.
//    Two tiles per CTA: O normalised, the fp32 is the row's LSE.  One tile per CTA: O UNNORMALISED relative to the
//    row's final reference maximum, the fp32 is that reference in log2 units, and the row sums (fp32
//    [group][grp_rows]) sit behind the bf16 rows inside the O region (which is sized for fp32 rows).
struct AttnPlan {
    int B, T_cap, W, Hq, Hkv, G, d;
    float sm_scale;
    int page_size;
    int max_ctx_len;
    int64_t kv_rows;
    int num_splits;   // prefix chunks
    int chunk_keys;   // mma.sync path: keys per chunk (multiple of 64); tcgen05 cuts whole key tiles on device
    int NS;           // row layout: num_splits + 1
    // tcgen05: the query rows (T*G) of one kv head are cut into 128-row M tiles; tiles (2p, 2p+1) form a pair
    // (a sharing cluster or a duo item), an odd last tile stands alone.  The kinds get their own chunk counts.
    int n_mt;                // 128-row query tiles per (request, kv head), from T_cap
    bool last_merges;        // several waves: the last CTA of a group to arrive merges it (nobody waits)
    bool use_duo;            // the two-tiles-per-CTA sub-unit kernel (attn_duo_sm100.cu): n_pair duo items, n_single solo item
    bool use_stream;         // the one-tile-per-CTA kernel (attn_stream_sm100.cu): chunks_a per paired tile, chunks_b for an odd last tile
    int n_pair, n_single;    // items per (request, kv head), from T_cap
    int chunks_a, chunks_b;  // CTAs (context chunks) per pair item / per single item
    int tps_min;             // a chunk never holds fewer key tiles than this (unless the request ends)
    int grp_rows;            // partial-state rows per group: rows per chunk x max(chunks_a, chunks_b)
    size_t off_cnt, cnt_bytes, off_o, off_lse, bytes;
};

struct AttnArgs {
    const __nv_bfloat16 *q, *k_cache, *v_cache, *tree_k, *tree_v;
    const int32_t *kv_indptr, *kv_indices, *ctx_len, *tree_len;
    const uint32_t* mask;
    __nv_bfloat16* out;
    float *lse, *dbg_state;
    float *part_o, *part_lse;
    __nv_bfloat16* part_o16;  // one-tile-per-CTA kernel: partial O rows in bf16
    unsigned* counters;  // tcgen05 path only: [group][2] arrivals / done
};

int32_t launch_attn_mma(const AttnPlan& pl, const AttnArgs& a, bool do_prefix, bool do_tree,
                        cudaStream_t s);
int32_t launch_attn_merge(const AttnPlan& pl, const AttnArgs& a, cudaStream_t s);
// mode: bit 0 = prefix tiles, bit 1 = tree tiles; dbg_rows: fp32 [B][T_cap][Hq][d+1] instead of out/lse
int32_t launch_attn_stream(const AttnPlan& pl, const AttnArgs& a, int mode, float* dbg_rows, cudaStream_t s);
bool attn_stream_supported(const AttnPlan& pl);
int32_t launch_attn_duo(const AttnPlan& pl, const AttnArgs& a, int mode, float* dbg_rows, cudaStream_t s);
bool attn_duo_supported(const AttnPlan& pl);

}  // namespace d2sd
