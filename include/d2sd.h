/*
 * d2sd.h -- C ABI of libd2sd: the verification hot path of a D2SD decoding step on B200 (sm_100a).
 *
 * Paper: "D2SD: Accelerating Speculative Decoding with Dual Diffusion Draft Models"
 * (arXiv 2606.04446; citations below are PAPER.md line numbers + section/equation).
 * One decoding cycle (Section 3.3) runs, between the caller's model forwards:
 *
 *   d2sd_select_prefixes      (ii)  top-K unmask: r(i), Eq. 4 (:93), S = Top-K r(i), Eq. 5 (:105)
 *   d2sd_build_tree           (iii)->(iv) the K+1 shared-prefix candidates (:107, :123-124) as one
 *                             flattened token tree with a bit-packed ancestor mask
 *   d2sd_cascade_verify_attn  (iv)  joint verification attention, "cascade attention" (:52, :124,
 *                             :154): shared committed prefix attended once for all tree queries,
 *                             tree-local pass under the ancestor mask, log-sum-exp merge
 *   d2sd_accept               (iv)  "longest-accepted-prefix search across branches" + bonus token
 *                             (:124, :69)
 *
 * Conventions
 *  - Every pointer is a DEVICE pointer unless its comment says "host".  The library never
 *    allocates, never synchronises and never reads device data on the host: every call only
 *    enqueues kernels on `stream` (a cudaStream_t passed as void*; NULL = legacy default stream)
 *    and is CUDA-graph capturable.  Data-dependent sizes (tree_len, ctx_len) stay on the device.
 *  - Ownership: the caller owns every buffer; the library borrows the pointers until the enqueued
 *    work has finished.  Outputs are fully overwritten unless stated otherwise.
 *  - Return value: D2SD_OK (0) or a negative d2sd_status; d2sd_last_error() gives a static,
 *    thread-local message for the most recent failure.  Argument errors are detected before
 *    anything is enqueued.
 *  - bf16 tensors are passed as `const void*` (2 bytes per element, IEEE bfloat16).
 *  - Notation: gamma = block size (position 0 is the anchor / bonus token, :69, :121); K = number
 *    of re-anchored branches; T_cap = capacity of the flattened tree (>= gamma + sum of branch
 *    lengths; the largest possible tree is gamma + K(gamma-1) - K(K-1)/2); W = ceil(T_cap/32) mask
 *    words per row; Hq/Hkv query/KV heads, G = Hq/Hkv; d head dimension; B requests.
 */
#ifndef D2SD_H_
#define D2SD_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum d2sd_status {
    D2SD_OK = 0,
    D2SD_ERR_INVALID_ARG = -1, /* NULL where a buffer is required, negative size, K > gamma-1 ... */
    D2SD_ERR_UNSUPPORTED = -2, /* shape outside the built specialisations (see each call)        */
    D2SD_ERR_WORKSPACE = -3,   /* workspace too small or misaligned                              */
    D2SD_ERR_CUDA = -4         /* a CUDA runtime / driver call failed (message has the detail)   */
} d2sd_status;

/* Static description of the last error on the calling thread ("" if none). Never NULL. */
const char* d2sd_last_error(void);

/* Library version string, e.g. "d2sd 0.1 sm_100a". */
const char* d2sd_version(void);

/* ---------------------------------------------------------------------------------------------
 * (a) Confidence-guided boundary selection.  PAPER.md:87-105, Eq. 3-5.
 *   P_0 = 1, P_i = c_1*...*c_i ;  r(i) = P_i * (1 - c_{i+1}),  i = 0..gamma-2 ;  S = Top-K_i r(i).
 * Arithmetic: confidences widened to fp64; the product is taken left to right with one rounding
 * per multiply, then one subtract and one multiply per r(i), no FMA contraction -- the same
 * operation order as the oracle, hence bit-identical r and a bit-exact selection.
 * Ties (real: any c_k = 1 gives r = 0 exactly) go to the smaller i; S is emitted ascending.
 *   conf        [B,gamma] fp32, conf[b,k] = c_k of Eq. 3; slot 0 (the anchor) is ignored
 *   prefix_len  out [B,K] int32, ascending, each in [0,gamma-2]
 *   r_out       out [B,gamma-1] fp64, or NULL
 * Requires 2 <= gamma <= 64, 0 <= K <= gamma-1 (else D2SD_ERR_INVALID_ARG), B >= 0.
 * Confidences outside [0,1] or NaN: behaviour unspecified.
 * ------------------------------------------------------------------------------------------- */
int32_t d2sd_select_prefixes(const float* conf, int32_t B, int32_t gamma, int32_t K,
                             int32_t* prefix_len, double* r_out, void* stream);

/* ---------------------------------------------------------------------------------------------
 * (b) Shared-prefix tree build.  PAPER.md:107, :123-124.
 * Branch k (k-th smallest selected prefix length i_k) keeps the anchor and the first i_k draft-1
 * tokens and re-drafts positions i_k+1..gamma-1 (:107).  Flattened layout: nodes 0..gamma-1 are
 * the draft-1 block (node 0 = anchor = root, parent[j] = j-1, depth[j] = j); branch k appends
 * gamma-1-i_k nodes holding draft2[b,k,i_k+1..gamma-1] at offset branch_off[b,k]; its first node's
 * parent is trunk node i_k, the rest chain.  depth = block position; pos_id = ctx_len + depth.
 * Ancestor mask: bit (a%32) of word a/32 of row n is 1 iff a == n or a is an ancestor of n.
 *   draft1      [B,gamma] int32        draft2  [B,K,gamma] int32 (only [i_k+1..gamma-1] is read)
 *   prefix_len  [B,K] int32 distinct, ascending, in [0,gamma-2] (as produced by (a))
 *   ctx_len     [B] int32 committed KV length L_b
 *   tokens, parent, depth, pos_id  out [B,T_cap] int32; rows n >= tree_len[b]: tokens = parent = -1,
 *               depth = pos_id = 0
 *   branch_off  out [B,K+1] int32 (branch_off[b,K] = tree_len[b])
 *   mask        out [B,T_cap,W] uint32, padding rows and padding bits 0
 *   tree_len    out [B] int32 = gamma + sum_k (gamma-1-i_k)
 * Requires 2 <= gamma <= 64, 0 <= K <= gamma-1, T_cap >= gamma + K(gamma-1) - K(K-1)/2,
 * T_cap <= 1024 (else D2SD_ERR_UNSUPPORTED).
 * ------------------------------------------------------------------------------------------- */
int32_t d2sd_build_tree(const int32_t* draft1, const int32_t* draft2, const int32_t* prefix_len,
                        const int32_t* ctx_len, int32_t B, int32_t gamma, int32_t K, int32_t T_cap,
                        int32_t* tokens, int32_t* parent, int32_t* depth, int32_t* pos_id,
                        int32_t* branch_off, uint32_t* mask, int32_t* tree_len, void* stream);

/* ---------------------------------------------------------------------------------------------
 * (c) Cascade tree-verify attention.  PAPER.md:52, :124, :154.
 * For request b, node t < tree_len[b], head h (kv head g = h / G):
 *   key set = { committed prefix j in [0, ctx_len[b]) }  U  { tree node a : mask[b,t] bit a }
 *   out[b,t,h,:] = softmax_j(sm_scale * q.k_j) . v_j      lse[b,t,h] = ln sum_j exp(sm_scale * q.k_j)
 * computed as a cascade: all T*G query rows of one kv head share one pass over that head's prefix
 * KV (streamed from HBM once), split along the context into `num_splits` chunks with a partial
 * (O, LSE) per chunk; the <= T_cap tree keys are attended under the ancestor mask; all partial
 * states are merged by log-sum-exp.  Contiguous or 16-key-paged KV with 128 % G == 0 runs as ONE fused
 * tcgen05 launch (tree keys = extra key tiles, merge in the same kernel); other group sizes run the
 * mma.sync kernels (prefix/tree pass + merge).  bf16 in, fp32 accumulate, bf16 out; the partial states
 * of the split-KV exchange are normalised O rows in bf16 and LSE in fp32.  Q and tree K are taken post q/k-norm and
 * post-RoPE (pos_id from (b) is for the caller's RoPE).  No sliding window / sinks / soft-cap.
 * ------------------------------------------------------------------------------------------- */
typedef struct d2sd_attn_params {
    int32_t B;           /* requests                                                            */
    int32_t T_cap;       /* tree capacity (row count of q / tree_k / tree_v / mask per request)  */
    int32_t Hq, Hkv;     /* Hq % Hkv == 0                                                        */
    int32_t d;           /* head dim; only 128 is built (else D2SD_ERR_UNSUPPORTED)              */
    float sm_scale;      /* <= 0 selects 1/sqrt(d)                                               */
    int32_t page_size;   /* 0 = contiguous KV; 16 = paged (only 16 is built)                     */
    int32_t max_ctx_len; /* host-side upper bound on ctx_len[b]; sizes the split-KV grid         */
    int64_t kv_rows;     /* token rows in k_cache/v_cache: contiguous: >= kv_indptr[B] (sum L_b);
                            paged: num_pages * page_size.  Bounds the TMA tensor maps.           */
    int32_t num_splits;  /* TEST KNOB, leave 0: key chunks per (request, kv head) chosen from the shape (<= 64);
                            one-tile-per-CTA kernel: values >= 256 mean (chunks of an odd last tile << 8) |
                            chunks of a paired tile                                                        */
    int32_t impl;        /* TEST KNOB, leave 0 (auto).  1 = force the mma.sync kernels; 2 = force the fused
                            two-query-tiles-per-CTA tcgen05 kernel; 3 = force the fused one-query-tile-per-
                            CTA tcgen05 kernel (2, 3: D2SD_ERR_UNSUPPORTED if the shape is outside them)  */
    int32_t phases;      /* TEST KNOB, leave 0 = the whole cascade.  For tests and profiling: 1 = attend the
                            committed prefix only, 2 = the tree keys only (out/lse then hold that
                            state; a prefix-only state with ctx_len = 0 is O = 0, LSE = -inf).
                            mma.sync kernels only: bit mask of 1 = prefix pass, 2 = tree pass,
                            4 = merge, the partial states staying in the workspace between calls.*/
} d2sd_attn_params;

/* Bytes of workspace d2sd_cascade_verify_attn needs for these params (0 on invalid params).
 * Depends on B, T_cap, Hq, Hkv, d, page_size, max_ctx_len, num_splits, impl only. */
size_t d2sd_cascade_workspace_bytes(const d2sd_attn_params* p /* host */);

/* Prepare a workspace for these params: enqueues a memset of its header (the arrival counters of
 * the fused kernel) on `stream`.  Call once after allocating the workspace, and again if a kernel of
 * this library ever failed on it; d2sd_cascade_verify_attn leaves the header zero after every call,
 * so the same workspace serves any number of calls (and any params it is large enough for) one
 * after another.  The rest of the workspace is scratch.  Two calls that may run concurrently need
 * two workspaces.
 * Co-scheduling: when every (request, kv head, query tile, chunk) CTA of a call fits on the device at
 * once (the plan sizes such grids to the SM count of the CURRENT device), the CTAs of a group wait for
 * each other inside the kernel and share the merge; this needs the whole device (no MPS / green-context
 * partition, no other kernel holding SMs for the ~20 us of the call).  A wait that does not end within
 * ~0.1 s gives up: the rows of that group are not written and the uint32 at byte offset 2^20 - 8 of the
 * workspace is set to 1 (it is otherwise 0; the caller may poll it).  Larger calls run in several waves,
 * never wait, and have no such requirement. */
int32_t d2sd_cascade_workspace_init(const d2sd_attn_params* p /* host */, void* workspace,
                                    size_t workspace_bytes, void* stream);

/*
 *   p           host; read during the call only
 *   q           bf16 [B,T_cap,Hq,d]
 *   k_cache, v_cache  bf16; contiguous: [kv_rows,Hkv,d], request b owns rows
 *               kv_indptr[b] .. kv_indptr[b]+ctx_len[b]-1; paged: pool [num_pages,16,Hkv,d]
 *   kv_indptr   int32 [B+1]; contiguous: token-row offsets (NULL allowed iff B == 1: offset 0);
 *               paged: offsets into kv_indices
 *   kv_indices  paged: int32 page ids of each request in sequence order; contiguous: NULL
 *   ctx_len     int32 [B], 0 <= ctx_len[b] <= max_ctx_len (0 is legal: the result is the tree state)
 *   tree_k, tree_v    bf16 [B,T_cap,Hkv,d]; rows t >= tree_len[b] may hold anything (NaN included)
 *   mask        uint32 [B,T_cap,W] as written by d2sd_build_tree (any ancestor-closed mask whose
 *               row n has its self bit and no bit > n is accepted)
 *   tree_len    int32 [B], 1 <= tree_len[b] <= T_cap
 *   out         bf16 [B,T_cap,Hq,d]; rows t >= tree_len[b] are left untouched
 *   lse         fp32 [B,T_cap,Hq] natural log, or NULL; padding rows untouched
 *   dbg_state   NULL, or fp32 [2,B,T_cap,Hq,d+1]: [0] = prefix-only state merged over the chunks,
 *               [1] = tree-only state; each row is the normalised O (d values) followed by its LSE.
 *               For tests: lets the two passes be checked separately.
 *   workspace   >= d2sd_cascade_workspace_bytes(p) bytes, 256-byte aligned, initialised by
 *               d2sd_cascade_workspace_init
 * 16-byte alignment is required of q, k_cache, v_cache, tree_k, tree_v and out.
 * Slots of a paged pool that no request owns (including the unused tail of a last page) may hold
 * anything, NaN included: they never reach an output.
 */
int32_t d2sd_cascade_verify_attn(const d2sd_attn_params* p, const void* q, const void* k_cache,
                                 const void* v_cache, const int32_t* kv_indptr,
                                 const int32_t* kv_indices, const int32_t* ctx_len,
                                 const void* tree_k, const void* tree_v, const uint32_t* mask,
                                 const int32_t* tree_len, void* out, float* lse, float* dbg_state,
                                 void* workspace, size_t workspace_bytes, void* stream);

/* ---------------------------------------------------------------------------------------------
 * (d) Greedy acceptance.  PAPER.md:69 ("accepting tokens up to (but not including) the first
 * mismatch"), :124 ("longest-accepted-prefix search across branches ... the target's prediction at
 * the rejection position becomes the next anchor").
 *   a[n]  = first index of the maximum of logits[b,n,:] (IEEE comparison: -0 == +0; NaN excluded)
 *   ok[0] = 1;  ok[n] = ok[parent[n]] && tokens[n] == a[parent[n]]
 *   best  = deepest ok node, ties -> smallest node index;  accept_len = depth[best] = number of
 *           accepted DRAFT tokens (anchor excluded), in [0,gamma-1];  bonus = a[best]
 *   logits      bf16, row n of request b at logits + (b*T_cap + n)*row_stride elements
 *   tokens, parent, depth  int32 [B,T_cap];  tree_len int32 [B]
 *   argmax_out  out int32 [B,T_cap]; -1 on rows n >= tree_len[b]
 *   accept_len, bonus, best_node  out int32 [B];  path out int32 [B,gamma]: node ids root..best,
 *               -1 padded
 *   workspace   >= d2sd_accept_workspace_bytes(B,T_cap,V) bytes, 16-byte aligned; scratch
 * Requires V >= 1, row_stride >= V, 2 <= gamma <= 64, T_cap <= 1024.
 * ------------------------------------------------------------------------------------------- */
size_t d2sd_accept_workspace_bytes(int32_t B, int32_t T_cap, int32_t V);

int32_t d2sd_accept(const void* logits, int64_t row_stride, int32_t V, const int32_t* tokens,
                    const int32_t* parent, const int32_t* depth, const int32_t* tree_len, int32_t B,
                    int32_t gamma, int32_t T_cap, int32_t* argmax_out, int32_t* accept_len,
                    int32_t* path, int32_t* bonus, int32_t* best_node, void* workspace,
                    size_t workspace_bytes, void* stream);

/* ---------------------------------------------------------------------------------------------
 * d2sd_accept without a workspace argument, for callers that cannot allocate one (code under CUDA
 * graph capture, serving loops or harnesses that forbid cudaMalloc).  Same inputs, outputs, kernels
 * and results as d2sd_accept; the chunk states live in a 1 MiB array built into the library
 * (d2sd_accept_static_max_bytes(); every GPU that loads the library holds it until exit).
 * Limit: B * T_cap * ceil(V/16384) * 16 bytes <= that size (65536 chunk states; BASELINE config 5
 * needs 11200), otherwise D2SD_ERR_UNSUPPORTED and nothing is enqueued.  The call allocates
 * nothing.  Every call on a device shares the one array: calls whose kernels may overlap on the
 * GPU (different streams, no dependency) RACE -- order them, or use d2sd_accept with separate
 * workspaces.  Nothing in the array has to be cleared between calls.
 * ------------------------------------------------------------------------------------------- */
size_t d2sd_accept_static_max_bytes(void);

int32_t d2sd_accept_static(const void* logits, int64_t row_stride, int32_t V, const int32_t* tokens,
                           const int32_t* parent, const int32_t* depth, const int32_t* tree_len, int32_t B,
                           int32_t gamma, int32_t T_cap, int32_t* argmax_out, int32_t* accept_len,
                           int32_t* path, int32_t* bonus, int32_t* best_node, void* stream);

/* =============================================================================================
 * The steps around the hot path (SURVEY.md 8f "next" rows), same conventions as above.
 * ============================================================================================= */

/* ---------------------------------------------------------------------------------------------
 * Confidence extraction, the step BEFORE (a).  PAPER.md:87-89, Eq. 3: the drafter emits a
 * categorical p_k(.) at block positions k = 1..gamma-1; t_k = argmax_v p_k(v) (greedy sample) and
 * c_k = p_k(t_k) = max_v p_k(v).  p_k = softmax of the logits row (temperature 1), so
 * c_k = 1 / sum_v exp(x_v - max_v x).  One vocabulary pass per row: (max, first index of the max,
 * sum of exponentials) per 16384-entry chunk, merged by a second small kernel.
 *   logits      bf16, drafter row of block position k (1..gamma-1) of request b at
 *               logits + (b*(gamma-1) + k-1)*row_stride elements, V entries
 *   anchor      int32 [B], the bonus token of the previous cycle (:69)
 *   draft       out int32 [B,gamma]: draft[b,0] = anchor[b], draft[b,k] = t_k (ties -> smallest v)
 *   conf        out fp32 [B,gamma]: conf[b,0] = 1, conf[b,k] = c_k -- the layout (a) and (b) consume
 *   workspace   >= d2sd_confidence_workspace_bytes(B,gamma,V) bytes, 16-byte aligned; scratch
 * Arithmetic: fp32 sums of ex2.approx exponentials; c_k agrees with the fp64 definition to ~1e-6
 * relative (tests gate 2e-5); t_k is bit-exact.  Requires 2 <= gamma <= 64, V >= 1, row_stride >= V.
 * ------------------------------------------------------------------------------------------- */
size_t d2sd_confidence_workspace_bytes(int32_t B, int32_t gamma, int32_t V);

int32_t d2sd_draft_confidence(const void* logits, int64_t row_stride, int32_t V, const int32_t* anchor,
                              int32_t B, int32_t gamma, int32_t* draft, float* conf, void* workspace,
                              size_t workspace_bytes, void* stream);

/* ---------------------------------------------------------------------------------------------
 * KV commit, the step AFTER (d).  PAPER.md:124 "commit the longest accepted prefix"; :119 each cycle
 * "consumes the verified KV caches ... and emits a new batch of accepted tokens"; :69 "refreshed
 * target hidden features that seed the next cycle".
 * The verify pass computed K/V of every tree node.  For j = 0..accept_len[b] the cache row at
 * position ctx_len[b] + j of EVERY layer receives the tree row of node path[b,j] (path[b,0] is the
 * root = this cycle's anchor, whose K/V the target had not seen before); the context grows by
 * accept_len[b] + 1.  The bonus token is the next cycle's anchor and has no K/V yet.
 *   tree_k, tree_v   bf16 [n_layers][B,T_cap,Hkv,d], layer l at + l*tree_layer_stride elements
 *   path, accept_len int32 [B,gamma] / [B] as written by d2sd_accept
 *   ctx_len          int32 [B] committed length before the call
 *   k_cache, v_cache bf16, in/out; layer l at + l*cache_layer_stride elements; addressing as in (c)
 *   kv_indptr        int32 [B+1]: contiguous: request b owns rows kv_indptr[b] .. kv_indptr[b+1]-1 of
 *                    which ctx_len[b] are in use (NULL iff B == 1: rows 0 .. kv_rows-1); paged: its
 *                    page-table segment kv_indices[kv_indptr[b] .. kv_indptr[b+1]) of which
 *                    ceil(ctx_len[b]/page_size) entries are in use
 *   kv_indices       paged: int32, in/out when a free list is given; contiguous: NULL
 *   free_pages, n_free, free_head   optional free list (NULL, 0, NULL: the unused entries of each
 *                    segment are already valid pages, reserved by the caller).  With a list, the pages a
 *                    request newly needs are taken from free_pages[*free_head ..) in request order
 *                    b = 0,1,.., written into its segment, and *free_head advances (device int32).
 *   ctx_len_out      out int32 [B] = ctx_len + rows committed; MAY alias ctx_len
 *   dropped          out int32 [B]: rows that did not fit (segment full / free list exhausted), cut
 *                    from the END of the path; 0 = everything committed
 *   feat, feat_out   optional (both or neither): bf16 [B,T_cap,F] target features of every node ->
 *                    [B,gamma,F], feat_out[b,j] = feat[b,path[b,j]] for j <= accept_len[b], zero rows behind
 *   workspace        >= d2sd_commit_workspace_bytes(B) bytes, 16-byte aligned; scratch
 * Byte-exact copies.  Requires (Hkv*d) % 8 == 0, F % 8 == 0, 16-byte aligned tensors and layer strides,
 * page_size 0 or > 0 (any), B <= 65535, n_layers <= 65535.
 * ------------------------------------------------------------------------------------------- */
typedef struct d2sd_commit_params {
    int32_t B, gamma, T_cap, Hkv, d, n_layers;
    int32_t page_size;          /* 0 = contiguous */
    int64_t kv_rows;            /* token rows per layer of k_cache / v_cache */
    int64_t tree_layer_stride;  /* elements between layers of tree_k / tree_v (>= B*T_cap*Hkv*d) */
    int64_t cache_layer_stride; /* elements between layers of the caches (>= kv_rows*Hkv*d) */
    int32_t F;                  /* feature width, 0 without feat */
} d2sd_commit_params;

size_t d2sd_commit_workspace_bytes(int32_t B);

int32_t d2sd_commit_kv(const d2sd_commit_params* p /* host */, const void* tree_k, const void* tree_v,
                       const int32_t* path, const int32_t* accept_len, const int32_t* ctx_len, void* k_cache,
                       void* v_cache, const int32_t* kv_indptr, int32_t* kv_indices, const int32_t* free_pages,
                       int32_t n_free, int32_t* free_head, int32_t* ctx_len_out, int32_t* dropped,
                       const void* feat, void* feat_out, void* workspace, size_t workspace_bytes, void* stream);

/* ---------------------------------------------------------------------------------------------
 * Third cascade level.  PAPER.md:228-240 (Ablation 3, Table 7): "for every i in S, we re-apply the
 * rejection-boundary estimator (Eq. 4) to that branch's second-draft tail, take the single top-1
 * location j_i, and dispatch a third VP-Drafter forward anchored there.  This yields up to 2K+1
 * shared-prefix candidates that the target jointly verifies in a single pass".
 * d2sd_select_third: branch k (prefix i_k) re-drafted positions i_k+1..gamma-1 with confidences
 * conf2[b,k,p].  r_k(j') = (prod_{m=1..j'} conf2[i_k+m]) * (1 - conf2[i_k+j'+1]) for j' = 1..n_k-1,
 * n_k = gamma-1-i_k (the third-level prefix strictly extends the branch's and leaves a position to
 * re-draft, so its block prefix length i_k+j' is in {1..gamma-2}, :228); top-1, ties -> smaller j';
 * same fp64 operation order as (a).
 *   conf2       fp32 [B,K,gamma];  prefix_len int32 [B,K] from (a)
 *   third_len   out int32 [B,K]: block prefix length j_k in [i_k+1, gamma-2], or -1 (n_k = 1: no child)
 *   r3_out      out fp64 [B,K,gamma-1] (entry j'; 0 outside the domain), or NULL
 * d2sd_build_tree3: the tree of d2sd_build_tree followed, in branch order, by the third-level
 * continuations: child of branch k holds draft3[b,k,j_k+1..gamma-1]; its first node's parent is branch
 * k's node at block position j_k.  branch_off out [B,2K+1]: [0..K) second-level starts, [K..2K)
 * third-level starts (an absent child: the next start), [2K] = tree_len.  T_cap must hold the largest
 * depth-3 tree: gamma + K(gamma-1) - K(K-1)/2 + K(gamma-2) - K(K-1)/2.  Everything else as (b); the
 * result feeds d2sd_cascade_verify_attn and d2sd_accept unchanged.
 * ------------------------------------------------------------------------------------------- */
int32_t d2sd_select_third(const float* conf2, const int32_t* prefix_len, int32_t B, int32_t gamma, int32_t K,
                          int32_t* third_len, double* r3_out, void* stream);

int32_t d2sd_build_tree3(const int32_t* draft1, const int32_t* draft2, const int32_t* draft3,
                         const int32_t* prefix_len, const int32_t* third_len, const int32_t* ctx_len, int32_t B,
                         int32_t gamma, int32_t K, int32_t T_cap, int32_t* tokens, int32_t* parent,
                         int32_t* depth, int32_t* pos_id, int32_t* branch_off, uint32_t* mask,
                         int32_t* tree_len, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* D2SD_H_ */
