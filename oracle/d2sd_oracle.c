/*
 * d2sd_oracle.c -- CPU oracle for the D2SD verification hot path.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load this library.  It shares no code, header,
 * table or helper with the CUDA path under paper_2606_04446_b200/ and neither imports the other.
 *
 * Plain, slow, obviously-correct C written from /root/reference/PAPER.md (arXiv 2606.04446) and,
 * where the paper is silent or garbled, from the readings G1..G21 listed in DESIGN.md.
 * Floating point is fp64 throughout; bf16 inputs are widened exactly.  No blocking, fusion or
 * re-association: attention is the explicit full masked softmax per (node, head); selection is a
 * full ranking; the mask is built by parent chasing; acceptance is the path walk.  The only
 * parallelism is an OpenMP "for" over independent output items.
 *
 * Pins (tests/test_oracle_pins.py, all run under -m "not gpu"):
 *   select : P1 telescoping closed form, P2 special cases + exhaustive grids vs an independent sort
 *   build  : P3 brute force over the K+1 flat candidate sequences, P4 structural invariants
 *   attn   : P3 (flat-sequence causal attention), P5 merge invariant, P6 torch SDPA fp64 special case
 *   accept : P7 special cases, P8 per-candidate linear rule, P9 numpy.argmax + planted ties
 *   next rows: confidence -> P10 torch.softmax fp64 + closed forms; commit_kv -> P11 two-cycle invariant
 *   (attention over the committed cache == attention over prefix + accepted path) + brute-force
 *   page walk; select_third / build_tree3 -> P12 exact-rational ranking, flat 2K+1 candidates, T formula
 * Parity unpinned: none of the functions below.  (alpha / speedup tables of the paper are not
 * computed here at all: they need weights and datasets.)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* bf16 bit pattern -> double, exact. */
static double bf16_to_f64(uint16_t b) {
    uint32_t u = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

/* ------------------------------------------------------------------------------------------
 * Stage (a): rejection-boundary posterior and top-K prefix selection.
 * PAPER.md:87-97 Eq. 3-4: r(i) = (prod_{k=1..i} c_k) * (1 - c_{i+1}),  i = 0..gamma-2   [G1]
 * PAPER.md:103-105 Eq. 5: S = Top-K_i r(i) over i in {0..gamma-2}                       [G2-G4]
 * Readings: fp32 confidences widened to fp64; sequential left-to-right product, one subtract and
 * one multiply per r(i), no FMA [G7]; ties -> smaller i [G5]; S emitted ascending [G6];
 * conf[.,0] (anchor slot) ignored [G9].
 * conf [B,gamma] -> prefix_len [B,K]; r_out [B,gamma-1] optional.
 * ------------------------------------------------------------------------------------------ */
void d2sd_oracle_select(const float* conf, int32_t B, int32_t gamma, int32_t K,
                        int32_t* prefix_len, double* r_out) {
    int32_t n = gamma - 1;
    double* r = (double*)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    int32_t* order = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
    for (int32_t b = 0; b < B; ++b) {
        const float* c = conf + (size_t)b * gamma;
        volatile double P = 1.0; /* volatile: forbid contraction/reordering of the stated order */
        for (int32_t i = 0; i < n; ++i) {
            volatile double one_minus = 1.0 - (double)c[i + 1];
            volatile double ri = P * one_minus;
            r[i] = ri;
            volatile double Pn = P * (double)c[i + 1];
            P = Pn;
        }
        if (r_out) memcpy(r_out + (size_t)b * n, r, sizeof(double) * (size_t)n);
        /* full ranking by (r descending, i ascending): stable insertion sort */
        for (int32_t i = 0; i < n; ++i) order[i] = i;
        for (int32_t i = 1; i < n; ++i) {
            int32_t x = order[i];
            int32_t j = i - 1;
            while (j >= 0 && r[order[j]] < r[x]) { order[j + 1] = order[j]; --j; }
            order[j + 1] = x;
        }
        /* first K of the ranking, emitted ascending in i */
        int32_t* out = prefix_len + (size_t)b * K;
        for (int32_t k = 0; k < K; ++k) out[k] = order[k];
        for (int32_t i = 1; i < K; ++i) {
            int32_t x = out[i];
            int32_t j = i - 1;
            while (j >= 0 && out[j] > x) { out[j + 1] = out[j]; --j; }
            out[j + 1] = x;
        }
    }
    free(r);
    free(order);
}

/* ------------------------------------------------------------------------------------------
 * Stage (b): shared-prefix tree.
 * branch i keeps the anchor and the first i draft-1 tokens and re-drafts
 * positions i+1..gamma-1; it shares its first i+1 tokens with draft 1.  Flattened-tree layout is
 * BASELINE.json's; node order / mask packing per [G12-G14]: trunk nodes 0..gamma-1 first, then
 * branches in ascending prefix length; pos_id = ctx_len + depth; uint32 mask words, bit (a%32)
 * of word a/32, self bit set; padding rows get tokens/parent = -1, depth/pos = 0, mask = 0.
 * The mask is built by PARENT CHASING (row n = row parent[n] plus bit n).
 * ------------------------------------------------------------------------------------------ */
void d2sd_oracle_build_tree(const int32_t* draft1, const int32_t* draft2, const int32_t* prefix_len,
                            const int32_t* ctx_len, int32_t B, int32_t gamma, int32_t K,
                            int32_t T_cap, int32_t* tokens, int32_t* parent, int32_t* depth,
                            int32_t* pos_id, int32_t* branch_off, uint32_t* mask,
                            int32_t* tree_len) {
    int32_t W = (T_cap + 31) / 32;
    for (int32_t b = 0; b < B; ++b) {
        int32_t* tok = tokens + (size_t)b * T_cap;
        int32_t* par = parent + (size_t)b * T_cap;
        int32_t* dep = depth + (size_t)b * T_cap;
        int32_t* pos = pos_id + (size_t)b * T_cap;
        uint32_t* mk = mask + (size_t)b * T_cap * W;
        int32_t* boff = branch_off + (size_t)b * (K + 1);
        for (int32_t n = 0; n < T_cap; ++n) { tok[n] = -1; par[n] = -1; dep[n] = 0; pos[n] = 0; }
        memset(mk, 0, sizeof(uint32_t) * (size_t)T_cap * W);
        /* trunk = draft-1 block (position 0 = anchor, root of the tree [G10]) */
        for (int32_t j = 0; j < gamma; ++j) {
            tok[j] = draft1[(size_t)b * gamma + j];
            par[j] = j - 1;
            dep[j] = j;
        }
        int32_t off = gamma;
        for (int32_t k = 0; k < K; ++k) {
            int32_t i = prefix_len[(size_t)b * K + k];
            boff[k] = off;
            for (int32_t p = i + 1; p <= gamma - 1; ++p) {
                int32_t n = off + (p - i - 1);
                tok[n] = draft2[((size_t)b * K + k) * gamma + p];
                par[n] = (p == i + 1) ? i : n - 1;
                dep[n] = p;
            }
            off += gamma - 1 - i;
        }
        boff[K] = off;
        tree_len[b] = off;
        for (int32_t n = 0; n < off; ++n) {
            pos[n] = ctx_len[b] + dep[n];
            /* chase parents up to the root, setting one bit per ancestor (and the self bit) */
            for (int32_t a = n; a >= 0; a = par[a]) mk[(size_t)n * W + a / 32] |= (1u << (a % 32));
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * Stage (c): verification attention, explicit definition.
 * every tree query attends to the shared committed prefix and to its own
 * candidate's in-block tokens ("cascade attention" is an exact re-association of this).
 * For request b, node t, head h, kv head g = h / (Hq/Hkv) [G15]:
 *   key set = { prefix j in [0,L_b) }  U  { tree a : bit a of mask row t }
 *   s = (q . k) * sm_scale ;  m = max s ;  l = sum e^(s-m) ;  O = sum e^(s-m) v / l ;
 *   LSE = m + ln l (natural log [G16]).
 * which: 0 = full key set, 1 = prefix only, 2 = tree only.  Empty key set (prefix-only with L=0):
 * O = 0, LSE = -inf.
 * KV addressing: page_size == 0 -> contiguous rows kv_indptr[b] + j (kv_indptr NULL => 0);
 * page_size > 0 -> page = kv_indices[kv_indptr[b] + j/page_size], row = page*page_size + j%page_size.
 * ------------------------------------------------------------------------------------------ */
static void attend_one(int which, const uint16_t* q, const uint16_t* k_cache, const uint16_t* v_cache,
                       const int32_t* kv_indptr, const int32_t* kv_indices, int32_t page_size,
                       const int32_t* ctx_len, const uint16_t* tree_k, const uint16_t* tree_v,
                       const uint32_t* mask, int32_t T_cap, int32_t W, int32_t Hq, int32_t Hkv,
                       int32_t d, double sm_scale, int32_t b, int32_t t, int32_t h, double* out,
                       double* lse) {
    int32_t g = h / (Hq / Hkv);
    int32_t L = (which == 2) ? 0 : ctx_len[b];
    int32_t nt = (which == 1) ? 0 : T_cap;
    const uint16_t* qrow = q + (((size_t)b * T_cap + t) * Hq + h) * d;
    const uint32_t* mrow = mask + ((size_t)b * T_cap + t) * W;
    size_t cap = (size_t)L + (size_t)nt + 1;
    double* s = (double*)malloc(sizeof(double) * cap);
    const uint16_t** vptr = (const uint16_t**)malloc(sizeof(uint16_t*) * cap);
    size_t n = 0;
    for (int32_t j = 0; j < L; ++j) {
        size_t row;
        if (page_size > 0) {
            int32_t page = kv_indices[(size_t)kv_indptr[b] + j / page_size];
            row = (size_t)page * page_size + (size_t)(j % page_size);
        } else {
            row = (size_t)(kv_indptr ? kv_indptr[b] : 0) + (size_t)j;
        }
        const uint16_t* kr = k_cache + (row * Hkv + g) * d;
        double acc = 0.0;
        for (int32_t e = 0; e < d; ++e) acc += bf16_to_f64(qrow[e]) * bf16_to_f64(kr[e]);
        s[n] = acc * sm_scale;
        vptr[n] = v_cache + (row * Hkv + g) * d;
        ++n;
    }
    for (int32_t a = 0; a < nt; ++a) {
        if (!((mrow[a / 32] >> (a % 32)) & 1u)) continue;
        const uint16_t* kr = tree_k + (((size_t)b * T_cap + a) * Hkv + g) * d;
        double acc = 0.0;
        for (int32_t e = 0; e < d; ++e) acc += bf16_to_f64(qrow[e]) * bf16_to_f64(kr[e]);
        s[n] = acc * sm_scale;
        vptr[n] = tree_v + (((size_t)b * T_cap + a) * Hkv + g) * d;
        ++n;
    }
    for (int32_t e = 0; e < d; ++e) out[e] = 0.0;
    if (n == 0) {
        *lse = -INFINITY;
    } else {
        double m = s[0];
        for (size_t i = 1; i < n; ++i) if (s[i] > m) m = s[i];
        double l = 0.0;
        for (size_t i = 0; i < n; ++i) l += exp(s[i] - m);
        for (size_t i = 0; i < n; ++i) {
            double p = exp(s[i] - m) / l;
            for (int32_t e = 0; e < d; ++e) out[e] += p * bf16_to_f64(vptr[i][e]);
        }
        *lse = m + log(l);
    }
    free(s);
    free(vptr);
}

/* Attention for a list of (b,t,h) triples (sel [n_sel,3]); out [n_sel,d], lse [n_sel]. */
void d2sd_oracle_attention_rows(int32_t which, const uint16_t* q, const uint16_t* k_cache,
                                const uint16_t* v_cache, const int32_t* kv_indptr,
                                const int32_t* kv_indices, int32_t page_size, const int32_t* ctx_len,
                                const uint16_t* tree_k, const uint16_t* tree_v, const uint32_t* mask,
                                int32_t T_cap, int32_t W, int32_t Hq, int32_t Hkv, int32_t d,
                                double sm_scale, const int32_t* sel, int64_t n_sel, double* out,
                                double* lse) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < n_sel; ++i) {
        attend_one(which, q, k_cache, v_cache, kv_indptr, kv_indices, page_size, ctx_len, tree_k,
                   tree_v, mask, T_cap, W, Hq, Hkv, d, sm_scale, sel[3 * i], sel[3 * i + 1],
                   sel[3 * i + 2], out + (size_t)i * d, lse + i);
    }
}

/* Attention for every (b, t < tree_len[b], h); out [B,T_cap,Hq,d], lse [B,T_cap,Hq].
 * Rows t >= tree_len[b] are left untouched. */
void d2sd_oracle_attention(int32_t which, const uint16_t* q, const uint16_t* k_cache,
                           const uint16_t* v_cache, const int32_t* kv_indptr,
                           const int32_t* kv_indices, int32_t page_size, const int32_t* ctx_len,
                           const uint16_t* tree_k, const uint16_t* tree_v, const uint32_t* mask,
                           const int32_t* tree_len, int32_t B, int32_t T_cap, int32_t W, int32_t Hq,
                           int32_t Hkv, int32_t d, double sm_scale, double* out, double* lse) {
    int64_t total = (int64_t)B * T_cap * Hq;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < total; ++i) {
        int32_t h = (int32_t)(i % Hq);
        int32_t t = (int32_t)((i / Hq) % T_cap);
        int32_t b = (int32_t)(i / ((int64_t)Hq * T_cap));
        if (t >= tree_len[b]) continue;
        attend_one(which, q, k_cache, v_cache, kv_indptr, kv_indices, page_size, ctx_len, tree_k,
                   tree_v, mask, T_cap, W, Hq, Hkv, d, sm_scale, b, t, h, out + (size_t)i * d,
                   lse + i);
    }
}

/* ------------------------------------------------------------------------------------------
 * Stage (d): greedy acceptance.
 * "accepting tokens up to (but not including) the first mismatch"; :124: "a
 * longest-accepted-prefix search across branches ... the target's prediction at the rejection
 * position becomes the next anchor".
 * a[n] = first index of the maximum of logits[n,.] under IEEE comparison (-0 == +0) [G18].
 * ok[0] = 1; ok[n] = ok[parent[n]] && tokens[n] == a[parent[n]]; best = deepest ok node, ties ->
 * smallest node index [G17]; accept_len = depth[best] (accepted DRAFT tokens, anchor excluded
 * [G19]); path = node ids root..best, -1 padded to gamma; bonus = a[best].
 * logits bf16 bits, row n of request b at logits + (b*T_cap + n)*row_stride.
 * ------------------------------------------------------------------------------------------ */
void d2sd_oracle_argmax(const uint16_t* logits, int64_t row_stride, int32_t V, const int32_t* tree_len,
                        int32_t B, int32_t T_cap, int32_t* argmax_out) {
    int64_t total = (int64_t)B * T_cap;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < total; ++i) {
        int32_t b = (int32_t)(i / T_cap), n = (int32_t)(i % T_cap);
        if (n >= tree_len[b]) { argmax_out[i] = -1; continue; }
        const uint16_t* row = logits + (size_t)i * row_stride;
        int32_t best = 0;
        double bv = bf16_to_f64(row[0]);
        for (int32_t v = 1; v < V; ++v) {
            double x = bf16_to_f64(row[v]);
            if (x > bv) { bv = x; best = v; }
        }
        argmax_out[i] = best;
    }
}

void d2sd_oracle_accept_walk(const int32_t* argmax, const int32_t* tokens, const int32_t* parent,
                             const int32_t* depth, const int32_t* tree_len, int32_t B, int32_t gamma,
                             int32_t T_cap, int32_t* accept_len, int32_t* path, int32_t* bonus,
                             int32_t* best_node) {
    uint8_t* ok = (uint8_t*)malloc((size_t)T_cap);
    for (int32_t b = 0; b < B; ++b) {
        const int32_t* a = argmax + (size_t)b * T_cap;
        const int32_t* tok = tokens + (size_t)b * T_cap;
        const int32_t* par = parent + (size_t)b * T_cap;
        const int32_t* dep = depth + (size_t)b * T_cap;
        int32_t T = tree_len[b];
        int32_t best = 0;
        ok[0] = 1;
        for (int32_t n = 1; n < T; ++n) {
            ok[n] = (uint8_t)(ok[par[n]] && tok[n] == a[par[n]]); /* parent[n] < n always */
            if (ok[n] && dep[n] > dep[best]) best = n;            /* strict: ties keep smaller n */
        }
        accept_len[b] = dep[best];
        best_node[b] = best;
        bonus[b] = a[best];
        int32_t* pth = path + (size_t)b * gamma;
        for (int32_t j = 0; j < gamma; ++j) pth[j] = -1;
        for (int32_t n = best; n >= 0; n = par[n]) pth[dep[n]] = n;
    }
    free(ok);
}

/* ------------------------------------------------------------------------------------------
 * Next row f3: confidence extraction (the step that feeds stage (a)).
 * PAPER.md:87-89 Eq. 3: the drafter emits a categorical p_k(.) at block positions k = 1..gamma-1;
 * t_k = argmax_v p_k(v) (greedy sample), c_k = p_k(t_k) = max_v p_k(v).
 * p_k = softmax of the drafter's logits row (temperature 1) [G23]; argmax ties -> smallest v, IEEE
 * comparison as in stage (d) [G18].  fp64: m = max x, s = sum_v e^(x_v - m) in index order,
 * c = e^(x_t - m) / s = 1 / s.
 * logits bf16 bits [B, gamma-1, V] (row r of request b at logits + (b*(gamma-1) + r)*row_stride holds
 * block position k = r+1); anchor int32 [B].  Outputs in the layout stages (a)/(b) consume [G9]:
 * draft [B,gamma] with draft[.,0] = anchor, conf [B,gamma] with conf[.,0] = 1.
 * ------------------------------------------------------------------------------------------ */
void d2sd_oracle_confidence(const uint16_t* logits, int64_t row_stride, int32_t V, const int32_t* anchor,
                            int32_t B, int32_t gamma, int32_t* draft, double* conf) {
    int64_t total = (int64_t)B * gamma;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < total; ++i) {
        int32_t b = (int32_t)(i / gamma), k = (int32_t)(i % gamma);
        if (k == 0) { draft[i] = anchor[b]; conf[i] = 1.0; continue; }
        const uint16_t* row = logits + ((size_t)b * (gamma - 1) + (size_t)(k - 1)) * row_stride;
        int32_t best = 0;
        double m = bf16_to_f64(row[0]);
        for (int32_t v = 1; v < V; ++v) {
            double x = bf16_to_f64(row[v]);
            if (x > m) { m = x; best = v; }
        }
        double s = 0.0;
        for (int32_t v = 0; v < V; ++v) s += exp(bf16_to_f64(row[v]) - m);
        draft[i] = best;
        conf[i] = 1.0 / s;
    }
}

/* ------------------------------------------------------------------------------------------
 * Next row f1: commit of the accepted path into the KV cache (the step after stage (d)).
 * PAPER.md:124 "commit the longest accepted prefix"; :119 each cycle "consumes the verified KV caches
 * ... and emits a new batch of accepted tokens"; :69 "refreshed target hidden features that seed the
 * next cycle".
 * The verify pass computed K/V of every tree node; the nodes of path[0..accept_len] (root = anchor,
 * then the accepted draft tokens [G10, G19]) become committed context: for j = 0..accept_len the
 * cache row at position L + j receives the tree row of node path[j], in every layer, and the context
 * grows by n = accept_len + 1 [G24].  The bonus token is the NEXT cycle's anchor; its K/V does not
 * exist yet.
 * Addressing as in stage (c).  Capacity [G25]: contiguous: request b owns rows
 * kv_indptr[b]..kv_indptr[b+1] (kv_indptr NULL: kv_rows rows); paged: its page-table segment
 * kv_indices[kv_indptr[b]..kv_indptr[b+1]) has ceil(L/page) pages in use; with a free list
 * (free_pages != NULL) the next entries are filled from free_pages[*free_head ..) in request order
 * b = 0,1,.. as far as the list lasts, without one the remaining entries are taken as already
 * reserved by the caller.  Rows that do not fit are dropped from the END of the path:
 * n_fit <= n, ctx_len_out = L + n_fit, dropped[b] = n - n_fit (0 = everything committed).
 * tree_k/tree_v [n_layers][B][T_cap][Hkv][d] with element stride tree_layer_stride between layers;
 * caches with element stride cache_layer_stride between layers.  Plain loops, byte-exact copy.
 * ------------------------------------------------------------------------------------------ */
void d2sd_oracle_commit_kv(const uint16_t* tree_k, const uint16_t* tree_v, int64_t tree_layer_stride,
                           const int32_t* path, const int32_t* accept_len, const int32_t* ctx_len,
                           uint16_t* k_cache, uint16_t* v_cache, int64_t cache_layer_stride,
                           int64_t kv_rows, const int32_t* kv_indptr, int32_t* kv_indices,
                           int32_t page_size, const int32_t* free_pages, int32_t n_free,
                           int32_t* free_head, int32_t B, int32_t gamma, int32_t T_cap, int32_t Hkv,
                           int32_t d, int32_t n_layers, int32_t* ctx_len_out, int32_t* dropped) {
    size_t row_elems = (size_t)Hkv * d;
    for (int32_t b = 0; b < B; ++b) {
        int32_t L = ctx_len[b];
        int32_t n = accept_len[b] + 1;
        int64_t cap_rows;
        if (page_size > 0) cap_rows = (int64_t)(kv_indptr[b + 1] - kv_indptr[b]) * page_size;
        else cap_rows = kv_indptr ? (int64_t)(kv_indptr[b + 1] - kv_indptr[b]) : kv_rows;
        int32_t n_fit = n;
        if ((int64_t)L + n_fit > cap_rows) n_fit = (int32_t)(cap_rows > L ? cap_rows - L : 0);
        if (page_size > 0 && free_pages) {
            int32_t owned = (L + page_size - 1) / page_size;
            int32_t want = (L + n_fit + page_size - 1) / page_size - owned;
            int32_t left = n_free - *free_head;
            int32_t got = want < left ? want : (left > 0 ? left : 0);
            for (int32_t e = 0; e < got; ++e)
                kv_indices[(size_t)kv_indptr[b] + owned + e] = free_pages[*free_head + e];
            *free_head += got;
            int64_t room = (int64_t)(owned + got) * page_size - L;
            if (n_fit > room) n_fit = (int32_t)room;
        }
        for (int32_t layer = 0; layer < n_layers; ++layer) {
            for (int32_t j = 0; j < n_fit; ++j) {
                int32_t node = path[(size_t)b * gamma + j];
                int32_t pos = L + j;
                size_t row;
                if (page_size > 0)
                    row = (size_t)kv_indices[(size_t)kv_indptr[b] + pos / page_size] * page_size + (size_t)(pos % page_size);
                else
                    row = (size_t)(kv_indptr ? kv_indptr[b] : 0) + (size_t)pos;
                size_t src = (size_t)layer * tree_layer_stride + ((size_t)b * T_cap + node) * row_elems;
                size_t dst = (size_t)layer * cache_layer_stride + row * row_elems;
                memcpy(k_cache + dst, tree_k + src, row_elems * sizeof(uint16_t));
                memcpy(v_cache + dst, tree_v + src, row_elems * sizeof(uint16_t));
            }
        }
        ctx_len_out[b] = L + n_fit;
        dropped[b] = n - n_fit;
    }
}

/* Same passage (:69): the target features of the accepted path, in path order, for the next cycle's
 * drafters.  feat bf16 bits [B,T_cap,F] -> out [B,gamma,F]: out[b,j] = feat[b,path[b,j]] for
 * j <= accept_len[b], zero rows behind. */
void d2sd_oracle_gather_path(const uint16_t* feat, const int32_t* path, const int32_t* accept_len,
                             int32_t B, int32_t gamma, int32_t T_cap, int32_t F, uint16_t* out) {
    for (int32_t b = 0; b < B; ++b)
        for (int32_t j = 0; j < gamma; ++j) {
            uint16_t* o = out + ((size_t)b * gamma + j) * F;
            if (j <= accept_len[b])
                memcpy(o, feat + ((size_t)b * T_cap + path[(size_t)b * gamma + j]) * F, (size_t)F * sizeof(uint16_t));
            else
                memset(o, 0, (size_t)F * sizeof(uint16_t));
        }
}

/* ------------------------------------------------------------------------------------------
 * Next row f2: third cascade level (Ablation 3, Table 7).
 * "for every i in S, we re-apply the rejection-boundary estimator (Eq. 4) to that branch's
 * second-draft tail, take the single top-1 location j_i, and dispatch a third VP-Drafter forward
 * anchored there.  This yields up to 2K+1 shared-prefix candidates".
 * Branch b (prefix i_b) re-drafted block positions i_b+1..gamma-1 with confidences conf2[b][p].
 * Eq. 4 on the tail: keeping the first j' tail tokens and losing the next one has posterior
 *   r_b(j') = (prod_{k=1..j'} conf2[b][i_b+k]) * (1 - conf2[b][i_b+j'+1]).
 * Reading [G22]: a third-level prefix strictly extends its branch's prefix and leaves at least one
 * position to re-draft, j' in {1..n_b-1} with n_b = gamma-1-i_b, so the third-level prefix length
 * in block terms j_b = i_b + j' lies in {1..gamma-2} (the set :228 names) and a branch with
 * n_b = 1 has no third-level child ("up to" 2K+1).  Top-1, ties -> smaller j' [G5]; same fp64
 * operation order as stage (a) [G7].
 * conf2 fp32 [B,K,gamma]; prefix_len [B,K] -> third_len int32 [B,K] (block prefix length j_b, or
 * -1: no child); r3_out optional fp64 [B,K,gamma-1], entry j' (0 where j' is outside the domain).
 * ------------------------------------------------------------------------------------------ */
void d2sd_oracle_select_third(const float* conf2, const int32_t* prefix_len, int32_t B, int32_t gamma,
                              int32_t K, int32_t* third_len, double* r3_out) {
    for (int32_t b = 0; b < B; ++b)
        for (int32_t k = 0; k < K; ++k) {
            const float* c = conf2 + ((size_t)b * K + k) * gamma;
            int32_t i = prefix_len[(size_t)b * K + k];
            int32_t nb = gamma - 1 - i;
            double* r3 = r3_out ? r3_out + ((size_t)b * K + k) * (gamma - 1) : NULL;
            if (r3) for (int32_t j = 0; j < gamma - 1; ++j) r3[j] = 0.0;
            int32_t best = -1;
            double best_r = 0.0;
            volatile double P = 1.0;
            for (int32_t j = 0; j <= nb - 1; ++j) { /* j tail tokens kept, tail token j+1 rejected */
                volatile double one_minus = 1.0 - (double)c[i + j + 1];
                volatile double rj = P * one_minus;
                if (j >= 1) {
                    if (r3) r3[j] = rj;
                    if (best < 0 || rj > best_r) { best = j; best_r = rj; } /* strict: ties keep smaller j */
                }
                volatile double Pn = P * (double)c[i + j + 1];
                P = Pn;
            }
            third_len[(size_t)b * K + k] = best < 0 ? -1 : i + best;
        }
}

/* Depth-3 tree: the two-level tree of stage (b) followed, in branch order, by the third-level
 * continuations.  Child of branch k with third_len j (>= i_k + 1): nodes for block positions
 * p = j+1..gamma-1 with tokens draft3[k][p]; the first hangs under branch k's node at position j
 * (node boff[k] + j - i_k - 1), the rest form a chain.  branch_off has 2K+1 entries + the end:
 * [0..K) second-level starts, [K..2K) third-level starts (== next start when absent), [2K] = tree_len.
 * Everything else (pos_id, mask by parent chasing, padding) as d2sd_oracle_build_tree. */
void d2sd_oracle_build_tree3(const int32_t* draft1, const int32_t* draft2, const int32_t* draft3,
                             const int32_t* prefix_len, const int32_t* third_len, const int32_t* ctx_len,
                             int32_t B, int32_t gamma, int32_t K, int32_t T_cap, int32_t* tokens,
                             int32_t* parent, int32_t* depth, int32_t* pos_id, int32_t* branch_off,
                             uint32_t* mask, int32_t* tree_len) {
    int32_t W = (T_cap + 31) / 32;
    for (int32_t b = 0; b < B; ++b) {
        int32_t* tok = tokens + (size_t)b * T_cap;
        int32_t* par = parent + (size_t)b * T_cap;
        int32_t* dep = depth + (size_t)b * T_cap;
        int32_t* pos = pos_id + (size_t)b * T_cap;
        uint32_t* mk = mask + (size_t)b * T_cap * W;
        int32_t* boff = branch_off + (size_t)b * (2 * K + 1);
        for (int32_t n = 0; n < T_cap; ++n) { tok[n] = -1; par[n] = -1; dep[n] = 0; pos[n] = 0; }
        memset(mk, 0, sizeof(uint32_t) * (size_t)T_cap * W);
        for (int32_t j = 0; j < gamma; ++j) {
            tok[j] = draft1[(size_t)b * gamma + j];
            par[j] = j - 1;
            dep[j] = j;
        }
        int32_t off = gamma;
        for (int32_t k = 0; k < K; ++k) {
            int32_t i = prefix_len[(size_t)b * K + k];
            boff[k] = off;
            for (int32_t p = i + 1; p <= gamma - 1; ++p) {
                int32_t n = off + (p - i - 1);
                tok[n] = draft2[((size_t)b * K + k) * gamma + p];
                par[n] = (p == i + 1) ? i : n - 1;
                dep[n] = p;
            }
            off += gamma - 1 - i;
        }
        for (int32_t k = 0; k < K; ++k) {
            int32_t i = prefix_len[(size_t)b * K + k];
            int32_t j = third_len[(size_t)b * K + k];
            boff[K + k] = off;
            if (j < 0) continue;
            for (int32_t p = j + 1; p <= gamma - 1; ++p) {
                int32_t n = off + (p - j - 1);
                tok[n] = draft3[((size_t)b * K + k) * gamma + p];
                par[n] = (p == j + 1) ? boff[k] + (j - i - 1) : n - 1;
                dep[n] = p;
            }
            off += gamma - 1 - j;
        }
        boff[2 * K] = off;
        tree_len[b] = off;
        for (int32_t n = 0; n < off; ++n) {
            pos[n] = ctx_len[b] + dep[n];
            for (int32_t a = n; a >= 0; a = par[a]) mk[(size_t)n * W + a / 32] |= (1u << (a % 32));
        }
    }
}

/* Number of OpenMP threads the parallel loops above will use (reported by bench.py). */
#ifdef _OPENMP
#include <omp.h>
int32_t d2sd_oracle_num_threads(void) { return (int32_t)omp_get_max_threads(); }
#else
int32_t d2sd_oracle_num_threads(void) { return 1; }
#endif
