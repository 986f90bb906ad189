// Stage (a) top-K prefix selection and stage (b) shared-prefix tree build.
// PAPER.md:87-105 (Eq. 3-5), :107, :123-124.  Launch-latency-sized kernels: one CTA per request.
#include "common.cuh"

namespace d2sd {

__device__ __forceinline__ void sb_pdl() {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}
static cudaLaunchConfig_t sb_config(dim3 grid, dim3 block, cudaStream_t s, cudaLaunchAttribute* attr) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.stream = s;
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cfg;
}

// ---------------------------------------------------------------------------------------------
// (a) r(i) = (prod_{k<=i} c_k) * (1 - c_{i+1}), i = 0..gamma-2 (Eq. 4);
//     S = Top-K_i r(i) (Eq. 5).
// One warp per request.  Candidate i recomputes its own prefix product left to right with
// __dmul_rn (one rounding per multiply, never contracted into an FMA) so that r is bit-identical
// to a sequential host evaluation; a warp scan would re-associate the product.
// Rank by (r descending, i ascending); the K best are emitted in ascending i.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(32) select_prefixes_kernel(const float* __restrict__ conf, int gamma,
                                                             int K, int32_t* __restrict__ prefix_len,
                                                             double* __restrict__ r_out) {
    __shared__ double r_s[64];
    __shared__ int sel_s[64];
    sb_pdl();
    const int b = blockIdx.x;
    const int lane = threadIdx.x;
    const int n = gamma - 1;
    const float* c = conf + (size_t)b * gamma;
    for (int i = lane; i < n; i += 32) {
        double P = 1.0;
        for (int k = 1; k <= i; ++k) P = __dmul_rn(P, (double)c[k]);
        const double ri = __dmul_rn(P, __dsub_rn(1.0, (double)c[i + 1]));
        r_s[i] = ri;
        if (r_out) r_out[(size_t)b * n + i] = ri;
    }
    __syncwarp();
    for (int i = lane; i < n; i += 32) {
        const double ri = r_s[i];
        int rank = 0;
        for (int j = 0; j < n; ++j) {
            const double rj = r_s[j];
            rank += (rj > ri) || (rj == ri && j < i);
        }
        sel_s[i] = rank < K;
    }
    __syncwarp();
    for (int i = lane; i < n; i += 32) {
        if (sel_s[i]) {
            int pos = 0;
            for (int j = 0; j < i; ++j) pos += sel_s[j];
            prefix_len[(size_t)b * K + pos] = i;
        }
    }
}

int32_t launch_select(const float* conf, int B, int gamma, int K, int32_t* prefix_len, double* r_out,
                      cudaStream_t s) {
    if (B == 0) return D2SD_OK;
    cudaLaunchAttribute attr[1];
    cudaLaunchConfig_t cfg = sb_config(dim3(B), dim3(32), s, attr);
    D2SD_CHECK_CUDA(cudaLaunchKernelEx(&cfg, select_prefixes_kernel, conf, gamma, K, prefix_len, r_out));
    D2SD_CHECK_LAUNCH("select_prefixes_kernel");
    return D2SD_OK;
}

// ---------------------------------------------------------------------------------------------
// (b) Flattened shared-prefix tree.  One CTA per request, one thread per node.
// Branch k keeps trunk nodes 0..i_k and appends gamma-1-i_k nodes.
// The ancestor set of a branch node n is two contiguous ranges, trunk [0, i_k] and branch
// [off_k, n]; of a trunk node, [0, n].  Each thread writes its own W mask words from that
// closed form (the oracle chases parents instead).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t range_bits(int lo, int hi, int word) {
    // bits of [lo,hi] (inclusive) that fall into 32-bit word `word`
    const int wlo = word * 32, whi = wlo + 31;
    const int a = lo > wlo ? lo : wlo;
    const int z = hi < whi ? hi : whi;
    if (a > z) return 0u;
    const uint32_t upto_z = (z - wlo == 31) ? 0xFFFFFFFFu : ((1u << (z - wlo + 1)) - 1u);
    const uint32_t below_a = (1u << (a - wlo)) - 1u;
    return upto_z & ~below_a;
}

__global__ void build_tree_kernel(const int32_t* __restrict__ draft1, const int32_t* __restrict__ draft2,
                                  const int32_t* __restrict__ prefix_len,
                                  const int32_t* __restrict__ ctx_len, int gamma, int K, int T_cap, int W,
                                  int32_t* __restrict__ tokens, int32_t* __restrict__ parent,
                                  int32_t* __restrict__ depth, int32_t* __restrict__ pos_id,
                                  int32_t* __restrict__ branch_off, uint32_t* __restrict__ mask,
                                  int32_t* __restrict__ tree_len) {
    __shared__ int off_s[65];
    __shared__ int pre_s[64];
    sb_pdl();
    const int b = blockIdx.x;
    if (threadIdx.x == 0) {
        int off = gamma;
        for (int k = 0; k < K; ++k) {
            const int i = prefix_len[(size_t)b * K + k];
            pre_s[k] = i;
            off_s[k] = off;
            off += gamma - 1 - i;
        }
        off_s[K] = off;
        tree_len[b] = off;
    }
    __syncthreads();
    for (int k = threadIdx.x; k <= K; k += blockDim.x) branch_off[(size_t)b * (K + 1) + k] = off_s[k];
    const int T = off_s[K];
    const int L = ctx_len[b];
    for (int n = threadIdx.x; n < T_cap; n += blockDim.x) {
        const size_t o = (size_t)b * T_cap + n;
        uint32_t* mrow = mask + o * W;
        if (n >= T) {
            tokens[o] = -1; parent[o] = -1; depth[o] = 0; pos_id[o] = 0;
            for (int w = 0; w < W; ++w) mrow[w] = 0u;
            continue;
        }
        if (n < gamma) {
            tokens[o] = draft1[(size_t)b * gamma + n];
            parent[o] = n - 1;
            depth[o] = n;
            pos_id[o] = L + n;
            for (int w = 0; w < W; ++w) mrow[w] = range_bits(0, n, w);
        } else {
            int k = 0;
            while (n >= off_s[k + 1]) ++k;
            const int i = pre_s[k];
            const int p = i + 1 + (n - off_s[k]);  // block position of this node
            tokens[o] = draft2[((size_t)b * K + k) * gamma + p];
            parent[o] = (n == off_s[k]) ? i : n - 1;
            depth[o] = p;
            pos_id[o] = L + p;
            for (int w = 0; w < W; ++w) mrow[w] = range_bits(0, i, w) | range_bits(off_s[k], n, w);
        }
    }
}

int32_t launch_build_tree(const int32_t* draft1, const int32_t* draft2, const int32_t* prefix_len,
                          const int32_t* ctx_len, int B, int gamma, int K, int T_cap, int32_t* tokens,
                          int32_t* parent, int32_t* depth, int32_t* pos_id, int32_t* branch_off,
                          uint32_t* mask, int32_t* tree_len, cudaStream_t s) {
    if (B == 0) return D2SD_OK;
    const int W = (T_cap + 31) / 32;
    int threads = ((T_cap + 31) / 32) * 32;
    if (threads > 256) threads = 256;
    if (threads < 32) threads = 32;
    cudaLaunchAttribute attr[1];
    cudaLaunchConfig_t cfg = sb_config(dim3(B), dim3(threads), s, attr);
    D2SD_CHECK_CUDA(cudaLaunchKernelEx(&cfg, build_tree_kernel, draft1, draft2, prefix_len, ctx_len, gamma, K, T_cap, W, tokens,
                                       parent, depth, pos_id, branch_off, mask, tree_len));
    D2SD_CHECK_LAUNCH("build_tree_kernel");
    return D2SD_OK;
}

// ---------------------------------------------------------------------------------------------
// Third cascade level (Ablation 3): "for every i in S, we re-apply
// the rejection-boundary estimator (Eq. 4) to that branch's second-draft tail, take the single top-1
// location j_i".  Branch k (prefix i) re-drafted positions i+1..gamma-1 with confidences conf2[k][p];
// keeping j' tail tokens and losing the next has r(j') = (prod_{m<=j'} conf2[i+m]) (1 - conf2[i+j'+1]);
// the third-level prefix strictly extends the branch's (j' in 1..n-1, n = gamma-1-i), so its block
// prefix length i+j' lies in {1..gamma-2} (:228) and a branch with n = 1 has no child.
// One warp per (request, branch); lane j' recomputes its own product left to right (same arithmetic
// rule as stage (a)); top-1 with ties to the smaller j'.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(32) select_third_kernel(const float* __restrict__ conf2,
                                                          const int32_t* __restrict__ prefix_len, int gamma,
                                                          int32_t* __restrict__ third_len,
                                                          double* __restrict__ r3_out) {
    sb_pdl();
    const int bk = blockIdx.x;  // b*K + k
    const int lane = threadIdx.x;
    const float* c = conf2 + (size_t)bk * gamma;
    const int i = prefix_len[bk];
    const int n = gamma - 1 - i;
    double best_r = -1.0;
    int best_j = 0x7fffffff;
    for (int j = lane; j < gamma - 1; j += 32) {
        double rj = 0.0;
        if (j >= 1 && j <= n - 1) {
            double P = 1.0;
            for (int m = 1; m <= j; ++m) P = __dmul_rn(P, (double)c[i + m]);
            rj = __dmul_rn(P, __dsub_rn(1.0, (double)c[i + j + 1]));
            if (rj > best_r) { best_r = rj; best_j = j; }  // ascending j per lane: ties keep the smaller
        }
        if (r3_out) r3_out[(size_t)bk * (gamma - 1) + j] = rj;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double orr = __shfl_xor_sync(0xffffffffu, best_r, o);
        const int oj = __shfl_xor_sync(0xffffffffu, best_j, o);
        if (orr > best_r || (orr == best_r && oj < best_j)) { best_r = orr; best_j = oj; }
    }
    if (lane == 0) third_len[bk] = best_j == 0x7fffffff ? -1 : i + best_j;
}

int32_t launch_select_third(const float* conf2, const int32_t* prefix_len, int B, int gamma, int K,
                            int32_t* third_len, double* r3_out, cudaStream_t s) {
    if (B == 0 || K == 0) return D2SD_OK;
    cudaLaunchAttribute attr[1];
    cudaLaunchConfig_t cfg = sb_config(dim3(B * K), dim3(32), s, attr);
    D2SD_CHECK_CUDA(cudaLaunchKernelEx(&cfg, select_third_kernel, conf2, prefix_len, gamma, third_len, r3_out));
    D2SD_CHECK_LAUNCH("select_third_kernel");
    return D2SD_OK;
}

// Depth-3 tree: the two-level tree followed, in branch order, by the third-level continuations
// (child of branch k with prefix length j: block positions j+1..gamma-1 from draft3[k], hanging under
// branch k's node at position j).  Ancestors of a third-level node n: trunk [0, i_k], branch
// [off_k, off_k + j - i_k - 1], own [off3_k, n] -- three ranges (the oracle chases parents).
__global__ void build_tree3_kernel(const int32_t* __restrict__ draft1, const int32_t* __restrict__ draft2,
                                   const int32_t* __restrict__ draft3, const int32_t* __restrict__ prefix_len,
                                   const int32_t* __restrict__ third_len, const int32_t* __restrict__ ctx_len,
                                   int gamma, int K, int T_cap, int W, int32_t* __restrict__ tokens,
                                   int32_t* __restrict__ parent, int32_t* __restrict__ depth,
                                   int32_t* __restrict__ pos_id, int32_t* __restrict__ branch_off,
                                   uint32_t* __restrict__ mask, int32_t* __restrict__ tree_len) {
    __shared__ int off_s[129];   // [0..K) second level, [K..2K) third level, [2K] = end
    __shared__ int pre_s[64], thr_s[64];
    sb_pdl();
    const int b = blockIdx.x;
    if (threadIdx.x == 0) {
        int off = gamma;
        for (int k = 0; k < K; ++k) {
            const int i = prefix_len[(size_t)b * K + k];
            pre_s[k] = i;
            off_s[k] = off;
            off += gamma - 1 - i;
        }
        for (int k = 0; k < K; ++k) {
            const int j = third_len[(size_t)b * K + k];
            thr_s[k] = j;
            off_s[K + k] = off;
            if (j >= 0) off += gamma - 1 - j;
        }
        off_s[2 * K] = off;
        tree_len[b] = off;
    }
    __syncthreads();
    for (int k = threadIdx.x; k <= 2 * K; k += blockDim.x) branch_off[(size_t)b * (2 * K + 1) + k] = off_s[k];
    const int T = off_s[2 * K];
    const int L = ctx_len[b];
    for (int n = threadIdx.x; n < T_cap; n += blockDim.x) {
        const size_t o = (size_t)b * T_cap + n;
        uint32_t* mrow = mask + o * W;
        if (n >= T) {
            tokens[o] = -1; parent[o] = -1; depth[o] = 0; pos_id[o] = 0;
            for (int w = 0; w < W; ++w) mrow[w] = 0u;
        } else if (n < gamma) {
            tokens[o] = draft1[(size_t)b * gamma + n];
            parent[o] = n - 1;
            depth[o] = n;
            pos_id[o] = L + n;
            for (int w = 0; w < W; ++w) mrow[w] = range_bits(0, n, w);
        } else if (n < off_s[K]) {
            int k = 0;
            while (n >= off_s[k + 1]) ++k;
            const int i = pre_s[k];
            const int p = i + 1 + (n - off_s[k]);
            tokens[o] = draft2[((size_t)b * K + k) * gamma + p];
            parent[o] = (n == off_s[k]) ? i : n - 1;
            depth[o] = p;
            pos_id[o] = L + p;
            for (int w = 0; w < W; ++w) mrow[w] = range_bits(0, i, w) | range_bits(off_s[k], n, w);
        } else {
            int k = 0;
            while (n >= off_s[K + k + 1]) ++k;  // empty third-level slots have equal offsets and are skipped
            const int i = pre_s[k], j = thr_s[k];
            const int p = j + 1 + (n - off_s[K + k]);
            const int anchor = off_s[k] + (j - i - 1);  // branch k's node at block position j
            tokens[o] = draft3[((size_t)b * K + k) * gamma + p];
            parent[o] = (n == off_s[K + k]) ? anchor : n - 1;
            depth[o] = p;
            pos_id[o] = L + p;
            for (int w = 0; w < W; ++w)
                mrow[w] = range_bits(0, i, w) | range_bits(off_s[k], anchor, w) | range_bits(off_s[K + k], n, w);
        }
    }
}

int32_t launch_build_tree3(const int32_t* draft1, const int32_t* draft2, const int32_t* draft3,
                           const int32_t* prefix_len, const int32_t* third_len, const int32_t* ctx_len, int B,
                           int gamma, int K, int T_cap, int32_t* tokens, int32_t* parent, int32_t* depth,
                           int32_t* pos_id, int32_t* branch_off, uint32_t* mask, int32_t* tree_len, cudaStream_t s) {
    if (B == 0) return D2SD_OK;
    const int W = (T_cap + 31) / 32;
    int threads = ((T_cap + 31) / 32) * 32;
    if (threads > 256) threads = 256;
    if (threads < 32) threads = 32;
    cudaLaunchAttribute attr[1];
    cudaLaunchConfig_t cfg = sb_config(dim3(B), dim3(threads), s, attr);
    D2SD_CHECK_CUDA(cudaLaunchKernelEx(&cfg, build_tree3_kernel, draft1, draft2, draft3, prefix_len, third_len, ctx_len, gamma, K,
                                       T_cap, W, tokens, parent, depth, pos_id, branch_off, mask, tree_len));
    D2SD_CHECK_LAUNCH("build_tree3_kernel");
    return D2SD_OK;
}

}  // namespace d2sd
