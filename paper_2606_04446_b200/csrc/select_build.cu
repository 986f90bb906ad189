// Stage (a) top-K prefix selection and stage (b) shared-prefix tree build.
// PAPER.md:87-105 (Eq. 3-5), :107, :123-124.  Launch-latency-sized kernels: one CTA per request.
#include "common.cuh"

namespace d2sd {

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
    select_prefixes_kernel<<<B, 32, 0, s>>>(conf, gamma, K, prefix_len, r_out);
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
    build_tree_kernel<<<B, threads, 0, s>>>(draft1, draft2, prefix_len, ctx_len, gamma, K, T_cap, W, tokens,
                                            parent, depth, pos_id, branch_off, mask, tree_len);
    D2SD_CHECK_LAUNCH("build_tree_kernel");
    return D2SD_OK;
}

}  // namespace d2sd
