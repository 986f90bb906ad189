// Stage (d): vocab-wide argmax + longest-accepted-path walk.  PAPER.md:69, :124.
// Kernel 1 is a pure HBM scan (T*V bf16 values read once, 128-bit loads, no reuse -> no shared
// memory staging, no tensor cores); kernel 2 is launch-latency-sized.
#include <climits>

#include "common.cuh"

namespace d2sd {

struct ArgPart {
    float v;
    int32_t i;
};

// "x at index xi beats the current best": larger value, or equal value (IEEE: -0 == +0) at a
// smaller index.  With best initialised to (-inf, INT_MAX) this also handles all -inf rows.
__device__ __forceinline__ void arg_update(float x, int xi, float& bv, int& bi) {
    if (x > bv || (x == bv && xi < bi)) {
        bv = x;
        bi = xi;
    }
}

__device__ __forceinline__ uint4 ld_stream_16B(const void* p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}

__device__ __forceinline__ void arg_update_word(uint32_t w, int idx, float& bv, int& bi) {
    arg_update(__uint_as_float(w << 16), idx, bv, bi);
    arg_update(__uint_as_float(w & 0xFFFF0000u), idx + 1, bv, bi);
}

constexpr int kArgmaxThreads = 256;
constexpr int kArgmaxVecPerThread = kArgmaxChunk / 8 / kArgmaxThreads;  // 4 x 16 B in flight

// grid = (B*T_cap, chunks).  Each CTA scans kArgmaxChunk vocabulary entries of one logits row.
__global__ void __launch_bounds__(kArgmaxThreads)
argmax_partial_kernel(const __nv_bfloat16* __restrict__ logits, int64_t row_stride, int V,
                      const int32_t* __restrict__ tree_len, int T_cap, int n_chunks,
                      ArgPart* __restrict__ part) {
    const int row = blockIdx.x;
    const int b = row / T_cap, n = row - b * T_cap;
    if (n >= tree_len[b]) return;  // padding rows are never read
    const __nv_bfloat16* rowp = logits + (size_t)row * row_stride;
    const int start = blockIdx.y * kArgmaxChunk;
    const int end = min(V, start + kArgmaxChunk);
    float bv = -INFINITY;
    int bi = INT_MAX;
    const int tid = threadIdx.x;
    if ((reinterpret_cast<uintptr_t>(rowp) & 15) == 0) {
        const int nvec = (end - start) >> 3;
        const uint4* vp = reinterpret_cast<const uint4*>(rowp + start);
        uint4 x[kArgmaxVecPerThread];
#pragma unroll
        for (int u = 0; u < kArgmaxVecPerThread; ++u) {
            const int v = tid + u * kArgmaxThreads;
            if (v < nvec) x[u] = ld_stream_16B(vp + v);
        }
#pragma unroll
        for (int u = 0; u < kArgmaxVecPerThread; ++u) {
            const int v = tid + u * kArgmaxThreads;
            if (v < nvec) {
                const int idx = start + v * 8;
                arg_update_word(x[u].x, idx, bv, bi);
                arg_update_word(x[u].y, idx + 2, bv, bi);
                arg_update_word(x[u].z, idx + 4, bv, bi);
                arg_update_word(x[u].w, idx + 6, bv, bi);
            }
        }
        for (int i = start + nvec * 8 + tid; i < end; i += kArgmaxThreads)
            arg_update(__bfloat162float(rowp[i]), i, bv, bi);
    } else {
        for (int i = start + tid; i < end; i += kArgmaxThreads)
            arg_update(__bfloat162float(rowp[i]), i, bv, bi);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float ov = __shfl_xor_sync(0xffffffffu, bv, o);
        const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
        arg_update(ov, oi, bv, bi);
    }
    __shared__ float sv[kArgmaxThreads / 32];
    __shared__ int si[kArgmaxThreads / 32];
    if ((tid & 31) == 0) {
        sv[tid >> 5] = bv;
        si[tid >> 5] = bi;
    }
    __syncthreads();
    if (tid == 0) {
        for (int w = 1; w < kArgmaxThreads / 32; ++w) arg_update(sv[w], si[w], bv, bi);
        part[(size_t)row * n_chunks + blockIdx.y] = ArgPart{bv, bi};
    }
}

// grid = B.  Finishes the argmax per node, then walks the tree:
//   ok[n] = every edge on the path root..n has tokens[child] == a[parent]
//   best  = deepest ok node, ties -> smallest node index.
__global__ void __launch_bounds__(256)
accept_walk_kernel(const ArgPart* __restrict__ part, int n_chunks, const int32_t* __restrict__ tokens,
                   const int32_t* __restrict__ parent, const int32_t* __restrict__ depth,
                   const int32_t* __restrict__ tree_len, int gamma, int T_cap,
                   int32_t* __restrict__ argmax_out, int32_t* __restrict__ accept_len,
                   int32_t* __restrict__ path, int32_t* __restrict__ bonus,
                   int32_t* __restrict__ best_node) {
    extern __shared__ int32_t sm[];
    int32_t* a_s = sm;              // [T_cap]
    int32_t* par_s = sm + T_cap;    // [T_cap]
    int32_t* tok_s = sm + 2 * T_cap;
    __shared__ int red_s[8];
    const int b = blockIdx.x;
    const int T = tree_len[b];
    const int tid = threadIdx.x;
    for (int n = tid; n < T_cap; n += blockDim.x) {
        const size_t o = (size_t)b * T_cap + n;
        int a = -1;
        if (n < T) {
            float bv = -INFINITY;
            int bi = INT_MAX;
            const ArgPart* p = part + o * n_chunks;
            for (int c = 0; c < n_chunks; ++c) arg_update(p[c].v, p[c].i, bv, bi);
            a = bi == INT_MAX ? 0 : bi;  // a row of NaNs only: index 0, never an out-of-range token id
            par_s[n] = parent[o];
            tok_s[n] = tokens[o];
        }
        a_s[n] = a;
        argmax_out[o] = a;
    }
    __syncthreads();
    int key = -1;
    for (int n = tid; n < T; n += blockDim.x) {
        bool ok = true;
        for (int m = n; m > 0;) {
            const int p = par_s[m];
            if (tok_s[m] != a_s[p]) { ok = false; break; }
            m = p;
        }
        if (ok) key = max(key, (depth[(size_t)b * T_cap + n] << 11) | (2047 - n));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) key = max(key, __shfl_xor_sync(0xffffffffu, key, o));
    if ((tid & 31) == 0) red_s[tid >> 5] = key;
    __syncthreads();
    if (tid == 0) {
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) key = max(key, red_s[w]);
        const int best = 2047 - (key & 2047);
        const int len = key >> 11;
        accept_len[b] = len;
        best_node[b] = best;
        bonus[b] = a_s[best];
        int32_t* pth = path + (size_t)b * gamma;
        for (int j = len + 1; j < gamma; ++j) pth[j] = -1;
        int m = best;
        for (int j = len; j >= 0; --j) {
            pth[j] = m;
            m = par_s[m];
        }
    }
}

int32_t launch_accept(const __nv_bfloat16* logits, int64_t row_stride, int V, const int32_t* tokens,
                      const int32_t* parent, const int32_t* depth, const int32_t* tree_len, int B,
                      int gamma, int T_cap, int32_t* argmax_out, int32_t* accept_len, int32_t* path,
                      int32_t* bonus, int32_t* best_node, void* workspace, cudaStream_t s) {
    if (B == 0) return D2SD_OK;
    const int n_chunks = ceil_div(V, kArgmaxChunk);
    ArgPart* part = static_cast<ArgPart*>(workspace);
    dim3 grid(B * T_cap, n_chunks);
    argmax_partial_kernel<<<grid, kArgmaxThreads, 0, s>>>(logits, row_stride, V, tree_len, T_cap, n_chunks,
                                                         part);
    D2SD_CHECK_LAUNCH("argmax_partial_kernel");
    accept_walk_kernel<<<B, 256, 3 * T_cap * sizeof(int32_t), s>>>(part, n_chunks, tokens, parent, depth,
                                                                   tree_len, gamma, T_cap, argmax_out,
                                                                   accept_len, path, bonus, best_node);
    D2SD_CHECK_LAUNCH("accept_walk_kernel");
    return D2SD_OK;
}

}  // namespace d2sd
