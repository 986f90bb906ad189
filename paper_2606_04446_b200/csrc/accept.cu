// Vocabulary scans: stage (d) argmax + longest-accepted-path walk and the drafter
// confidence extraction that feeds stage (a) (Eq. 3: t_k = argmax_v p_k(v), c_k = max_v p_k(v)).
// The scan is a pure HBM stream (rows*V bf16 values read once, 128-bit loads, no reuse -> no shared
// tensor cores): a CTA covers kScanChunk vocabulary entries of one row, brought into shared memory by
// two 16 KiB bulk copies (cp.async.bulk, mbarrier completion, evict-first) so that 32 KiB per CTA are in
// flight by construction; all CTAs of a launch are co-resident (4-5 per SM at config 2: ~150 KiB per SM).  The finishing kernels are
// launch-latency-sized and start under programmatic dependent launch.
#include <climits>

#include "common.cuh"

namespace d2sd {

struct ScanPart {  // partial state of one (row, chunk): maximum, its first index, sum of e^(x - maximum)
    float v;
    int32_t i;
    float s;
    float pad;
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
__device__ __forceinline__ float bf_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf_hi(uint32_t w) { return __uint_as_float(w & 0xFFFF0000u); }

__device__ __forceinline__ void arg_update_word(uint32_t w, int idx, float& bv, int& bi) {
    arg_update(bf_lo(w), idx, bv, bi);
    arg_update(bf_hi(w), idx + 1, bv, bi);
}
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

__device__ __forceinline__ void scan_mbar_wait(uint32_t bar) {  // phase 0 of a one-shot barrier
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "W_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], 0;\n\t"
        "@!p bra W_%=;\n\t}" ::"r"(bar)
        : "memory");
}

constexpr int kScanThreads = 256;
constexpr int kVec = kScanChunk / 8 / kScanThreads;  // 8 x 16 B in flight per thread
static_assert(kVec * 8 * kScanThreads == kScanChunk, "chunk = threads x vectors");

// softmax-state merge of (m, i, s) pairs: first-index maximum, sums rescaled to the common maximum
__device__ __forceinline__ void state_merge(float ov, int oi, float os, float& bv, int& bi, float& bs) {
    const float m = fmaxf(ov, bv);
    const float a = ov == m ? 1.f : __expf(ov - m), c = bv == m ? 1.f : __expf(bv - m);
    bs = (os > 0.f ? os * a : 0.f) + (bs > 0.f ? bs * c : 0.f);
    arg_update(ov, oi, bv, bi);
}

// grid = (rows, chunks).  Row r of group b = r / rows_per_group is skipped when its index inside the
// group is >= row_limit[b] (tree padding rows; row_limit == NULL: every row is real).  kSum: also the
// sum of e^(x - max) over the chunk (confidence extraction); otherwise argmax only.
template <bool kSum>
__global__ void __launch_bounds__(kScanThreads)
vocab_scan_kernel(const __nv_bfloat16* __restrict__ logits, int64_t row_stride, int V,
                  const int32_t* __restrict__ row_limit, int rows_per_group, int n_chunks,
                  ScanPart* __restrict__ part) {
    const int row = blockIdx.x;
    pdl_launch_dependents();
    pdl_wait();  // logits and row_limit (tree_len) are written by earlier kernels of the stream
    if (row_limit) {
        const int b = row / rows_per_group;
        if (row - b * rows_per_group >= row_limit[b]) return;  // padding rows are never read
    }
    const __nv_bfloat16* rowp = logits + (size_t)row * row_stride;
    const int start = blockIdx.y * kScanChunk;
    const int end = min(V, start + kScanChunk);
    const int tid = threadIdx.x;
    const bool aligned = (reinterpret_cast<uintptr_t>(rowp) & 15) == 0;
    __shared__ __align__(128) uint4 stage[kScanChunk / 8];
    __shared__ __align__(8) unsigned long long bars[2];
    __shared__ float red_v[kScanThreads / 32], red_s[kScanThreads / 32];
    __shared__ int red_i;
    // Two passes over the thread's 64 values, both out of registers.  Pass 1 is the maximum alone, two bf16
    // values per instruction (max.bf16x2 returns the other operand for a NaN, so NaNs drop out); the block
    // agrees on it; pass 2 -- only in the threads that hold the maximum -- finds its first index.  The index
    // bookkeeping of a one-pass argmax (two compares and two selects per value) made the scan ALU-bound.
    uint4 x[kVec];
    int nvec = 0;
    float xt = -INFINITY;  // this thread's element of the < 8 values behind the last whole vector
    float m = -INFINITY;
    if (aligned) {
        // The chunk is staged through shared memory by two bulk copies (one elected thread, mbarrier
        // completion): 32 KiB per CTA are in flight whatever the compiler does with the consuming loop
        // (ptxas interleaves plain vector loads with their compares and keeps only two in flight).
        nvec = (end - start) >> 3;
        const uint32_t bar0 = (uint32_t)__cvta_generic_to_shared(bars);
        const uint32_t st0 = (uint32_t)__cvta_generic_to_shared(stage);
        const int nv0 = min(nvec, kScanChunk / 16), nv1 = nvec - nv0;  // first / second half
        if (tid == 0) {
            red_i = INT_MAX;
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar0));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar0 + 8));
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            const char* src = reinterpret_cast<const char*>(rowp + start);
            if (nv0 > 0) {
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar0), "r"(nv0 * 16) : "memory");
                asm volatile(
                    "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                    ::"r"(st0), "l"(src), "r"(nv0 * 16), "r"(bar0), "l"(0x12F0000000000000ull) : "memory");
            }
            if (nv1 > 0) {
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar0 + 8), "r"(nv1 * 16) : "memory");
                asm volatile(
                    "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                    ::"r"(st0 + nv0 * 16), "l"(src + (size_t)nv0 * 16), "r"(nv1 * 16), "r"(bar0 + 8),
                    "l"(0x12F0000000000000ull) : "memory");
            }
        }
        const int tail0 = start + nvec * 8;
        if (tail0 + tid < end) xt = __bfloat162float(rowp[tail0 + tid]);
        __syncthreads();  // barrier initialisation visible to the waiting threads
#pragma unroll
        for (int u = 0; u < kVec; ++u) {
            if (u == 0 && nv0 > 0) scan_mbar_wait(bar0);
            if (u == kVec / 2 && nv1 > 0) scan_mbar_wait(bar0 + 8);
            const int v = tid + u * kScanThreads;  // absent vectors hold -inf
            x[u] = v < nvec ? stage[v] : make_uint4(0xFF80FF80u, 0xFF80FF80u, 0xFF80FF80u, 0xFF80FF80u);
        }
        uint32_t m2[4] = {0xFF80FF80u, 0xFF80FF80u, 0xFF80FF80u, 0xFF80FF80u};
#pragma unroll
        for (int u = 0; u < kVec; ++u) {
            asm("max.bf16x2 %0, %0, %1;" : "+r"(m2[0]) : "r"(x[u].x));
            asm("max.bf16x2 %0, %0, %1;" : "+r"(m2[1]) : "r"(x[u].y));
            asm("max.bf16x2 %0, %0, %1;" : "+r"(m2[2]) : "r"(x[u].z));
            asm("max.bf16x2 %0, %0, %1;" : "+r"(m2[3]) : "r"(x[u].w));
        }
        asm("max.bf16x2 %0, %0, %1;" : "+r"(m2[0]) : "r"(m2[1]));
        asm("max.bf16x2 %0, %0, %1;" : "+r"(m2[2]) : "r"(m2[3]));
        asm("max.bf16x2 %0, %0, %1;" : "+r"(m2[0]) : "r"(m2[2]));
        m = fmaxf(fmaxf(bf_lo(m2[0]), bf_hi(m2[0])), xt);  // fmaxf drops a NaN as well
    } else {  // misaligned row start (odd strides): plain loads
        if (tid == 0) red_i = INT_MAX;
        for (int i = start + tid; i < end; i += kScanThreads) m = fmaxf(m, __bfloat162float(rowp[i]));
        __syncthreads();
    }
    // the block's maximum
    float mb = m;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mb = fmaxf(mb, __shfl_xor_sync(0xffffffffu, mb, o));
    if ((tid & 31) == 0) red_v[tid >> 5] = mb;
    __syncthreads();
    mb = red_v[0];
#pragma unroll
    for (int w = 1; w < kScanThreads / 32; ++w) mb = fmaxf(mb, red_v[w]);
    // its first index (IEEE equality: -0 == +0, a NaN never matches), and the sum of e^(x - max)
    float bs = 0.f;
    if (aligned) {
        if (m == mb) {
            int cand = INT_MAX;
#pragma unroll
            for (int u = 0; u < kVec; ++u) {  // (unrolled: x stays in registers)
                const int v = tid + u * kScanThreads;
                if (cand != INT_MAX || v >= nvec) continue;
                const uint32_t w[4] = {x[u].x, x[u].y, x[u].z, x[u].w};
#pragma unroll
                for (int e = 3; e >= 0; --e) {
                    if (bf_hi(w[e]) == mb) cand = start + v * 8 + 2 * e + 1;
                    if (bf_lo(w[e]) == mb) cand = start + v * 8 + 2 * e;
                }
            }
            if (cand == INT_MAX && xt == mb) cand = start + nvec * 8 + tid;
            if (cand != INT_MAX) atomicMin(&red_i, cand);
        }
        if (kSum && mb > -INFINITY) {
#pragma unroll
            for (int u = 0; u < kVec; ++u) {
                const uint32_t w[4] = {x[u].x, x[u].y, x[u].z, x[u].w};
#pragma unroll
                for (int e = 0; e < 4; ++e) bs += __expf(bf_lo(w[e]) - mb) + __expf(bf_hi(w[e]) - mb);
            }
            bs += __expf(xt - mb);
        }
    } else {
        if (m == mb) {
            for (int i = start + tid; i < end; i += kScanThreads)
                if (__bfloat162float(rowp[i]) == mb) {
                    atomicMin(&red_i, i);
                    break;
                }
        }
        if (kSum && mb > -INFINITY)
            for (int i = start + tid; i < end; i += kScanThreads) bs += __expf(__bfloat162float(rowp[i]) - mb);
    }
    if (kSum) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) bs += __shfl_xor_sync(0xffffffffu, bs, o);
        if ((tid & 31) == 0) red_s[tid >> 5] = bs;
    }
    __syncthreads();
    if (tid == 0) {
        if (kSum)
            for (int w = 1; w < kScanThreads / 32; ++w) bs += red_s[w];
        part[(size_t)row * n_chunks + blockIdx.y] = ScanPart{mb, red_i, bs, 0.f};
    }
}

// grid = B.  Finishes the argmax per node, then walks the tree:
//   ok[n] = every edge on the path root..n has tokens[child] == a[parent]
//   best  = deepest ok node, ties -> smallest node index.
__global__ void __launch_bounds__(256)
accept_walk_kernel(const ScanPart* __restrict__ part, int n_chunks, const int32_t* __restrict__ tokens,
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
    const int tid = threadIdx.x;
    pdl_launch_dependents();
    pdl_wait();
    const int T = tree_len[b];
    for (int n = tid; n < T_cap; n += blockDim.x) {
        const size_t o = (size_t)b * T_cap + n;
        int a = -1;
        if (n < T) {
            float bv = -INFINITY;
            int bi = INT_MAX;
            const ScanPart* p = part + o * n_chunks;
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

// grid = ceil(B*gamma / 128).  One thread per (request, block position): merges the chunk states of a
// drafter row into t_k and c_k = e^(x_t - m) / sum_v e^(x_v - m) = 1 / sum (Eq. 3); slot 0 = (anchor, 1).
__global__ void __launch_bounds__(128)
confidence_finish_kernel(const ScanPart* __restrict__ part, int n_chunks, const int32_t* __restrict__ anchor,
                         int B, int gamma, int32_t* __restrict__ draft, float* __restrict__ conf) {
    pdl_launch_dependents();
    pdl_wait();
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= B * gamma) return;
    const int b = e / gamma, k = e - b * gamma;
    if (k == 0) {
        draft[e] = anchor[b];
        conf[e] = 1.0f;
        return;
    }
    const ScanPart* p = part + ((size_t)b * (gamma - 1) + (k - 1)) * n_chunks;
    float bv = -INFINITY, bs = 0.f;
    int bi = INT_MAX;
    for (int c = 0; c < n_chunks; ++c) state_merge(p[c].v, p[c].i, p[c].s, bv, bi, bs);
    draft[e] = bi == INT_MAX ? 0 : bi;
    conf[e] = bs > 0.f ? 1.0f / bs : 0.f;
}

static cudaLaunchConfig_t pdl_config(dim3 grid, dim3 block, size_t smem, cudaStream_t s, cudaLaunchAttribute* attr) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cfg;
}

int32_t launch_accept(const __nv_bfloat16* logits, int64_t row_stride, int V, const int32_t* tokens,
                      const int32_t* parent, const int32_t* depth, const int32_t* tree_len, int B,
                      int gamma, int T_cap, int32_t* argmax_out, int32_t* accept_len, int32_t* path,
                      int32_t* bonus, int32_t* best_node, void* workspace, cudaStream_t s) {
    if (B == 0) return D2SD_OK;
    const int n_chunks = ceil_div(V, kScanChunk);
    ScanPart* part = static_cast<ScanPart*>(workspace);
    cudaLaunchAttribute attr[1];
    cudaLaunchConfig_t cfg = pdl_config(dim3(B * T_cap, n_chunks), dim3(kScanThreads), 0, s, attr);
    D2SD_CHECK_CUDA(cudaLaunchKernelEx(&cfg, vocab_scan_kernel<false>, logits, row_stride, V, tree_len, T_cap, n_chunks,
                                       part));
    D2SD_CHECK_LAUNCH("vocab_scan_kernel<argmax>");
    cfg = pdl_config(dim3(B), dim3(256), 3 * T_cap * sizeof(int32_t), s, attr);
    D2SD_CHECK_CUDA(cudaLaunchKernelEx(&cfg, accept_walk_kernel, (const ScanPart*)part, n_chunks, tokens, parent, depth,
                                       tree_len, gamma, T_cap, argmax_out, accept_len, path, bonus, best_node));
    D2SD_CHECK_LAUNCH("accept_walk_kernel");
    return D2SD_OK;
}

int32_t launch_confidence(const __nv_bfloat16* logits, int64_t row_stride, int V, const int32_t* anchor, int B,
                          int gamma, int32_t* draft, float* conf, void* workspace, cudaStream_t s) {
    if (B == 0) return D2SD_OK;
    const int n_chunks = ceil_div(V, kScanChunk);
    ScanPart* part = static_cast<ScanPart*>(workspace);
    cudaLaunchAttribute attr[1];
    cudaLaunchConfig_t cfg = pdl_config(dim3(B * (gamma - 1), n_chunks), dim3(kScanThreads), 0, s, attr);
    D2SD_CHECK_CUDA(cudaLaunchKernelEx(&cfg, vocab_scan_kernel<true>, logits, row_stride, V, (const int32_t*)nullptr,
                                       gamma - 1, n_chunks, part));
    D2SD_CHECK_LAUNCH("vocab_scan_kernel<softmax>");
    cfg = pdl_config(dim3(ceil_div(B * gamma, 128)), dim3(128), 0, s, attr);
    D2SD_CHECK_CUDA(cudaLaunchKernelEx(&cfg, confidence_finish_kernel, (const ScanPart*)part, n_chunks, anchor, B, gamma,
                                       draft, conf));
    D2SD_CHECK_LAUNCH("confidence_finish_kernel");
    return D2SD_OK;
}

// ---- d2sd_accept_static: the same two launches with the chunk states in a file-scope device array -----------
// For callers that cannot provide (or allocate) a workspace.  The array costs kStaticScratchBytes of device
// memory on every GPU that loads the library, until exit.  In host code `g_accept_scratch` is only a stand-in
// for the symbol, not a device address: the address the kernels get comes from cudaGetSymbolAddress, asked
// once per device with that device current.
constexpr size_t kStaticScratchBytes = 1u << 20;  // 65536 chunk states of 16 B (config 5 needs 11200)
static __device__ __align__(256) unsigned char g_accept_scratch[kStaticScratchBytes];
static_assert(sizeof(ScanPart) == kScanPartBytes, "chunk state size");

static int32_t accept_scratch_address(void** out) {
    static void* addr[64] = {};  // per device; a race between two first callers repeats an idempotent query
    int dev = 0;
    D2SD_CHECK_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return set_error(D2SD_ERR_UNSUPPORTED, "device ordinal %d outside [0,64)", dev);
    if (!addr[dev]) {
        void* p = nullptr;
        D2SD_CHECK_CUDA(cudaGetSymbolAddress(&p, g_accept_scratch));
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255)) return set_error(D2SD_ERR_CUDA, "static scratch at %p", p);
        addr[dev] = p;
    }
    *out = addr[dev];
    return D2SD_OK;
}

}  // namespace d2sd

using namespace d2sd;

extern "C" size_t d2sd_accept_static_max_bytes(void) { return kStaticScratchBytes; }

extern "C" int32_t d2sd_accept_static(const void* logits, int64_t row_stride, int32_t V, const int32_t* tokens,
                                      const int32_t* parent, const int32_t* depth, const int32_t* tree_len,
                                      int32_t B, int32_t gamma, int32_t T_cap, int32_t* argmax_out,
                                      int32_t* accept_len, int32_t* path, int32_t* bonus, int32_t* best_node,
                                      void* stream) {
    clear_error();
    D2SD_CHECK_ARG(B >= 0 && V >= 1 && row_stride >= V, "B = %d, V = %d, row_stride = %lld", B, V,
                   (long long)row_stride);
    D2SD_CHECK_ARG(gamma >= 2 && gamma <= 64, "gamma = %d outside [2,64]", gamma);
    D2SD_CHECK_ARG(T_cap >= 1, "T_cap = %d", T_cap);
    D2SD_CHECK_SUPPORTED(T_cap <= 1024, "T_cap = %d > 1024", T_cap);
    D2SD_CHECK_SUPPORTED(ceil_div(V, kScanChunk) <= 65535, "V = %d too large", V);
    const size_t need = (size_t)B * T_cap * ceil_div(V, kScanChunk) * sizeof(ScanPart);
    D2SD_CHECK_SUPPORTED(need <= kStaticScratchBytes,
                         "d2sd_accept_static: B*T_cap*ceil(V/%d) = %zu chunk states need %zu bytes, the built-in scratch "
                         "holds %zu; use d2sd_accept with a caller workspace",
                         kScanChunk, need / sizeof(ScanPart), need, kStaticScratchBytes);
    if (B == 0) return D2SD_OK;
    D2SD_CHECK_ARG(logits && tokens && parent && depth && tree_len && argmax_out && accept_len && path &&
                       bonus && best_node,
                   "a required buffer is NULL");
    void* scratch = nullptr;
    if (int32_t st = accept_scratch_address(&scratch)) return st;
    // nothing in the scratch has to start at zero: the scan writes the state of every (real row, chunk) and the
    // walk reads exactly those, so the previous call's contents are never seen
    return launch_accept(static_cast<const __nv_bfloat16*>(logits), row_stride, V, tokens, parent, depth, tree_len, B,
                         gamma, T_cap, argmax_out, accept_len, path, bonus, best_node, scratch,
                         static_cast<cudaStream_t>(stream));
}
