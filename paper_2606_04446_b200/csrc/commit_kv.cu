// KV commit after acceptance.  PAPER.md:124 "commit the longest accepted prefix";
// :119 a cycle "consumes the verified KV caches ... and emits a new batch of accepted tokens"; :69
// "refreshed target hidden features that seed the next cycle".
// The verify pass computed K/V of every tree node; the rows of path[0..accept_len] (root = anchor, then
// the accepted draft tokens) are gathered into the cache at positions L..L+accept_len of every layer and
// the context grows by accept_len + 1.  Pure data movement (<= gamma rows x 2 KiB per kv tensor and
// layer), three launches, no host round trip:
//   commit_plan_kernel   one CTA: capacity per request, pages from the free list in request order
//                        (exclusive scan of the requests' page needs), rows that fit -> n_fit[b]
//   commit_copy_kernel   grid (row j, request, layer): 16-byte copies of one K row and one V row
//   commit_finish_kernel ctx_len_out = ctx_len + n_fit (may alias ctx_len), dropped, free_head
// The copy kernel reads the old ctx_len, hence the separate last step.
#include "common.cuh"

namespace d2sd {
namespace {

__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

constexpr int kPlanThreads = 1024;

// n_fit[b] and, with a free list, the new page-table entries.  A single CTA; requests are taken in
// blocks of kPlanThreads so the free-list hand-out keeps request order for any B.
__global__ void __launch_bounds__(kPlanThreads) commit_plan_kernel(CommitArgs a, int32_t* got_total) {
    __shared__ int scan_s[kPlanThreads];
    __shared__ int base_s;
    pdl_launch_dependents();
    pdl_wait();
    const int tid = threadIdx.x;
    if (tid == 0) base_s = a.free_pages ? *a.free_head : 0;
    __syncthreads();
    for (int b0 = 0; b0 < a.B; b0 += kPlanThreads) {
        const int b = b0 + tid;
        int L = 0, n_fit = 0, owned = 0, want = 0;
        if (b < a.B) {
            L = a.ctx_len[b];
            const int n = a.accept_len[b] + 1;
            long long cap;
            if (a.page_size > 0) cap = (long long)(a.kv_indptr[b + 1] - a.kv_indptr[b]) * a.page_size;
            else cap = a.kv_indptr ? (long long)(a.kv_indptr[b + 1] - a.kv_indptr[b]) : (long long)a.kv_rows;
            n_fit = n;
            if ((long long)L + n_fit > cap) n_fit = (int)(cap > L ? cap - L : 0);
            if (a.page_size > 0 && a.free_pages) {
                owned = (L + a.page_size - 1) / a.page_size;
                want = (L + n_fit + a.page_size - 1) / a.page_size - owned;
            }
        }
        // inclusive scan of `want` over the block of requests (Hillis-Steele in shared memory)
        scan_s[tid] = want;
        __syncthreads();
        for (int o = 1; o < kPlanThreads; o <<= 1) {
            const int v = tid >= o ? scan_s[tid - o] : 0;
            __syncthreads();
            scan_s[tid] += v;
            __syncthreads();
        }
        const int excl = scan_s[tid] - want;
        const int block_total = scan_s[kPlanThreads - 1];
        const int base = base_s;
        if (b < a.B) {
            if (a.page_size > 0 && a.free_pages) {
                int left = a.n_free - (base + excl);
                if (left < 0) left = 0;
                const int got = want < left ? want : left;
                for (int e = 0; e < got; ++e)
                    a.kv_indices[(size_t)a.kv_indptr[b] + owned + e] = a.free_pages[base + excl + e];
                const long long room = (long long)(owned + got) * a.page_size - L;
                if (n_fit > room) n_fit = (int)room;
            }
            a.n_fit[b] = n_fit;
        }
        __syncthreads();
        if (tid == 0) {
            const int nb = base + block_total;
            base_s = nb < a.n_free ? nb : (a.n_free > base ? a.n_free : base);
        }
        __syncthreads();
    }
    if (tid == 0) *got_total = base_s;
}

// grid = (gamma, B, n_layers), 128 threads: path position j of request b in one layer.
__global__ void __launch_bounds__(128) commit_copy_kernel(CommitArgs a) {
    pdl_launch_dependents();
    pdl_wait();
    const int j = blockIdx.x, b = blockIdx.y, layer = blockIdx.z;
    if (layer == 0 && a.feat_out) {  // target features of the accepted path, in path order, zero rows behind (:69)
        uint4* df = reinterpret_cast<uint4*>(a.feat_out + ((size_t)b * a.gamma + j) * a.F);
        if (j <= a.accept_len[b]) {
            const int nd = a.path[(size_t)b * a.gamma + j];
            const uint4* sf = reinterpret_cast<const uint4*>(a.feat + ((size_t)b * a.T_cap + nd) * a.F);
            for (int e = threadIdx.x; e < a.F / 8; e += blockDim.x) df[e] = sf[e];
        } else {
            for (int e = threadIdx.x; e < a.F / 8; e += blockDim.x) df[e] = make_uint4(0, 0, 0, 0);
        }
    }
    if (j >= a.n_fit[b]) return;
    const int node = a.path[(size_t)b * a.gamma + j];
    const int pos = a.ctx_len[b] + j;
    size_t row;
    if (a.page_size > 0)
        row = (size_t)a.kv_indices[(size_t)a.kv_indptr[b] + pos / a.page_size] * a.page_size + (size_t)(pos % a.page_size);
    else
        row = (size_t)(a.kv_indptr ? a.kv_indptr[b] : 0) + (size_t)pos;
    const size_t row_elems = (size_t)a.Hkv * a.d;
    const size_t src = (size_t)layer * a.tree_layer_stride + ((size_t)b * a.T_cap + node) * row_elems;
    const size_t dst = (size_t)layer * a.cache_layer_stride + row * row_elems;
    const int n16 = (int)(row_elems * 2 / 16);  // rows are whole 16-byte units (api.cu checks d % 8 == 0)
    const uint4* sk = reinterpret_cast<const uint4*>(a.tree_k + src);
    const uint4* sv = reinterpret_cast<const uint4*>(a.tree_v + src);
    uint4* dk = reinterpret_cast<uint4*>(a.k_cache + dst);
    uint4* dv = reinterpret_cast<uint4*>(a.v_cache + dst);
    for (int e = threadIdx.x; e < n16; e += blockDim.x) {
        const uint4 x = sk[e], y = sv[e];
        dk[e] = x;
        dv[e] = y;
    }
}

__global__ void __launch_bounds__(256) commit_finish_kernel(CommitArgs a, const int32_t* got_total) {
    pdl_launch_dependents();
    pdl_wait();
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b == 0 && a.free_pages) *a.free_head = *got_total;
    if (b >= a.B) return;
    const int n = a.accept_len[b] + 1, n_fit = a.n_fit[b];
    const int L = a.ctx_len[b];
    a.ctx_len_out[b] = L + n_fit;
    a.dropped[b] = n - n_fit;
}

cudaLaunchConfig_t pdl_config(dim3 grid, dim3 block, cudaStream_t s, cudaLaunchAttribute* attr) {
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

}  // namespace

int32_t launch_commit_kv(const CommitArgs& a, cudaStream_t s) {
    if (a.B == 0) return D2SD_OK;
    int32_t* got_total = a.n_fit + a.B;  // one more workspace word
    cudaLaunchAttribute attr[1];
    cudaLaunchConfig_t cfg = pdl_config(dim3(1), dim3(kPlanThreads), s, attr);
    D2SD_CHECK_CUDA(cudaLaunchKernelEx(&cfg, commit_plan_kernel, a, got_total));
    D2SD_CHECK_LAUNCH("commit_plan_kernel");
    cfg = pdl_config(dim3(a.gamma, a.B, a.n_layers), dim3(128), s, attr);
    D2SD_CHECK_CUDA(cudaLaunchKernelEx(&cfg, commit_copy_kernel, a));
    D2SD_CHECK_LAUNCH("commit_copy_kernel");
    cfg = pdl_config(dim3(ceil_div(a.B, 256)), dim3(256), s, attr);
    D2SD_CHECK_CUDA(cudaLaunchKernelEx(&cfg, commit_finish_kernel, a, (const int32_t*)got_total));
    D2SD_CHECK_LAUNCH("commit_finish_kernel");
    return D2SD_OK;
}

}  // namespace d2sd
