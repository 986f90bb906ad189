// Stage (c), generic path: split-KV flash attention on mma.sync (m16n8k16 bf16, fp32 accumulate).
// Serves the shapes the fused tcgen05 kernels (attn_stream_sm100.cu, attn_duo_sm100.cu) do not cover -- GQA group sizes
// that do not divide a 128-row query tile -- and impl = 1 (tests: an independent second CUDA path):
// prefix chunks and the tree pass (<= T_cap keys under the ancestor mask) as one launch, merge as a
// second.  Contiguous and paged KV.  PAPER.md:52, :124, :154.
//
// CTA = 4 warps x 16 query rows = 64 rows of one (request, kv head); rows are the flattened
// (tree node t, head-in-group) pairs r = t*G + hh so that all GQA heads and all branches share one
// pass over the kv head's keys.  Keys arrive in 64-key tiles through a cp.async double buffer.
#include "common.cuh"

namespace d2sd {
namespace {

constexpr int D = 128;
constexpr int BM = 64;
constexpr int BN = 64;
constexpr int LDSM = D + 8;  // padded smem row (272 B): conflict-free fragment loads and ldmatrix
constexpr int NT = 128;
constexpr int SMEM_BYTES = 2 /*K,V*/ * 2 /*stages*/ * BN * LDSM * 2;

__device__ __forceinline__ void cp_async_16(uint32_t dst, const void* src, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;" ::"n"(N));
}

__device__ __forceinline__ void mma_bf16(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm volatile(
        "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, "
        "{%0,%1,%2,%3};"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
    __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&v);
}

struct KvSource {
    const __nv_bfloat16* k;
    const __nv_bfloat16* v;
    const int32_t* pages;  // paged: page ids of this request; else nullptr
    int64_t row0;          // contiguous / tree: first row of this request
    int page_size;
    int Hkv, g;
    __device__ __forceinline__ size_t row_elem(int j) const {
        int64_t row;
        if (pages) {
            row = (int64_t)pages[j / page_size] * page_size + (j % page_size);
        } else {
            row = row0 + j;
        }
        return ((size_t)row * Hkv + g) * D;
    }
};

__global__ void __launch_bounds__(NT)
attn_mma_kernel(AttnPlan pl, AttnArgs a, int split_first) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __nv_bfloat16* Ks = reinterpret_cast<__nv_bfloat16*>(smem_raw);  // [2][BN][LDSM]
    __nv_bfloat16* Vs = Ks + 2 * BN * LDSM;                           // [2][BN][LDSM]

    const int split = split_first + blockIdx.y;
    const int b = blockIdx.z / pl.Hkv;
    const int g = blockIdx.z - b * pl.Hkv;
    const int G = pl.G;
    const int T = a.tree_len[b];
    const int rows_valid = T * G;
    const int row_base = blockIdx.x * BM;
    if (row_base >= rows_valid) return;
    const bool is_tree = (split == pl.num_splits);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int quad = lane >> 2, tq = lane & 3;

    // this thread's two rows
    const int r0 = row_base + warp * 16 + quad, r1 = r0 + 8;
    const bool v0 = r0 < rows_valid, v1 = r1 < rows_valid;
    const int t0 = r0 / G, t1 = r1 / G;
    const int h0 = g * G + (r0 - t0 * G), h1 = g * G + (r1 - t1 * G);
    float* po = a.part_o + (((size_t)b * pl.NS + split) * pl.T_cap) * pl.Hq * D;
    float* plse = a.part_lse + (((size_t)b * pl.NS + split) * pl.T_cap) * pl.Hq;

    KvSource src;
    int k_begin, k_end;
    src.Hkv = pl.Hkv;
    src.g = g;
    src.page_size = pl.page_size;
    if (is_tree) {
        src.k = a.tree_k;
        src.v = a.tree_v;
        src.pages = nullptr;
        src.row0 = (int64_t)b * pl.T_cap;
        k_begin = 0;
        const int max_t = min(T - 1, (row_base + BM - 1) / G);  // row n has no mask bit above n
        k_end = max_t + 1;
    } else {
        src.k = a.k_cache;
        src.v = a.v_cache;
        const int L = a.ctx_len[b];
        const int base = a.kv_indptr ? a.kv_indptr[b] : 0;
        src.pages = pl.page_size > 0 ? a.kv_indices + base : nullptr;
        src.row0 = base;
        k_begin = split * pl.chunk_keys;
        k_end = min(L, k_begin + pl.chunk_keys);
        if (k_begin >= k_end) {  // empty chunk: state (O = 0, LSE = -inf); O is never read
            if (tid < BM && row_base + tid < rows_valid) {
                const int r = row_base + tid, t = r / G;
                plse[(size_t)t * pl.Hq + g * G + (r - t * G)] = -INFINITY;
            }
            return;
        }
    }

    const uint32_t ks_u32 = (uint32_t)__cvta_generic_to_shared(Ks);
    const uint32_t vs_u32 = (uint32_t)__cvta_generic_to_shared(Vs);
    auto load_tile = [&](int tile, int stage) {
        const int j0 = k_begin + tile * BN;
#pragma unroll
        for (int it = 0; it < (BN * D / 8) / NT; ++it) {
            const int c = tid + it * NT;
            const int key = c >> 4, part = c & 15;
            const int j = j0 + key;
            const bool ok = j < k_end;
            const size_t e = ok ? src.row_elem(j) + part * 8 : 0;
            const uint32_t off = (uint32_t)(((stage * BN + key) * LDSM + part * 8) * 2);
            cp_async_16(ks_u32 + off, src.k + e, ok ? 16 : 0);  // src-size 0 => zero fill
            cp_async_16(vs_u32 + off, src.v + e, ok ? 16 : 0);
        }
        cp_async_commit();
    };

    const int n_tiles = (k_end - k_begin + BN - 1) / BN;
    load_tile(0, 0);

    // Q fragments (A operand, row-major 16x16 per k-step), straight from global memory.
    uint32_t qf[8][4];
    {
        const __nv_bfloat16* q0 = a.q + (((size_t)b * pl.T_cap + (v0 ? t0 : 0)) * pl.Hq + (v0 ? h0 : 0)) * D;
        const __nv_bfloat16* q1 = a.q + (((size_t)b * pl.T_cap + (v1 ? t1 : 0)) * pl.Hq + (v1 ? h1 : 0)) * D;
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
            const int c = ks * 16 + tq * 2;
            qf[ks][0] = v0 ? *reinterpret_cast<const uint32_t*>(q0 + c) : 0u;
            qf[ks][1] = v1 ? *reinterpret_cast<const uint32_t*>(q1 + c) : 0u;
            qf[ks][2] = v0 ? *reinterpret_cast<const uint32_t*>(q0 + c + 8) : 0u;
            qf[ks][3] = v1 ? *reinterpret_cast<const uint32_t*>(q1 + c + 8) : 0u;
        }
    }
    const uint32_t* mrow0 = a.mask + ((size_t)b * pl.T_cap + (v0 ? t0 : 0)) * pl.W;
    const uint32_t* mrow1 = a.mask + ((size_t)b * pl.T_cap + (v1 ? t1 : 0)) * pl.W;

    const float c2 = pl.sm_scale * 1.4426950408889634f;  // scores -> log2 domain
    float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;
    float oacc[16][4];
#pragma unroll
    for (int i = 0; i < 16; ++i) oacc[i][0] = oacc[i][1] = oacc[i][2] = oacc[i][3] = 0.f;

    for (int tile = 0; tile < n_tiles; ++tile) {
        const int stage = tile & 1;
        if (tile + 1 < n_tiles) {
            load_tile(tile + 1, stage ^ 1);
            cp_async_wait<1>();
        } else {
            cp_async_wait<0>();
        }
        __syncthreads();
        const __nv_bfloat16* Kt = Ks + stage * BN * LDSM;
        const uint32_t vt_u32 = vs_u32 + (uint32_t)(stage * BN * LDSM * 2);

        float s[8][4];
#pragma unroll
        for (int nt = 0; nt < 8; ++nt) s[nt][0] = s[nt][1] = s[nt][2] = s[nt][3] = 0.f;
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
#pragma unroll
            for (int nt = 0; nt < 8; ++nt) {
                const __nv_bfloat16* kr = Kt + (nt * 8 + quad) * LDSM + ks * 16 + tq * 2;
                mma_bf16(s[nt], qf[ks], *reinterpret_cast<const uint32_t*>(kr),
                         *reinterpret_cast<const uint32_t*>(kr + 8));
            }
        }
        // bounds + ancestor mask
        const int j0 = k_begin + tile * BN;
        uint32_t w00 = 0xFFFFFFFFu, w01 = 0xFFFFFFFFu, w10 = 0xFFFFFFFFu, w11 = 0xFFFFFFFFu;
        if (is_tree) {
            const int wi = j0 >> 5;
            w00 = v0 ? mrow0[wi] : 0u;
            w10 = v1 ? mrow1[wi] : 0u;
            w01 = (v0 && wi + 1 < pl.W) ? mrow0[wi + 1] : 0u;
            w11 = (v1 && wi + 1 < pl.W) ? mrow1[wi + 1] : 0u;
        }
        const bool full = !is_tree && (j0 + BN <= k_end);
        if (!full) {
#pragma unroll
            for (int nt = 0; nt < 8; ++nt) {
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int kb = nt * 8 + tq * 2 + e;
                    const bool inb = j0 + kb < k_end;
                    const uint32_t wa = kb < 32 ? w00 : w01, wb = kb < 32 ? w10 : w11;
                    if (!(inb && ((wa >> (kb & 31)) & 1u))) s[nt][e] = -INFINITY;
                    if (!(inb && ((wb >> (kb & 31)) & 1u))) s[nt][2 + e] = -INFINITY;
                }
            }
        }
        // online softmax
        float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
        for (int nt = 0; nt < 8; ++nt) {
            mx0 = fmaxf(mx0, fmaxf(s[nt][0], s[nt][1]));
            mx1 = fmaxf(mx1, fmaxf(s[nt][2], s[nt][3]));
        }
        mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 1));
        mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 2));
        mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 1));
        mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 2));
        const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);
        const float mu0 = (mn0 == -INFINITY) ? 0.f : mn0, mu1 = (mn1 == -INFINITY) ? 0.f : mn1;
        const float al0 = exp2f((m0 - mu0) * c2), al1 = exp2f((m1 - mu1) * c2);
        m0 = mn0;
        m1 = mn1;
        const float ms0 = mu0 * c2, ms1 = mu1 * c2;
        float sum0 = 0.f, sum1 = 0.f;
#pragma unroll
        for (int nt = 0; nt < 8; ++nt) {
            s[nt][0] = exp2f(s[nt][0] * c2 - ms0);
            s[nt][1] = exp2f(s[nt][1] * c2 - ms0);
            s[nt][2] = exp2f(s[nt][2] * c2 - ms1);
            s[nt][3] = exp2f(s[nt][3] * c2 - ms1);
            sum0 += s[nt][0] + s[nt][1];
            sum1 += s[nt][2] + s[nt][3];
        }
        l0 = l0 * al0 + sum0;
        l1 = l1 * al1 + sum1;
#pragma unroll
        for (int dn = 0; dn < 16; ++dn) {
            oacc[dn][0] *= al0;
            oacc[dn][1] *= al0;
            oacc[dn][2] *= al1;
            oacc[dn][3] *= al1;
        }
        // O += P V
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
            uint32_t pa[4];
            pa[0] = pack_bf16(s[2 * kk][0], s[2 * kk][1]);
            pa[1] = pack_bf16(s[2 * kk][2], s[2 * kk][3]);
            pa[2] = pack_bf16(s[2 * kk + 1][0], s[2 * kk + 1][1]);
            pa[3] = pack_bf16(s[2 * kk + 1][2], s[2 * kk + 1][3]);
            const int mat = lane >> 3, rin = lane & 7;
            const int key = kk * 16 + (mat & 1) * 8 + rin;
#pragma unroll
            for (int dn = 0; dn < 16; dn += 2) {
                const uint32_t addr = vt_u32 + (uint32_t)((key * LDSM + (dn + (mat >> 1)) * 8) * 2);
                uint32_t b0, b1, b2, b3;
                asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                             : "=r"(b0), "=r"(b1), "=r"(b2), "=r"(b3)
                             : "r"(addr));
                mma_bf16(oacc[dn], pa, b0, b1);
                mma_bf16(oacc[dn + 1], pa, b2, b3);
            }
        }
        __syncthreads();
    }

    // epilogue: normalise, write the partial state
    l0 += __shfl_xor_sync(0xffffffffu, l0, 1);
    l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
    l1 += __shfl_xor_sync(0xffffffffu, l1, 1);
    l1 += __shfl_xor_sync(0xffffffffu, l1, 2);
    const float inv0 = l0 > 0.f ? 1.f / l0 : 0.f, inv1 = l1 > 0.f ? 1.f / l1 : 0.f;
    if (v0) {
        float* o = po + ((size_t)t0 * pl.Hq + h0) * D + tq * 2;
#pragma unroll
        for (int dn = 0; dn < 16; ++dn)
            *reinterpret_cast<float2*>(o + dn * 8) = make_float2(oacc[dn][0] * inv0, oacc[dn][1] * inv0);
        if (tq == 0) plse[(size_t)t0 * pl.Hq + h0] = l0 > 0.f ? m0 * pl.sm_scale + logf(l0) : -INFINITY;
    }
    if (v1) {
        float* o = po + ((size_t)t1 * pl.Hq + h1) * D + tq * 2;
#pragma unroll
        for (int dn = 0; dn < 16; ++dn)
            *reinterpret_cast<float2*>(o + dn * 8) = make_float2(oacc[dn][2] * inv1, oacc[dn][3] * inv1);
        if (tq == 0) plse[(size_t)t1 * pl.Hq + h1] = l1 > 0.f ? m1 * pl.sm_scale + logf(l1) : -INFINITY;
    }
}

// Merge: LSE = log sum_p e^{LSE_p};  O = sum_p e^{LSE_p - LSE} O_p over the prefix chunks and the
// tree state ("cascade attention" state merge).  One warp per (b,t,h) row.
__global__ void __launch_bounds__(128) attn_merge_kernel(AttnPlan pl, AttnArgs a) {
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    const int rows_per_req = pl.T_cap * pl.Hq;
    if (warp >= pl.B * rows_per_req) return;
    const int b = warp / rows_per_req;
    const int th = warp - b * rows_per_req;  // t*Hq + h
    const int t = th / pl.Hq;
    if (t >= a.tree_len[b]) return;
    const float* lsep = a.part_lse + (size_t)b * pl.NS * rows_per_req + th;
    const float* op = a.part_o + ((size_t)b * pl.NS * rows_per_req + th) * D + lane * 4;
    const size_t sstride = (size_t)rows_per_req;

    // prefix chunks first (kept separately for dbg_state), then the tree state
    float m = -INFINITY;
    for (int p = 0; p < pl.num_splits; ++p) m = fmaxf(m, lsep[p * sstride]);
    float wsum = 0.f;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    if (m > -INFINITY) {
        for (int p = 0; p < pl.num_splits; ++p) {
            const float l = lsep[p * sstride];
            if (l == -INFINITY) continue;
            const float w = __expf(l - m);
            const float4 o = *reinterpret_cast<const float4*>(op + p * sstride * D);
            wsum += w;
            acc.x += w * o.x; acc.y += w * o.y; acc.z += w * o.z; acc.w += w * o.w;
        }
    }
    const float lse_prefix = (m > -INFINITY) ? m + logf(wsum) : -INFINITY;
    const float lt = lsep[pl.num_splits * sstride];
    const float4 ot = *reinterpret_cast<const float4*>(op + pl.num_splits * sstride * D);
    if (a.dbg_state) {
        const size_t rs = (size_t)(D + 1);
        float* d0 = a.dbg_state + ((size_t)b * rows_per_req + th) * rs;
        float* d1 = d0 + (size_t)pl.B * rows_per_req * rs;
        const float inv = wsum > 0.f ? 1.f / wsum : 0.f;
        d0[lane * 4 + 0] = acc.x * inv; d0[lane * 4 + 1] = acc.y * inv;
        d0[lane * 4 + 2] = acc.z * inv; d0[lane * 4 + 3] = acc.w * inv;
        d1[lane * 4 + 0] = ot.x; d1[lane * 4 + 1] = ot.y; d1[lane * 4 + 2] = ot.z; d1[lane * 4 + 3] = ot.w;
        if (lane == 0) { d0[D] = lse_prefix; d1[D] = lt; }
    }
    // fold the tree state in (lt is finite: every row has its self bit)
    const float m2 = fmaxf(m, lt);
    const float sp = (m > -INFINITY) ? __expf(m - m2) : 0.f;
    const float wt = __expf(lt - m2);
    const float tot = wsum * sp + wt;
    const float inv = 1.f / tot;
    const float ox = (acc.x * sp + wt * ot.x) * inv, oy = (acc.y * sp + wt * ot.y) * inv;
    const float oz = (acc.z * sp + wt * ot.z) * inv, ow = (acc.w * sp + wt * ot.w) * inv;
    __nv_bfloat162 lo = __floats2bfloat162_rn(ox, oy), hi = __floats2bfloat162_rn(oz, ow);
    uint2 pk;
    pk.x = *reinterpret_cast<uint32_t*>(&lo);
    pk.y = *reinterpret_cast<uint32_t*>(&hi);
    *reinterpret_cast<uint2*>(a.out + ((size_t)b * rows_per_req + th) * D + lane * 4) = pk;
    if (a.lse && lane == 0) a.lse[(size_t)b * rows_per_req + th] = m2 + logf(tot);
}

}  // namespace

int32_t launch_attn_mma(const AttnPlan& pl, const AttnArgs& a, bool do_prefix, bool do_tree,
                        cudaStream_t s) {
    static unsigned long long attr_done = 0;
    if (first_use_on_device(attr_done))
        D2SD_CHECK_CUDA(cudaFuncSetAttribute(attn_mma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             SMEM_BYTES));
    const int first = do_prefix ? 0 : pl.num_splits;
    const int last = do_tree ? pl.num_splits : pl.num_splits - 1;
    if (last < first) return D2SD_OK;
    dim3 grid(ceil_div(pl.T_cap * pl.G, BM), last - first + 1, pl.B * pl.Hkv);
    attn_mma_kernel<<<grid, NT, SMEM_BYTES, s>>>(pl, a, first);
    D2SD_CHECK_LAUNCH("attn_mma_kernel");
    return D2SD_OK;
}

int32_t launch_attn_merge(const AttnPlan& pl, const AttnArgs& a, cudaStream_t s) {
    const int rows = pl.B * pl.T_cap * pl.Hq;
    attn_merge_kernel<<<ceil_div(rows, 4), 128, 0, s>>>(pl, a);
    D2SD_CHECK_LAUNCH("attn_merge_kernel");
    return D2SD_OK;
}

}  // namespace d2sd
