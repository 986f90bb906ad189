// Stage (c) prefix pass on tcgen05 / TMEM / TMA (sm_100a).  PAPER.md:52, :124, :154.
//
// One CTA = (request b, kv head g, context chunk `split`, group of <= 3 query tiles).  Every tree
// query of every branch and every GQA head of the group is a row of one batched query matrix
// (row r = t*G + hh), so the chunk's K/V tiles are pulled from HBM into this SM exactly once and are
// reused by all <= 384 rows:
//
//   S[128 x 64]  = Q_m[128 x 128] . K_j^T      tcgen05.mma, A/B from 128B-swizzled SMEM (TMA), D in TMEM
//   P            = exp2(c*(S - m_run))         softmax warps, one thread per row (TMEM lane), P -> TMEM
//   O_m[128x128] += P[128 x 64] . V_j[64x128]  tcgen05.mma, A = P from TMEM, B = V (MN-major SMEM)
//
// Warp roles (512 threads): warp 0 = TMA producer, warp 1 = MMA issuer (one thread), warp 2 = TMEM
// allocator, warps 4..15 = three softmax warpgroups, group m owning query tile m for the whole
// kernel (running max / sum stay in registers).  TMEM: O_0..O_2 at columns 0/128/256, two S/P
// buffers of 64 columns at 384/448.  The running max is only raised when the new tile maximum
// exceeds it by more than 2^8 (lazy rescale), in which case the owning softmax warp rescales its O
// rows in TMEM before the next P.V is issued.
#include <cuda.h>

#include "common.cuh"

namespace d2sd {
namespace {

constexpr int kD = 128;
constexpr int kTileM = 128;
constexpr int kTileN = 64;
constexpr int kMaxMT = 3;
constexpr int kStages = 4;
constexpr int kThreads = 512;
constexpr uint32_t kQTileBytes = kTileM * kD * 2;   // 32 KiB: [d_hi 2][128 rows][128 B]
constexpr uint32_t kKvTileBytes = kTileN * kD * 2;  // 16 KiB: [d_hi 2][64 keys][128 B]
constexpr uint32_t kStageBytes = 2 * kKvTileBytes;
constexpr uint32_t kOffQ = 0;
constexpr uint32_t kOffKv = kMaxMT * kQTileBytes;
constexpr uint32_t kOffBar = kOffKv + kStages * kStageBytes;
constexpr uint32_t kSmemBytes = kOffBar + 256 + 1024;  // + barriers + alignment slack
constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kTmemS = 384;  // S/P buffers behind the three O accumulators
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kRescaleThreshold = 8.0f;  // log2 units

// barrier slots (8 bytes each) at kOffBar
enum : uint32_t {
    kBarQFull = 0,
    kBarKvFull = 1,                      // [kStages]
    kBarKvEmpty = kBarKvFull + kStages,  // [kStages]
    // One S-ready / P-ready / O-ready barrier PER QUERY TILE m (phase = key tile j): a parity wait is only
    // sound if the waiter observes every phase, so barriers are never shared between softmax groups.
    kBarSFull = kBarKvEmpty + kStages,   // [kMaxMT]
    kBarPFull = kBarSFull + kMaxMT,      // [kMaxMT]
    kBarOReady = kBarPFull + kMaxMT,     // [kMaxMT]
    kNumBars = kBarOReady + kMaxMT,
    kTmemSlot = kNumBars  // uint32 written by tcgen05.alloc
};

// ---- PTX wrappers -------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
// Bounded wait: a protocol bug traps (reported as a launch failure) instead of hanging the GPU.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t spins = 0;
    while (!mbar_try_wait(bar, parity)) {
        if (++spins > (1u << 26)) __trap();
    }
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int c0, int c1, int c2,
                                            int c3, uint64_t hint) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
        " [%0], [%1, {%3, %4, %5, %6}], [%2], %7;" ::"r"(dst),
        "l"(reinterpret_cast<uint64_t>(tm)), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "l"(hint)
        : "memory");
}
__device__ __forceinline__ void tma_load_5d(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int c0, int c1, int c2,
                                            int c3, int c4, uint64_t hint) {
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
        " [%0], [%1, {%3, %4, %5, %6, %7}], [%2], %8;" ::"r"(dst),
        "l"(reinterpret_cast<uint64_t>(tm)), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "l"(hint)
        : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* tm) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(tm)) : "memory");
}
constexpr uint64_t kEvictFirst = 0x12F0000000000000ull;  // streamed once: KV
constexpr uint64_t kEvictLast = 0x14F0000000000000ull;   // re-read by every chunk CTA of the head: Q

// D[tmem] (+)= A[smem] . B[smem]
__device__ __forceinline__ void umma_ss(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc,
                                        uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// D[tmem] (+)= A[tmem] . B[smem]
__device__ __forceinline__ void umma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc,
                                        uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem),
        "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}

// Shared-memory matrix descriptor, 128B swizzle, descriptor version 1 (Blackwell).
//   K-major  operand: rows of 128 B (64 bf16 along K); 8-row groups SBO = 1024 B apart; LBO unused (1).
//   MN-major operand: rows of 128 B (64 bf16 along MN); the next 64 along MN is LBO bytes away, the next
//                     8 along K is SBO = 1024 B away.
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    return (uint64_t)((addr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) |
           ((uint64_t)(sbo_bytes >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// Instruction descriptor, kind::f16: fp32 accumulate, bf16 x bf16.
constexpr uint32_t idesc(uint32_t M, uint32_t N, uint32_t b_mn_major) {
    return (1u << 4) | (1u << 7) | (1u << 10) | (b_mn_major << 16) | ((N >> 3) << 17) | ((M >> 4) << 24);
}
constexpr uint32_t kIdescQK = idesc(kTileM, kTileN, 0);
constexpr uint32_t kIdescPV = idesc(kTileM, kD, 1);

__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"
        "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
          "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
          "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr));
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,"
        "%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};" ::"r"(taddr),
        "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]),
        "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]), "r"(r[18]),
        "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]),
        "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31])
        : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

__device__ __forceinline__ float ex2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ uint32_t pack2_bf16(float lo, float hi) {
    __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&v);
}

// -------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads, 1)
attn_prefix_tc_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
                      const __grid_constant__ CUtensorMap tm_v, AttnPlan pl, AttnArgs a, int n_mgroups) {
    extern __shared__ unsigned char smem_raw[];
    const uint32_t smem_raw_u32 = (uint32_t)__cvta_generic_to_shared(smem_raw);
    const uint32_t smem = (smem_raw_u32 + 1023u) & ~1023u;  // 128B swizzle atoms need 1024 B alignment
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int split = blockIdx.x, g = blockIdx.y;
    const int b = blockIdx.z / n_mgroups, mg = blockIdx.z - b * n_mgroups;
    const int G = pl.G;
    const int rows_valid = a.tree_len[b] * G;
    const int row_base = mg * (kMaxMT * kTileM);
    if (row_base >= rows_valid) return;
    const int MT = min(kMaxMT, (rows_valid - row_base + kTileM - 1) / kTileM);
    const int L = a.ctx_len[b];
    const int k_begin = split * pl.chunk_keys;
    const int k_end = min(L, k_begin + pl.chunk_keys);
    float* po = a.part_o + (((size_t)b * pl.NS + split) * pl.T_cap) * pl.Hq * kD;
    float* plse = a.part_lse + (((size_t)b * pl.NS + split) * pl.T_cap) * pl.Hq;
    if (k_begin >= k_end) {  // empty chunk: state (O = 0, LSE = -inf); O is never read by the merge
        for (int r = row_base + tid; r < min(rows_valid, row_base + kMaxMT * kTileM); r += kThreads) {
            const int t = r / G;
            plse[(size_t)t * pl.Hq + g * G + (r - t * G)] = -INFINITY;
        }
        return;
    }
    const int n_tiles = (k_end - k_begin + kTileN - 1) / kTileN;
    const int kv_row0 = (a.kv_indptr ? a.kv_indptr[b] : 0) + k_begin;

    const uint32_t bar0 = smem + kOffBar;
    auto bar = [&](uint32_t i) { return bar0 + 8u * i; };
    volatile uint32_t* tmem_slot =
        reinterpret_cast<volatile uint32_t*>(smem_raw + (smem - smem_raw_u32) + kOffBar + 8u * kTmemSlot);

    if (warp == 0 && lane == 0) {
        mbar_init(bar(kBarQFull), 1);
        for (int s = 0; s < kStages; ++s) {
            mbar_init(bar(kBarKvFull + s), 1);
            mbar_init(bar(kBarKvEmpty + s), 1);
        }
        for (int m = 0; m < kMaxMT; ++m) {
            mbar_init(bar(kBarSFull + m), 1);
            mbar_init(bar(kBarPFull + m), kTileM);
            mbar_init(bar(kBarOReady + m), 1);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        tma_prefetch_desc(&tm_q);
        tma_prefetch_desc(&tm_k);
        tma_prefetch_desc(&tm_v);
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(bar(kTmemSlot)),
                     "r"(kTmemCols)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp == 0) {
        // ===== TMA producer =====
        if (lane == 0) {
            mbar_expect_tx(bar(kBarQFull), MT * kQTileBytes);
            for (int m = 0; m < MT; ++m) {
                const int t0 = b * pl.T_cap + (row_base + m * kTileM) / G;
                tma_load_5d(smem + kOffQ + m * kQTileBytes, &tm_q, bar(kBarQFull), 0, 0, t0, 0, g, kEvictLast);
            }
            for (int j = 0; j < n_tiles; ++j) {
                const int s = j % kStages;
                mbar_wait(bar(kBarKvEmpty + s), ((j / kStages) & 1) ^ 1);
                mbar_expect_tx(bar(kBarKvFull + s), kStageBytes);
                const uint32_t dst = smem + kOffKv + s * kStageBytes;
                tma_load_4d(dst, &tm_k, bar(kBarKvFull + s), 0, kv_row0 + j * kTileN, 0, g, kEvictFirst);
                tma_load_4d(dst + kKvTileBytes, &tm_v, bar(kBarKvFull + s), 0, kv_row0 + j * kTileN, 0, g, kEvictFirst);
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (one thread) =====
        if (lane == 0) {
            const int U = n_tiles * MT;
            mbar_wait(bar(kBarQFull), 0);
            for (int u = 0; u <= U; ++u) {
                if (u < U) {  // S_u = Q_m K_j^T into S buffer u&1
                    const int j = u / MT, m = u - j * MT, s = j % kStages;
                    if (m == 0) mbar_wait(bar(kBarKvFull + s), (j / kStages) & 1);
                    tc_fence_after();
                    const uint32_t qa = smem + kOffQ + m * kQTileBytes;
                    const uint32_t ka = smem + kOffKv + s * kStageBytes;
#pragma unroll
                    for (int kk = 0; kk < kD / 16; ++kk) {
                        const uint64_t ad = smem_desc(qa + (kk >> 2) * (kQTileBytes / 2) + (kk & 3) * 32, 16, 1024);
                        const uint64_t bd = smem_desc(ka + (kk >> 2) * (kKvTileBytes / 2) + (kk & 3) * 32, 16, 1024);
                        umma_ss(tmem + kTmemS + (u & 1) * kTileN, ad, bd, kIdescQK, kk > 0);
                    }
                    tc_commit(bar(kBarSFull + m));
                }
                if (u >= 1) {  // O_m += P_v V_j, P read from TMEM (aliases S buffer v&1)
                    const int v = u - 1;
                    const int j = v / MT, m = v - j * MT, s = j % kStages;
                    mbar_wait(bar(kBarPFull + m), j & 1);
                    tc_fence_after();
                    const uint32_t va = smem + kOffKv + s * kStageBytes + kKvTileBytes;
#pragma unroll
                    for (int kk = 0; kk < kTileN / 16; ++kk) {
                        const uint64_t bd = smem_desc(va + kk * 2048, kKvTileBytes / 2, 1024);
                        umma_ts(tmem + m * kD, tmem + kTmemS + (v & 1) * kTileN + kk * 8, bd, kIdescPV,
                                (j > 0 || kk > 0));
                    }
                    tc_commit(bar(kBarOReady + m));
                    if (m == MT - 1) tc_commit(bar(kBarKvEmpty + s));
                }
            }
        }
    } else if (warp >= 4) {
        // ===== softmax warpgroup m: one thread per query row =====
        const int m = (warp - 4) >> 2;
        if (m < MT) {
            const int w = warp & 3;
            const int r = row_base + m * kTileM + w * 32 + lane;  // this thread's row
            const bool warp_active = (row_base + m * kTileM + w * 32) < rows_valid;
            const uint32_t lane_addr = (uint32_t)(w * 32) << 16;
            const float c2 = pl.sm_scale * kLog2e;
            const float thr = kRescaleThreshold / c2;  // in raw score units
            float m_run = -INFINITY, l_run = 0.f;
            for (int j = 0; j < n_tiles; ++j) {
                const int u = j * MT + m;
                const uint32_t sbuf = tmem + kTmemS + (u & 1) * kTileN + lane_addr;
                mbar_wait(bar(kBarSFull + m), j & 1);
                bool saw_o = false;  // every phase of O-ready must be observed (parity waits)
                if (warp_active) {
                    tc_fence_after();
                    uint32_t s0[32], s1[32];
                    tmem_ld32(sbuf, s0);
                    tmem_ld32(sbuf + 32, s1);
                    tmem_wait_ld();
                    const int valid = k_end - (k_begin + j * kTileN);  // keys of this tile inside the chunk
                    if (valid < kTileN) {
#pragma unroll
                        for (int c = 0; c < 32; ++c) {
                            if (c >= valid) s0[c] = 0xFF800000u;       // -inf
                            if (c + 32 >= valid) s1[c] = 0xFF800000u;
                        }
                    }
                    float mx = -INFINITY;
#pragma unroll
                    for (int c = 0; c < 32; ++c) mx = fmaxf(mx, fmaxf(__uint_as_float(s0[c]), __uint_as_float(s1[c])));
                    // lazy rescale: raise the running max only when it is exceeded by more than 2^8
                    const bool need = mx > m_run + thr;
                    if (j == 0) {
                        m_run = mx;
                    } else if (__any_sync(0xffffffffu, need)) {
                        const float alpha = need ? ex2((m_run - mx) * c2) : 1.f;
                        mbar_wait(bar(kBarOReady + m), (j - 1) & 1);  // previous P.V into O_m has landed
                        saw_o = true;
                        tc_fence_after();
#pragma unroll 1
                        for (int c0 = 0; c0 < kD; c0 += 32) {
                            uint32_t o[32];
                            tmem_ld32(tmem + m * kD + c0 + lane_addr, o);
                            tmem_wait_ld();
#pragma unroll
                            for (int c = 0; c < 32; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * alpha);
                            tmem_st32(tmem + m * kD + c0 + lane_addr, o);
                        }
                        tmem_wait_st();
                        if (need) {
                            m_run = mx;
                            l_run *= alpha;
                        }
                    }
                    const float ms = m_run * c2;
                    float sum = 0.f;
                    uint32_t p[32];
#pragma unroll
                    for (int c = 0; c < 16; ++c) {
                        const float e0 = ex2(__uint_as_float(s0[2 * c]) * c2 - ms);
                        const float e1 = ex2(__uint_as_float(s0[2 * c + 1]) * c2 - ms);
                        const float e2 = ex2(__uint_as_float(s1[2 * c]) * c2 - ms);
                        const float e3 = ex2(__uint_as_float(s1[2 * c + 1]) * c2 - ms);
                        sum += (e0 + e1) + (e2 + e3);
                        p[c] = pack2_bf16(e0, e1);
                        p[16 + c] = pack2_bf16(e2, e3);
                    }
                    l_run += sum;
                    tmem_st32(sbuf, p);  // P[128 x 64] bf16 = 32 columns, K contiguous, 2 per column
                    tmem_wait_st();
                    tc_fence_before();
                }
                mbar_arrive(bar(kBarPFull + m));
                if (j > 0 && !saw_o) mbar_wait(bar(kBarOReady + m), (j - 1) & 1);
            }
            // epilogue: O_m / l -> partial state of this chunk
            mbar_wait(bar(kBarOReady + m), (n_tiles - 1) & 1);
            if (warp_active) {
                tc_fence_after();
                const bool row_ok = r < rows_valid;
                const int t = r / G;
                const int h = g * G + (r - t * G);
                const float inv = 1.f / l_run;
                float* orow = po + ((size_t)t * pl.Hq + h) * kD;
#pragma unroll 1
                for (int c0 = 0; c0 < kD; c0 += 32) {
                    uint32_t o[32];
                    tmem_ld32(tmem + m * kD + c0 + lane_addr, o);
                    tmem_wait_ld();
                    if (row_ok) {
#pragma unroll
                        for (int c = 0; c < 32; c += 4)
                            *reinterpret_cast<float4*>(orow + c0 + c) =
                                make_float4(__uint_as_float(o[c]) * inv, __uint_as_float(o[c + 1]) * inv,
                                            __uint_as_float(o[c + 2]) * inv, __uint_as_float(o[c + 3]) * inv);
                    }
                }
                if (row_ok) plse[(size_t)t * pl.Hq + h] = m_run * pl.sm_scale + logf(l_run);
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 2) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(kTmemCols) : "memory");
    }
}

// ---- host side ----------------------------------------------------------------------------------
using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

int32_t encode(CUtensorMap* tm, const void* base, int rank, const cuuint64_t* dims, const cuuint64_t* strides,
               const cuuint32_t* box, const char* what) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return set_error(D2SD_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
    cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, (cuuint32_t)rank, const_cast<void*>(base), dims, strides, box,
                    estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return set_error(D2SD_ERR_CUDA, "cuTensorMapEncodeTiled(%s) failed with CUresult %d", what, (int)r);
    return D2SD_OK;
}

}  // namespace

bool attn_prefix_tc_supported(const AttnPlan& pl) {
    // contiguous KV only (paged KV stays on the mma.sync path), rows of one query tile must be whole
    // tree nodes (128 % G == 0), and the tensor-map extents must fit.
    return pl.page_size == 0 && pl.d == kD && pl.G <= 128 && (128 % pl.G) == 0 && pl.kv_rows > 0 &&
           pl.max_ctx_len > 0 && (int64_t)pl.B * pl.T_cap < (1ll << 31) && pl.kv_rows < (1ll << 31);
}

int32_t launch_attn_prefix_tc(const AttnPlan& pl, const AttnArgs& a, cudaStream_t s) {
    static bool attr_set = false;
    if (!attr_set) {
        D2SD_CHECK_CUDA(cudaFuncSetAttribute(attn_prefix_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)kSmemBytes));
        attr_set = true;
    }
    CUtensorMap tm_q, tm_k, tm_v;
    {   // Q [B*T_cap, Hq, d] viewed as (d_lo 64, hh G, t B*T_cap, d_hi 2, g Hkv): one box = one 128-row query tile
        const cuuint64_t dims[5] = {64, (cuuint64_t)pl.G, (cuuint64_t)pl.B * pl.T_cap, 2, (cuuint64_t)pl.Hkv};
        const cuuint64_t strides[4] = {(cuuint64_t)kD * 2, (cuuint64_t)pl.Hq * kD * 2, 128, (cuuint64_t)pl.G * kD * 2};
        const cuuint32_t box[5] = {64, (cuuint32_t)pl.G, (cuuint32_t)(kTileM / pl.G), 2, 1};
        if (int32_t st = encode(&tm_q, a.q, 5, dims, strides, box, "q")) return st;
    }
    {   // K/V [kv_rows, Hkv, d] viewed as (d_lo 64, row, d_hi 2, g): one box = one 64-key tile
        const cuuint64_t dims[4] = {64, (cuuint64_t)pl.kv_rows, 2, (cuuint64_t)pl.Hkv};
        const cuuint64_t strides[3] = {(cuuint64_t)pl.Hkv * kD * 2, 128, (cuuint64_t)kD * 2};
        const cuuint32_t box[4] = {64, kTileN, 2, 1};
        if (int32_t st = encode(&tm_k, a.k_cache, 4, dims, strides, box, "k_cache")) return st;
        if (int32_t st = encode(&tm_v, a.v_cache, 4, dims, strides, box, "v_cache")) return st;
    }
    const int n_mgroups = ceil_div(pl.T_cap * pl.G, kMaxMT * kTileM);
    dim3 grid(pl.num_splits, pl.Hkv, pl.B * n_mgroups);
    attn_prefix_tc_kernel<<<grid, kThreads, kSmemBytes, s>>>(tm_q, tm_k, tm_v, pl, a, n_mgroups);
    D2SD_CHECK_LAUNCH("attn_prefix_tc_kernel");
    return D2SD_OK;
}

}  // namespace d2sd
