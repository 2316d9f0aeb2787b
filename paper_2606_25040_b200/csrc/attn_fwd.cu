// attn_fwd.cu — chorus_block_sparse_attn_fwd kernel for sm_100a ("skip pruned block
// pairs and evaluate only the retained ones in QK^T, softmax, and PV").
//
// v0 (correctness first): one CTA of 128 threads per (batch, head, 128-row query block).  For each
// kept 64-key tile of the CSR row, TMA stages the K and V tiles in shared memory (128-byte
// swizzle), one thread issues tcgen05.mma for S = Q K^T into tensor memory, the four warps read
// their 32 TMEM lanes (one query row per thread), run the online softmax in fp32 with warp-free
// per-row state, write P (bf16) back to tensor memory, and one thread issues O += P V with P as
// the TMEM A operand and V as an MN-major shared-memory B operand.  O stays in TMEM across the row.
#include <cuda_bf16.h>

#include "chorus_internal.h"
#include "sm100_ptx.cuh"

namespace chorus {
namespace {

using namespace ptx;

constexpr int BQ = 128, BK = 64, HD = 128;

// shared memory map (bytes, from a 1024-aligned base)
constexpr uint32_t SQ_OFF = 0;                      // Q: 2 slabs [128 rows][64 ch] bf16 = 32 KB
constexpr uint32_t SK_OFF = 32768;                  // K: 2 slabs [64 keys][64 ch]      = 16 KB
constexpr uint32_t SV_OFF = 49152;                  // V: 2 slabs [64 keys][64 ch]      = 16 KB
constexpr uint32_t BAR_OFF = 65536;                 // 4 mbarriers + tmem slot
constexpr uint32_t SMEM_BYTES_V0 = 65536 + 64 + 1024;  // + alignment slack

// tensor-memory map (columns)
constexpr uint32_t TM_S = 0;     // S: 64 fp32 columns
constexpr uint32_t TM_P = 64;    // P: 64 bf16 = 32 columns
constexpr uint32_t TM_O = 128;   // O: 128 fp32 columns
constexpr uint32_t TM_COLS = 256;

constexpr uint32_t IDESC_S_BF16 = make_idesc(1, 1, 128, 64, 0, 0);    // Q K^T : both K-major
constexpr uint32_t IDESC_PV_BF16 = make_idesc(1, 1, 128, 128, 0, 1);  // P V   : V is MN-major

__global__ void __launch_bounds__(128, 1)
attn_fwd_v0_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                   const __grid_constant__ CUtensorMap tmV, const AttnParams p) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* gen_base = smem_raw + (base - smem_u32(smem_raw));
    const uint32_t sQ = base + SQ_OFF, sK = base + SK_OFF, sV = base + SV_OFF;
    const uint32_t bar_q = base + BAR_OFF, bar_kv = bar_q + 8, bar_s = bar_q + 16,
                   bar_o = bar_q + 24;
    volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(gen_base + BAR_OFF + 32);

    const int qb = blockIdx.x, h = blockIdx.y, b = blockIdx.z;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        mbar_init(bar_q, 1);
        mbar_init(bar_kv, 1);
        mbar_init(bar_s, 1);
        mbar_init(bar_o, 1);
        fence_mbar_init();
    }
    if (warp == 0) tmem_alloc(base + BAR_OFF + 32, TM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const uint32_t tlane = tmem + (static_cast<uint32_t>(warp * 32) << 16);

    const int r0 = p.row_ptr[h * p.nq + qb], r1 = p.row_ptr[h * p.nq + qb + 1];
    const int ntiles = r1 - r0;
    const int q_row = qb * BQ + warp * 32 + lane;

    if (threadIdx.x == 0 && ntiles > 0) {
        mbar_arrive_expect_tx(bar_q, 32768);
        tma_load_4d(sQ, &tmQ, bar_q, 0, qb * BQ, h, b);
        tma_load_4d(sQ + 16384, &tmQ, bar_q, 64, qb * BQ, h, b);
    }

    float m = -INFINITY, l = 0.f;
    for (int t = 0; t < ntiles; ++t) {
        const int kb = p.col_idx[r0 + t];
        const uint32_t ph = t & 1;
        if (threadIdx.x == 0) {
            mbar_arrive_expect_tx(bar_kv, 32768);
            tma_load_4d(sK, &tmK, bar_kv, 0, kb * BK, h, b);
            tma_load_4d(sK + 8192, &tmK, bar_kv, 64, kb * BK, h, b);
            tma_load_4d(sV, &tmV, bar_kv, 0, kb * BK, h, b);
            tma_load_4d(sV + 8192, &tmV, bar_kv, 64, kb * BK, h, b);
            if (t == 0) mbar_wait(bar_q, 0);
            mbar_wait(bar_kv, ph);
            tc_fence_after();
#pragma unroll
            for (int ks = 0; ks < 8; ++ks) {  // 8 x K=16 over head_dim
                const uint32_t slab = ks >> 2, koff = (ks & 3) * 32;
                const uint64_t da = smem_desc_sw128(sQ + slab * 16384 + koff, 16, 1024);
                const uint64_t db = smem_desc_sw128(sK + slab * 8192 + koff, 16, 1024);
                mma_f16_ss(tmem + TM_S, da, db, IDESC_S_BF16, ks > 0);
            }
            tc_commit(bar_s);
        }
        mbar_wait(bar_s, ph);
        tc_fence_after();

        uint32_t s0[32], s1[32];
        tmem_ld32(tlane + TM_S, s0);
        tmem_ld32(tlane + TM_S + 32, s1);
        tc_wait_ld();
        const int valid = min(BK, p.N - kb * BK);
        float x[64];
        float mx = -INFINITY;
#pragma unroll
        for (int j = 0; j < 32; ++j) {
            x[j] = (j < valid) ? __uint_as_float(s0[j]) * p.scale_log2 : -INFINITY;
            x[32 + j] = (32 + j < valid) ? __uint_as_float(s1[j]) * p.scale_log2 : -INFINITY;
        }
#pragma unroll
        for (int j = 0; j < 64; ++j) mx = fmaxf(mx, x[j]);
        const float m_new = fmaxf(m, mx);
        const float alpha = ex2(m - m_new);  // m = -inf on the first tile -> 0
        float sum = 0.f;
        uint32_t pk[32];
#pragma unroll
        for (int j = 0; j < 32; ++j) {
            const float p0 = ex2(x[2 * j] - m_new), p1 = ex2(x[2 * j + 1] - m_new);
            sum += p0 + p1;
            pk[j] = pack_bf16x2(p0, p1);
        }
        l = l * alpha + sum;
        m = m_new;
        tmem_st32(tlane + TM_P, pk);
        if (t > 0) {  // rescale the running O (previous P V has completed: bar_o was waited)
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                uint32_t o[32];
                tmem_ld32(tlane + TM_O + c * 32, o);
                tc_wait_ld();
#pragma unroll
                for (int j = 0; j < 32; ++j) o[j] = __float_as_uint(__uint_as_float(o[j]) * alpha);
                tmem_st32(tlane + TM_O + c * 32, o);
            }
        }
        tc_wait_st();
        tc_fence_before();
        __syncthreads();
        if (threadIdx.x == 0) {
            tc_fence_after();
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) {  // 4 x K=16 over the 64 keys
                const uint64_t db = smem_desc_sw128(sV + ks * 2048, 8192, 1024);
                mma_f16_ts(tmem + TM_O, tmem + TM_P + ks * 8, db, IDESC_PV_BF16, (t > 0) || (ks > 0));
            }
            tc_commit(bar_o);
        }
        mbar_wait(bar_o, ph);
        tc_fence_after();
    }

    // epilogue: O / l -> bf16 -> global (one 256-byte row per thread, 16-byte stores).  The TMEM
    // loads are warp-collective, so every thread issues them; only the stores are predicated.
    {
        __nv_bfloat16* orow = static_cast<__nv_bfloat16*>(p.O) + b * p.o_sb +
                              static_cast<int64_t>(q_row) * p.o_sn + h * p.o_sh;
        const float inv = (ntiles > 0) ? 1.f / l : 0.f;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            uint32_t o[32];
            if (ntiles > 0) {  // CTA-uniform
                tmem_ld32(tlane + TM_O + c * 32, o);
                tc_wait_ld();
            } else {
#pragma unroll
                for (int j = 0; j < 32; ++j) o[j] = 0u;
            }
            if (q_row < p.N) {
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    uint4 v;
                    v.x = pack_bf16x2(__uint_as_float(o[8 * j + 0]) * inv, __uint_as_float(o[8 * j + 1]) * inv);
                    v.y = pack_bf16x2(__uint_as_float(o[8 * j + 2]) * inv, __uint_as_float(o[8 * j + 3]) * inv);
                    v.z = pack_bf16x2(__uint_as_float(o[8 * j + 4]) * inv, __uint_as_float(o[8 * j + 5]) * inv);
                    v.w = pack_bf16x2(__uint_as_float(o[8 * j + 6]) * inv, __uint_as_float(o[8 * j + 7]) * inv);
                    reinterpret_cast<uint4*>(orow + c * 32)[j] = v;
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, TM_COLS);
}

}  // namespace

cudaError_t launch_attn_fwd(const CUtensorMap& tmQ, const CUtensorMap& tmK, const CUtensorMap& tmV,
                            const CUtensorMap& tmO, const AttnParams& p, chorus_dtype dtype,
                            cudaStream_t stream) {
    (void)tmO;
    if (dtype != CHORUS_BF16) return cudaErrorNotSupported;
    cudaError_t e = cudaFuncSetAttribute(attn_fwd_v0_kernel,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES_V0);
    if (e != cudaSuccess) return e;
    dim3 grid(p.nq, p.H, p.B);
    attn_fwd_v0_kernel<<<grid, 128, SMEM_BYTES_V0, stream>>>(tmQ, tmK, tmV, p);
    count_launch(1);
    return cudaGetLastError();
}

}  // namespace chorus
