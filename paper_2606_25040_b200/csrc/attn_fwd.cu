// attn_fwd.cu — chorus_block_sparse_attn_fwd for sm_100a ("skip pruned block pairs and
// evaluate only the retained ones in QK^T, softmax, and PV").
//
// Persistent, warp-specialised kernel, one CTA (384 threads) per SM:
//   warp 8        TMA producer: Q tile once per work item, then the kept K / V tiles of the CSR row,
//                 two 64-key tiles ("a pair") per pipeline stage, 128-byte swizzle
//   warp 9        MMA issuer (one thread): S = Q K^T (M=128, N=128, K=128) into tensor memory,
//                 O += P V (M=128, N=128, K=128) with P as the TMEM A operand and V as an MN-major
//                 shared-memory B operand
//   warps 0-3     softmax warpgroup of stream 0 (pairs 0, 2, 4, ...)
//   warps 4-7     softmax warpgroup of stream 1 (pairs 1, 3, 5, ...)
// A work item is one (batch, head, 128-row query block).  Its kept tiles are paired (any two kept
// tiles, not necessarily adjacent keys) so that QK^T runs at N=128; even and odd pairs form two
// independent online-softmax streams with their own S and O accumulators in tensor memory
// (S0 S1 O0 O1 = 4 x 128 columns), so the tensor pipe works on one stream while the other stream's
// warpgroup does its exponentials.  Each thread owns one query row (TMEM lane): row max and row sum
// need no shuffles.  O is rescaled lazily (only when the row max grows by more than 2^8).  The two
// streams are merged in the epilogue, normalised, converted to bf16, staged in shared memory and
// written with TMA stores (coalesced 128-byte rows; rows beyond N are clipped by the tensor map).
#include <cuda_bf16.h>

#include "chorus_internal.h"
#include "sm100_ptx.cuh"

namespace chorus {
namespace {

using namespace ptx;

constexpr int BQ = 128, BK = 64;
constexpr int KSTAGES = 2, VSTAGES = 3;
constexpr int NUM_THREADS = 384;
constexpr int PRODUCER_WARP = 8, MMA_WARP = 9;

// shared memory map (bytes from a 1024-aligned base)
constexpr uint32_t SQ_OFF = 0;                         // Q : 2 slabs [128 rows][128 B]      32 KB
constexpr uint32_t SK_OFF = 32768;                     // K : KSTAGES x 2 slabs [128 keys][128 B]
constexpr uint32_t SV_OFF = SK_OFF + KSTAGES * 32768;  // V : VSTAGES x 2 slabs [128 keys][128 B]
constexpr uint32_t SO_OFF = SV_OFF + VSTAGES * 32768;  // O staging: 2 slabs [128 rows][128 B]
constexpr uint32_t SML_OFF = SO_OFF + 32768;           // (m, l) exchange: 2 x 128 x float2  2 KB
constexpr uint32_t BAR_OFF = SML_OFF + 2048;
constexpr uint32_t SMEM_BYTES = BAR_OFF + 256;
static_assert(SMEM_BYTES <= 232448, "exceeds the 227 KB per-CTA shared memory of sm_100");

// mbarrier slots (8 bytes each) from BAR_OFF
enum : uint32_t {
    B_Q_FULL = 0, B_Q_EMPTY = 1, B_K_FULL = 2, B_K_EMPTY = B_K_FULL + KSTAGES,
    B_V_FULL = B_K_EMPTY + KSTAGES, B_V_EMPTY = B_V_FULL + VSTAGES, B_S_FULL = B_V_EMPTY + VSTAGES,
    B_P_READY = B_S_FULL + 2, B_O_FULL = B_P_READY + 2, B_O_FREE = B_O_FULL + 1,
    B_COUNT = B_O_FREE + 1
};
static_assert(B_COUNT * 8 + 8 <= 256, "barrier area too small");

// tensor-memory map (columns)
constexpr uint32_t TM_S0 = 0, TM_S1 = 128, TM_O0 = 256, TM_O1 = 384, TM_COLS = 512;

constexpr float RESCALE_THRESHOLD = 8.0f;  // log2 units: p stays below 2^8

__device__ __forceinline__ void setmaxnreg_inc_224() { asm volatile("setmaxnreg.inc.sync.aligned.u32 224;"); }
__device__ __forceinline__ void setmaxnreg_dec_56() { asm volatile("setmaxnreg.dec.sync.aligned.u32 56;"); }

struct Item {
    int b, h, qb, r0, nt, np;
};
__device__ __forceinline__ Item get_item(const AttnParams& p, int idx) {
    Item it;
    it.qb = idx % p.nq;
    const int bh = idx / p.nq;
    it.h = bh % p.H;
    it.b = bh / p.H;
    const int row = it.h * p.nq + it.qb;
    it.r0 = __ldg(p.row_ptr + row);
    it.nt = __ldg(p.row_ptr + row + 1) - it.r0;
    it.np = (it.nt + 1) >> 1;
    return it;
}

template <bool kFp8>
__global__ void __launch_bounds__(NUM_THREADS, 1)
attn_fwd_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmO,
                const AttnParams p) {
    // 128-byte swizzle needs a 1024-byte aligned base; the kernel has no static shared memory, so
    // the dynamic window starts at the CTA's (1 KB granular) allocation.  Checked, not assumed.
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t base = smem_u32(smem_raw);
    if (base & 1023u) __trap();
    uint8_t* gbase = smem_raw;
    const uint32_t sQ = base + SQ_OFF, sK = base + SK_OFF, sV = base + SV_OFF, sO = base + SO_OFF;
    const uint32_t bars = base + BAR_OFF;
    auto bar = [&](uint32_t i) { return bars + 8u * i; };
    volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(gbase + BAR_OFF + 8 * B_COUNT);
    float2* sml = reinterpret_cast<float2*>(gbase + SML_OFF);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_items = p.B * p.H * p.nq;

    if (threadIdx.x == 0) {
        mbar_init(bar(B_Q_FULL), 1);
        mbar_init(bar(B_Q_EMPTY), 1);
        for (int i = 0; i < KSTAGES; ++i) { mbar_init(bar(B_K_FULL + i), 1); mbar_init(bar(B_K_EMPTY + i), 1); }
        for (int i = 0; i < VSTAGES; ++i) { mbar_init(bar(B_V_FULL + i), 1); mbar_init(bar(B_V_EMPTY + i), 1); }
        for (int i = 0; i < 2; ++i) { mbar_init(bar(B_S_FULL + i), 1); mbar_init(bar(B_P_READY + i), 4); }
        mbar_init(bar(B_O_FULL), 1);
        mbar_init(bar(B_O_FREE), 8);
        fence_mbar_init();
    }
    if (warp == MMA_WARP) tmem_alloc(bars + 8 * B_COUNT, TM_COLS);
    if (warp == PRODUCER_WARP && lane == 0) {
        prefetch_tmap(&tmQ); prefetch_tmap(&tmK); prefetch_tmap(&tmV); prefetch_tmap(&tmO);
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp >= 8) {
        // ======================= producer / MMA warpgroup ==========================================
        setmaxnreg_dec_56();
        if (warp == PRODUCER_WARP && lane == 0) {
            uint32_t kcnt = 0, vcnt = 0, icnt = 0;
            for (int idx = blockIdx.x; idx < n_items; idx += gridDim.x) {
                const Item it = get_item(p, idx);
                if (it.nt == 0) continue;   // empty rows touch no barrier: icnt counts non-empty items
                mbar_wait(bar(B_Q_EMPTY), (icnt & 1) ^ 1);
                mbar_arrive_expect_tx(bar(B_Q_FULL), 32768);
                tma_load_4d(sQ, &tmQ, bar(B_Q_FULL), 0, it.qb * BQ, it.h, it.b);
                tma_load_4d(sQ + 16384, &tmQ, bar(B_Q_FULL), 64, it.qb * BQ, it.h, it.b);
                for (int j = 0; j < it.np; ++j) {
                    const int ntile = (2 * j + 1 < it.nt) ? 2 : 1;
                    const int kb0 = __ldg(p.col_idx + it.r0 + 2 * j);
                    const int kb1 = (ntile == 2) ? __ldg(p.col_idx + it.r0 + 2 * j + 1) : 0;
                    {
                        const uint32_t st = kcnt % KSTAGES, ph = (kcnt / KSTAGES) & 1;
                        mbar_wait(bar(B_K_EMPTY + st), ph ^ 1);
                        mbar_arrive_expect_tx(bar(B_K_FULL + st), ntile * 16384);
                        const uint32_t dst = sK + st * 32768;
                        tma_load_4d(dst, &tmK, bar(B_K_FULL + st), 0, kb0 * BK, it.h, it.b);
                        tma_load_4d(dst + 16384, &tmK, bar(B_K_FULL + st), 64, kb0 * BK, it.h, it.b);
                        if (ntile == 2) {
                            tma_load_4d(dst + 8192, &tmK, bar(B_K_FULL + st), 0, kb1 * BK, it.h, it.b);
                            tma_load_4d(dst + 16384 + 8192, &tmK, bar(B_K_FULL + st), 64, kb1 * BK, it.h, it.b);
                        }
                        ++kcnt;
                    }
                    {
                        const uint32_t st = vcnt % VSTAGES, ph = (vcnt / VSTAGES) & 1;
                        mbar_wait(bar(B_V_EMPTY + st), ph ^ 1);
                        mbar_arrive_expect_tx(bar(B_V_FULL + st), ntile * 16384);
                        const uint32_t dst = sV + st * 32768;
                        tma_load_4d(dst, &tmV, bar(B_V_FULL + st), 0, kb0 * BK, it.h, it.b);
                        tma_load_4d(dst + 16384, &tmV, bar(B_V_FULL + st), 64, kb0 * BK, it.h, it.b);
                        if (ntile == 2) {
                            tma_load_4d(dst + 8192, &tmV, bar(B_V_FULL + st), 0, kb1 * BK, it.h, it.b);
                            tma_load_4d(dst + 16384 + 8192, &tmV, bar(B_V_FULL + st), 64, kb1 * BK, it.h, it.b);
                        }
                        ++vcnt;
                    }
                }
                ++icnt;
            }
        } else if (warp == MMA_WARP && lane == 0) {
            constexpr uint32_t IDESC_S128 = make_idesc(1, 1, 128, 128, 0, 0);
            constexpr uint32_t IDESC_S64 = make_idesc(1, 1, 128, 64, 0, 0);
            constexpr uint32_t IDESC_PV = make_idesc(1, 1, 128, 128, 0, 1);
            uint32_t kcnt = 0, vcnt = 0, icnt = 0, pcnt[2] = {0, 0};
            for (int idx = blockIdx.x; idx < n_items; idx += gridDim.x) {
                const Item it = get_item(p, idx);
                if (it.nt == 0) continue;
                auto issue_pv = [&](int jj) {
                    const int s = jj & 1;
                    const int ntile = (2 * jj + 1 < it.nt) ? 2 : 1;
                    mbar_wait(bar(B_P_READY + s), pcnt[s] & 1);
                    ++pcnt[s];
                    const uint32_t st = vcnt % VSTAGES, ph = (vcnt / VSTAGES) & 1;
                    mbar_wait(bar(B_V_FULL + st), ph);
                    tc_fence_after();
                    const uint32_t tP = tmem + (s ? TM_S1 : TM_S0), tO = tmem + (s ? TM_O1 : TM_O0);
                    const int nks = 4 * ntile;
                    for (int ks = 0; ks < nks; ++ks) {
                        const uint64_t db = smem_desc_sw128(sV + st * 32768 + ks * 2048, 16384, 1024);
                        mma_f16_ts(tO, tP + ks * 8, db, IDESC_PV, (jj >= 2) || (ks > 0));
                    }
                    tc_commit(bar(B_V_EMPTY + st));
                    ++vcnt;
                };
                mbar_wait(bar(B_Q_FULL), icnt & 1);
                mbar_wait(bar(B_O_FREE), (icnt & 1) ^ 1);
                for (int j = 0; j < it.np; ++j) {
                    const int s = j & 1;
                    const int ntile = (2 * j + 1 < it.nt) ? 2 : 1;
                    const uint32_t st = kcnt % KSTAGES, ph = (kcnt / KSTAGES) & 1;
                    mbar_wait(bar(B_K_FULL + st), ph);
                    tc_fence_after();
                    const uint32_t tS = tmem + (s ? TM_S1 : TM_S0);
                    const uint32_t idesc = (ntile == 2) ? IDESC_S128 : IDESC_S64;
#pragma unroll
                    for (int ks = 0; ks < 8; ++ks) {
                        const uint32_t off = (ks >> 2) * 16384 + (ks & 3) * 32;
                        const uint64_t da = smem_desc_sw128(sQ + off, 16, 1024);
                        const uint64_t db = smem_desc_sw128(sK + st * 32768 + off, 16, 1024);
                        mma_f16_ss(tS, da, db, idesc, ks > 0);
                    }
                    tc_commit(bar(B_K_EMPTY + st));
                    tc_commit(bar(B_S_FULL + s));
                    ++kcnt;
                    if (j == it.np - 1) tc_commit(bar(B_Q_EMPTY));
                    if (j >= 1) issue_pv(j - 1);
                }
                issue_pv(it.np - 1);
                tc_commit(bar(B_O_FULL));
                ++icnt;
            }
        }
    } else {
        // ======================= softmax warpgroups =================================================
        setmaxnreg_inc_224();
        const int s = warp >> 2;                 // stream
        const int wq = warp & 3;                 // TMEM lane quarter
        const int row = wq * 32 + lane;          // query row inside the block == TMEM lane
        const uint32_t tlane = tmem + (static_cast<uint32_t>(wq * 32) << 16);
        const uint32_t tS = tlane + (s ? TM_S1 : TM_S0);
        const uint32_t tO = tlane + (s ? TM_O1 : TM_O0);
        const float sl2 = p.scale_log2;
        uint32_t scnt = 0, icnt = 0;
        for (int idx = blockIdx.x; idx < n_items; idx += gridDim.x) {
            const Item it = get_item(p, idx);
            float m = -INFINITY, l = 0.f;
            if (it.nt > 0) {
                for (int j = s; j < it.np; j += 2) {
                    mbar_wait(bar(B_S_FULL + s), scnt & 1);
                    ++scnt;
                    tc_fence_after();
                    uint32_t sv[128];
                    tmem_ld32(tS, *reinterpret_cast<uint32_t(*)[32]>(sv));
                    tmem_ld32(tS + 32, *reinterpret_cast<uint32_t(*)[32]>(sv + 32));
                    tmem_ld32(tS + 64, *reinterpret_cast<uint32_t(*)[32]>(sv + 64));
                    tmem_ld32(tS + 96, *reinterpret_cast<uint32_t(*)[32]>(sv + 96));
                    tc_wait_ld();
                    if (j == it.np - 1) {  // only the last pair can be odd or hold the ragged key block
                        const int kb0 = __ldg(p.col_idx + it.r0 + 2 * j);
                        const int v0 = min(BK, p.N - kb0 * BK);
                        int v1 = 0;
                        if (2 * j + 1 < it.nt) {
                            const int kb1 = __ldg(p.col_idx + it.r0 + 2 * j + 1);
                            v1 = min(BK, p.N - kb1 * BK);
                        }
                        if (v0 < BK || v1 < BK) {
#pragma unroll
                            for (int k = 0; k < 64; ++k) {
                                if (k >= v0) sv[k] = 0xff800000u;       // -inf
                                if (k >= v1) sv[64 + k] = 0xff800000u;
                            }
                        }
                    }
                    float mx = -INFINITY;
#pragma unroll
                    for (int k = 0; k < 128; ++k) mx = fmaxf(mx, __uint_as_float(sv[k]));
                    const float m_new = fmaxf(m, mx * sl2);
                    if (__any_sync(0xffffffffu, m_new > m + RESCALE_THRESHOLD)) {
                        const float alpha = ex2(m - m_new);   // m = -inf (first pair) -> 0
                        l *= alpha;
                        m = m_new;
                        if (j >= 2) {
                            // previous P V of this stream has completed (S_FULL tracks all earlier MMAs)
#pragma unroll
                            for (int c = 0; c < 4; ++c) {
                                uint32_t o[32];
                                tmem_ld32(tO + c * 32, o);
                                tc_wait_ld();
#pragma unroll
                                for (int k = 0; k < 32; ++k) o[k] = __float_as_uint(__uint_as_float(o[k]) * alpha);
                                tmem_st32(tO + c * 32, o);
                            }
                        }
                    }
                    const float neg_m = -m;
                    float sum0 = 0.f, sum1 = 0.f;
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        uint32_t pk[16];
#pragma unroll
                        for (int k = 0; k < 16; ++k) {
                            const float p0 = ex2(fmaf(__uint_as_float(sv[c * 32 + 2 * k]), sl2, neg_m));
                            const float p1 = ex2(fmaf(__uint_as_float(sv[c * 32 + 2 * k + 1]), sl2, neg_m));
                            sum0 += p0;
                            sum1 += p1;
                            pk[k] = pack_bf16x2(p0, p1);
                        }
                        tmem_st16(tS + c * 16, pk);
                    }
                    l += sum0 + sum1;
                    tc_wait_st();
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar(B_P_READY + s));
                }
            }
            // ---------------- epilogue: merge the two streams, normalise, store ------------------
            sml[s * 128 + row] = make_float2(m, l);
            if (lane == 0 && wq == 0) tma_store_wait_read();   // staging slab s free again
            named_bar_sync(1, 256);
            const float2 other = sml[(s ^ 1) * 128 + row];
            named_bar_sync(4, 256);   // both reads done before either warpgroup rewrites its slot
            const float m_all = fmaxf(m, other.x);
            const float a_self = (m == -INFINITY) ? 0.f : ex2(m - m_all);
            const float a_oth = (other.x == -INFINITY) ? 0.f : ex2(other.x - m_all);
            const float L = l * a_self + other.y * a_oth;
            const float inv = (L > 0.f) ? 1.f / L : 0.f;
            const float w_s0 = (s == 0 ? a_self : a_oth) * inv, w_s1 = (s == 0 ? a_oth : a_self) * inv;
            const bool has0 = it.np > 0, has1 = it.np > 1;
            if (it.nt > 0) {
                mbar_wait(bar(B_O_FULL), icnt & 1);
                ++icnt;
                tc_fence_after();
            }
            // this warpgroup finalises output columns [64 s, 64 s + 64)
            const uint32_t srow = sO + s * 16384 + row * 128;
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                uint32_t o0[32], o1[32];
                if (has0) tmem_ld32(tlane + TM_O0 + s * 64 + c * 32, o0);
                if (has1) tmem_ld32(tlane + TM_O1 + s * 64 + c * 32, o1);
                if (has0) tc_wait_ld();
                uint32_t pk[16];
#pragma unroll
                for (int k = 0; k < 16; ++k) {
                    float x0 = 0.f, x1 = 0.f;
                    if (has0) { x0 = __uint_as_float(o0[2 * k]) * w_s0; x1 = __uint_as_float(o0[2 * k + 1]) * w_s0; }
                    if (has1) { x0 = fmaf(__uint_as_float(o1[2 * k]), w_s1, x0); x1 = fmaf(__uint_as_float(o1[2 * k + 1]), w_s1, x1); }
                    pk[k] = pack_bf16x2(x0, x1);
                }
#pragma unroll
                for (int q4 = 0; q4 < 4; ++q4) {
                    const uint32_t chunk = (c * 4 + q4) ^ (row & 7);
                    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(srow + chunk * 16),
                                 "r"(pk[4 * q4]), "r"(pk[4 * q4 + 1]), "r"(pk[4 * q4 + 2]), "r"(pk[4 * q4 + 3])
                                 : "memory");
                }
            }
            if (it.nt > 0) {
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(B_O_FREE));
            }
            fence_proxy_async_smem();
            named_bar_sync(2 + s, 128);
            if (lane == 0 && wq == 0) {
                tma_store_4d(&tmO, sO + s * 16384, s * 64, it.qb * BQ, it.h, it.b);
                tma_store_commit();
            }
        }
        if (lane == 0 && wq == 0) tma_store_wait_all();
    }
    tc_fence_before();
    __syncthreads();
    if (warp == MMA_WARP) tmem_dealloc(tmem, TM_COLS);
}

}  // namespace

cudaError_t launch_attn_fwd(const CUtensorMap& tmQ, const CUtensorMap& tmK, const CUtensorMap& tmV,
                            const CUtensorMap& tmO, const AttnParams& p, chorus_dtype dtype,
                            cudaStream_t stream) {
    if (dtype != CHORUS_BF16) return cudaErrorNotSupported;
    cudaError_t e = cudaFuncSetAttribute(attn_fwd_kernel<false>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    if (e != cudaSuccess) return e;
    int dev = 0, sms = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    const int n_items = p.B * p.H * p.nq;
    const int grid = n_items < sms ? n_items : sms;
    attn_fwd_kernel<false><<<grid, NUM_THREADS, SMEM_BYTES, stream>>>(tmQ, tmK, tmV, tmO, p);
    count_launch(1);
    return cudaGetLastError();
}

}  // namespace chorus
