// attn_fwd.cu — chorus_block_sparse_attn_fwd for sm_100a ("skip pruned block pairs and
// evaluate only the retained ones in QK^T, softmax, and PV").
//
// Persistent, warp-specialised kernel, one CTA (384 threads) per SM:
//   warp 8        TMA producer: Q tile once per work item, then the kept K / V tiles of the CSR row,
//                 two 64-key tiles ("a pair") per pipeline stage, 128-byte swizzle
//   warp 9        MMA issuer (one thread): S = Q K^T (M=128, N=128, K=128) into one of THREE S
//                 buffers in tensor memory, up to two pairs ahead of the softmax; O += P V
//                 (M=128, N=128, K=128) with P as the TMEM A operand and V as an MN-major
//                 shared-memory B operand
//   warps 0-7     softmax.  Warp w owns TMEM lanes 32*(w%4).. (one query row per thread) and the
//                 64 score columns of tile (w/4) of the pair: warps w and w+4 share their rows'
//                 running max through shared memory and a 64-thread named barrier per pair.
// A work item is one (batch, head, 128-row query block).  Its kept tiles are paired (any two kept
// tiles, not necessarily adjacent keys) so that QK^T runs at N=128.  P (bf16) overwrites the first
// half of each warp's own S columns.  O (fp32, 128 columns of TMEM) is rescaled lazily: only when
// a row max grows by more than 2^8 over the reference that the accumulators currently use.  The
// epilogue normalises, converts to bf16, stages in shared memory and writes with TMA stores
// (coalesced 128-byte rows; rows beyond N are clipped by the tensor map).
//
// FP8 variant (template kFp8; R10-R12): e4m3 Q / K / V tiles (one 128-byte row holds all
// 128 channels), tcgen05.mma kind::f8f6f4 with fp32 accumulation, V again an MN-major B operand,
// P cast to e4m3 after a 2^5 shift, the Q / K block scales folded into the exp2 constant of each
// 64-key tile and V's per-channel scale applied in the epilogue.
#include <cuda_bf16.h>

#include "chorus_internal.h"
#include "sm100_ptx.cuh"

namespace chorus {
namespace {

using namespace ptx;

#ifndef CHORUS_POLY_MASK
#define CHORUS_POLY_MASK 0x00u   // e.g. 0x4A = 3 of every 8 element pairs
#endif
constexpr int BQ = 128, BK = 64;
constexpr int SBUFS = 3;
constexpr int NUM_THREADS = 384;
constexpr int PRODUCER_WARP = 8, MMA_WARP = 9;

// Per-dtype geometry.  A "slab" is a [128 rows][128 B] swizzled tile: 64 bf16 channels or all 128
// e4m3 channels of 128 rows (one Q block, or the two 64-key tiles of a pair).
template <bool kFp8>
struct Cfg {
    static constexpr uint32_t SLABS = kFp8 ? 1 : 2;                 // slabs per 128-row, 128-channel tile
    static constexpr uint32_t TILE_BYTES = SLABS * 16384;           // Q block, or one K / V pair stage
    static constexpr uint32_t HALF_BYTES = 8192;                    // second tile of a pair inside a slab
    static constexpr int KSTAGES = kFp8 ? 4 : 2, VSTAGES = kFp8 ? 4 : 3;
    static constexpr uint32_t KSTEPS = kFp8 ? 4 : 8;                // MMAs per 128-deep contraction
    // shared memory map (bytes from a 1024-aligned base)
    static constexpr uint32_t SQ_OFF = 0;
    static constexpr uint32_t SK_OFF = TILE_BYTES;
    static constexpr uint32_t SV_OFF = SK_OFF + KSTAGES * TILE_BYTES;
    static constexpr uint32_t SO_OFF = SV_OFF + VSTAGES * TILE_BYTES;   // O staging: 2 slabs (bf16 out)
    static constexpr uint32_t XCH_OFF = SO_OFF + 32768;   // row max / sum exchange [2 parity][2 half][128] f32
    static constexpr uint32_t BAR_OFF = XCH_OFF + 2048;
    static constexpr uint32_t SMEM_BYTES = BAR_OFF + 256;
    // mbarrier slots (8 bytes each) from BAR_OFF
    static constexpr uint32_t B_Q_FULL = 0, B_Q_EMPTY = 1, B_K_FULL = 2, B_K_EMPTY = B_K_FULL + KSTAGES,
        B_V_FULL = B_K_EMPTY + KSTAGES, B_V_EMPTY = B_V_FULL + VSTAGES, B_S_FULL = B_V_EMPTY + VSTAGES,
        B_P_READY = B_S_FULL + SBUFS, B_PV_DONE = B_P_READY + SBUFS, B_O_FREE = B_PV_DONE + SBUFS,
        B_COUNT = B_O_FREE + 1;
    static_assert(SMEM_BYTES <= 232448, "exceeds the 227 KB per-CTA shared memory of sm_100");
    static_assert(B_COUNT * 8 + 8 <= 256, "barrier area too small");
    // P: exp2(x - m_ref + P_SHIFT).  bf16 keeps P <= 2^8 under the lazy threshold; e4m3 (max 448,
    // smallest normal 2^-6) shifts P up by 2^5 and tightens the threshold to 2^3 so that P <= 2^8
    // still holds while probabilities down to 2^-11 of the row maximum stay normal numbers.
    static constexpr float RESCALE_THRESHOLD = kFp8 ? 3.0f : 8.0f;   // log2 units
    static constexpr float P_SHIFT = kFp8 ? 5.0f : 0.0f;
    // which element pairs (index mod 8) take the FMA-pipe polynomial exp2 instead of the MUFU, and
    // its degree (relative error 7.5e-5 / 1.7e-3, below the bf16 / e4m3 rounding of P)
    static constexpr uint32_t POLY_MASK = CHORUS_POLY_MASK;
    static constexpr int POLY_DEG = kFp8 ? 2 : 3;
};

// tensor-memory map (columns): three S buffers and the O accumulator
constexpr uint32_t TM_S = 0, TM_O = 384, TM_COLS = 512;

// named barriers: 0 = __syncthreads, 1..4 = warp pair (w, w+4), 5..6 = column-half warpgroup
constexpr uint32_t NB_PAIR = 1, NB_HALF = 5;

__device__ __forceinline__ void setmaxnreg_inc_216() { asm volatile("setmaxnreg.inc.sync.aligned.u32 216;"); }
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

__device__ __forceinline__ float max3(float a, float b, float c) { return fmaxf(fmaxf(a, b), c); }

template <bool kFp8>
__global__ void __launch_bounds__(NUM_THREADS, 1)
attn_fwd_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmO,
                const AttnParams p) {
    using C = Cfg<kFp8>;
    constexpr int KSTAGES = C::KSTAGES, VSTAGES = C::VSTAGES;
    constexpr uint32_t TILE = C::TILE_BYTES, HALF = C::HALF_BYTES;
    // 128-byte swizzle needs a 1024-byte aligned base; the kernel has no static shared memory, so
    // the dynamic window starts at the CTA's (1 KB granular) allocation.  Checked, not assumed.
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t base = smem_u32(smem_raw);
    if (base & 1023u) __trap();
    uint8_t* gbase = smem_raw;
    const uint32_t sQ = base + C::SQ_OFF, sK = base + C::SK_OFF, sV = base + C::SV_OFF, sO = base + C::SO_OFF;
    const uint32_t bars = base + C::BAR_OFF;
    auto bar = [&](uint32_t i) { return bars + 8u * i; };
    volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(gbase + C::BAR_OFF + 8 * C::B_COUNT);
    volatile float* xch = reinterpret_cast<volatile float*>(gbase + C::XCH_OFF);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_items = p.B * p.H * p.nq;

    if (threadIdx.x == 0) {
        mbar_init(bar(C::B_Q_FULL), 1);
        mbar_init(bar(C::B_Q_EMPTY), 1);
        for (int i = 0; i < KSTAGES; ++i) { mbar_init(bar(C::B_K_FULL + i), 1); mbar_init(bar(C::B_K_EMPTY + i), 1); }
        for (int i = 0; i < VSTAGES; ++i) { mbar_init(bar(C::B_V_FULL + i), 1); mbar_init(bar(C::B_V_EMPTY + i), 1); }
        for (int i = 0; i < SBUFS; ++i) {
            mbar_init(bar(C::B_S_FULL + i), 1);
            mbar_init(bar(C::B_P_READY + i), 8);
            mbar_init(bar(C::B_PV_DONE + i), 1);
        }
        mbar_init(bar(C::B_O_FREE), 8);
        fence_mbar_init();
    }
    if (warp == MMA_WARP) tmem_alloc(bars + 8 * C::B_COUNT, TM_COLS);
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
            // one 128-row, 128-channel box = SLABS loads of [rows][128 B]
            auto load_tile = [&](uint32_t dst, const CUtensorMap* tm, uint32_t b, int row0, int h, int bb) {
                tma_load_4d(dst, tm, b, 0, row0, h, bb);
                if constexpr (!kFp8) tma_load_4d(dst + 16384, tm, b, 64, row0, h, bb);
            };
            uint32_t g = 0, icnt = 0;   // pairs and non-empty items issued so far
            for (int idx = blockIdx.x; idx < n_items; idx += gridDim.x) {
                const Item it = get_item(p, idx);
                if (it.nt == 0) continue;   // empty rows touch no barrier
                mbar_wait(bar(C::B_Q_EMPTY), (icnt & 1) ^ 1);
                mbar_arrive_expect_tx(bar(C::B_Q_FULL), TILE);
                load_tile(sQ, &tmQ, bar(C::B_Q_FULL), it.qb * BQ, it.h, it.b);
                for (int j = 0; j < it.np; ++j, ++g) {
                    const int ntile = (2 * j + 1 < it.nt) ? 2 : 1;
                    const int kb0 = __ldg(p.col_idx + it.r0 + 2 * j);
                    const int kb1 = (ntile == 2) ? __ldg(p.col_idx + it.r0 + 2 * j + 1) : 0;
                    {
                        const uint32_t st = g % KSTAGES, ph = (g / KSTAGES) & 1;
                        mbar_wait(bar(C::B_K_EMPTY + st), ph ^ 1);
                        mbar_arrive_expect_tx(bar(C::B_K_FULL + st), ntile * (TILE / 2));
                        const uint32_t dst = sK + st * TILE;
                        load_tile(dst, &tmK, bar(C::B_K_FULL + st), kb0 * BK, it.h, it.b);
                        if (ntile == 2) load_tile(dst + HALF, &tmK, bar(C::B_K_FULL + st), kb1 * BK, it.h, it.b);
                    }
                    {
                        const uint32_t st = g % VSTAGES, ph = (g / VSTAGES) & 1;
                        mbar_wait(bar(C::B_V_EMPTY + st), ph ^ 1);
                        mbar_arrive_expect_tx(bar(C::B_V_FULL + st), ntile * (TILE / 2));
                        const uint32_t dst = sV + st * TILE;
                        load_tile(dst, &tmV, bar(C::B_V_FULL + st), kb0 * BK, it.h, it.b);
                        if (ntile == 2) load_tile(dst + HALF, &tmV, bar(C::B_V_FULL + st), kb1 * BK, it.h, it.b);
                    }
                }
                ++icnt;
            }
        } else if (warp == MMA_WARP && lane == 0) {
            // kind::f16: format 1 = bf16; kind::f8f6f4: format 0 = e4m3.  PV: B (= V) is MN-major.
            constexpr uint32_t FMT = kFp8 ? 0u : 1u;
            constexpr uint32_t IDESC_S128 = make_idesc(FMT, FMT, 128, 128, 0, 0);
            constexpr uint32_t IDESC_S64 = make_idesc(FMT, FMT, 128, 64, 0, 0);
            constexpr uint32_t IDESC_PV = make_idesc(FMT, FMT, 128, 128, 0, 1);
            const uint64_t dQ = smem_desc_sw128(sQ, 16, 1024);
            const uint64_t dK = smem_desc_sw128(sK, 16, 1024);
            const uint64_t dV = smem_desc_sw128(sV, 16384, 1024);
            uint32_t g0 = 0, icnt = 0;   // pairs before this item, non-empty items so far
            for (int idx = blockIdx.x; idx < n_items; idx += gridDim.x) {
                const Item it = get_item(p, idx);
                if (it.nt == 0) continue;
                mbar_wait(bar(C::B_Q_FULL), icnt & 1);
                for (int jj = 0; jj < it.np + 2; ++jj) {
                    if (jj < it.np) {   // S[g % 3] = Q K^T of pair jj (runs up to two pairs ahead)
                        const uint32_t g = g0 + jj;
                        const uint32_t st = g % KSTAGES, ph = (g / KSTAGES) & 1, sb = g % SBUFS;
                        const int ntile = (2 * jj + 1 < it.nt) ? 2 : 1;
                        mbar_wait(bar(C::B_K_FULL + st), ph);
                        tc_fence_after();
                        const uint32_t tS = tmem + TM_S + sb * 128;
                        const uint32_t idesc = (ntile == 2) ? IDESC_S128 : IDESC_S64;
                        const uint64_t dKs = dK + ((st * TILE) >> 4);
                        if constexpr (kFp8) {
#pragma unroll
                            for (int ks = 0; ks < 4; ++ks)       // 32 e4m3 channels = 32 B per step
                                mma_f8_ss(tS, dQ + ((ks * 32) >> 4), dKs + ((ks * 32) >> 4), idesc, ks > 0);
                        } else {
#pragma unroll
                            for (int ks = 0; ks < 8; ++ks) {     // 16 bf16 channels = 32 B per step, 2 slabs
                                const uint32_t off = ((ks >> 2) * 16384 + (ks & 3) * 32) >> 4;
                                mma_f16_ss(tS, dQ + off, dKs + off, idesc, ks > 0);
                            }
                        }
                        tc_commit(bar(C::B_K_EMPTY + st));
                        tc_commit(bar(C::B_S_FULL + sb));
                        if (jj == it.np - 1) tc_commit(bar(C::B_Q_EMPTY));
                    }
                    if (jj >= 2) {      // O += P V of pair jj - 2
                        const int jp = jj - 2;
                        const uint32_t g = g0 + jp;
                        const uint32_t st = g % VSTAGES, ph = (g / VSTAGES) & 1, sb = g % SBUFS;
                        const int ntile = (2 * jp + 1 < it.nt) ? 2 : 1;
                        mbar_wait(bar(C::B_P_READY + sb), (g / SBUFS) & 1);
                        mbar_wait(bar(C::B_V_FULL + st), ph);
                        if (jp == 0) mbar_wait(bar(C::B_O_FREE), (icnt & 1) ^ 1);
                        tc_fence_after();
                        const uint32_t tP = tmem + TM_S + sb * 128, tO = tmem + TM_O;
                        const uint64_t dVs = dV + ((st * TILE) >> 4);
                        if constexpr (kFp8) {
#pragma unroll
                            for (int ks = 0; ks < 4; ++ks) {     // 32 keys per step: 8 TMEM columns of e4m3 P
                                if (ks < 2 * ntile) {
                                    // P of tile 0 lives in S columns [0, 16), P of tile 1 in [64, 80)
                                    const uint32_t ta = tP + (ks >> 1) * 64 + (ks & 1) * 8;
                                    mma_f8_ts(tO, ta, dVs + ((ks * 4096u) >> 4), IDESC_PV, (jp > 0) || (ks > 0));
                                }
                            }
                        } else {
#pragma unroll
                            for (int ks = 0; ks < 8; ++ks) {     // 16 keys per step: 8 TMEM columns of bf16 P
                                if (ks < 4 * ntile) {
                                    // P of tile 0 lives in S columns [0, 32), P of tile 1 in [64, 96)
                                    const uint32_t ta = tP + (ks >> 2) * 64 + (ks & 3) * 8;
                                    mma_f16_ts(tO, ta, dVs + ((ks * 2048u) >> 4), IDESC_PV, (jp > 0) || (ks > 0));
                                }
                            }
                        }
                        tc_commit(bar(C::B_V_EMPTY + st));
                        tc_commit(bar(C::B_PV_DONE + sb));
                    }
                }
                g0 += it.np;
                ++icnt;
            }
        }
    } else {
        // ======================= softmax warps ======================================================
        setmaxnreg_inc_216();
        const int s = warp >> 2;                 // which tile of the pair: score columns [64 s, 64 s + 64)
        const int wq = warp & 3;                 // TMEM lane quarter
        const int row = wq * 32 + lane;          // query row inside the block == TMEM lane
        const uint32_t tlane = tmem + (static_cast<uint32_t>(wq * 32) << 16);
        const uint32_t tO = tlane + TM_O + s * 64;   // this warp rescales / finalises O columns [64 s, 64 s + 64)
        const int nsb = (p.N + 127) >> 7;        // FP8: Q/K scale blocks of 128 tokens
        uint32_t g = 0;                          // pairs processed so far (all items)
        uint32_t xc = 0;                         // exchanges so far: slot parity (two slots, one barrier each)
        for (int idx = blockIdx.x; idx < n_items; idx += gridDim.x) {
            const Item it = get_item(p, idx);
            float m_ref = -INFINITY, l0 = 0.f, l1 = 0.f;
            // FP8 (R10): scores are (q8 . k8) * s_q[qb] * s_k[kb / 2]; the per-tile factor is
            // folded into the exp2 FMA constant.  kb (and its scale) of the NEXT pair are fetched
            // one pair ahead so that the loads are off the critical path.
            float sl2 = p.scale_log2;
            float qsl2 = 0.f;
            const float* ksc = nullptr;
            int kb_next = 0;
            if constexpr (kFp8) {
                const int64_t sbase = (static_cast<int64_t>(it.b) * p.H + it.h) * nsb;
                qsl2 = p.scale_log2 * __ldg(p.q_scale + sbase + it.qb);
                ksc = p.k_scale + sbase;
                if (s < it.nt) kb_next = __ldg(p.col_idx + it.r0 + s);
            }
            for (int j = 0; j < it.np; ++j, ++g) {
                const uint32_t sb = g % SBUFS;
                const uint32_t tS = tlane + TM_S + sb * 128 + s * 64;
                int valid = BK;                  // valid keys in this warp's tile of the pair
                int kb = 0;
                if constexpr (kFp8) {
                    kb = kb_next;
                    if (2 * (j + 1) + s < it.nt) kb_next = __ldg(p.col_idx + it.r0 + 2 * (j + 1) + s);
                    sl2 = qsl2 * __ldg(ksc + (kb >> 1));
                }
                if (j == it.np - 1) {            // only the last pair can be odd or hold the ragged key block
                    if (2 * j + s < it.nt) {
                        if constexpr (!kFp8) kb = __ldg(p.col_idx + it.r0 + 2 * j + s);
                        valid = min(BK, p.N - kb * BK);
                    } else {
                        valid = 0;
                    }
                }
                mbar_wait(bar(C::B_S_FULL + sb), (g / SBUFS) & 1);
                tc_fence_after();
                uint32_t sv[64];
                float mx = -INFINITY;
                if (valid > 0) {
                    tmem_ld32(tS, *reinterpret_cast<uint32_t(*)[32]>(sv));
                    tmem_ld32(tS + 32, *reinterpret_cast<uint32_t(*)[32]>(sv + 32));
                    tc_wait_ld();
                    if (valid < BK) {
#pragma unroll
                        for (int k = 0; k < 64; ++k)
                            if (k >= valid) sv[k] = 0xff800000u;   // -inf
                    }
                    float a0 = -INFINITY, a1 = -INFINITY, a2 = -INFINITY, a3 = -INFINITY;
#pragma unroll
                    for (int k = 0; k < 64; k += 8) {
                        a0 = max3(a0, __uint_as_float(sv[k]), __uint_as_float(sv[k + 1]));
                        a1 = max3(a1, __uint_as_float(sv[k + 2]), __uint_as_float(sv[k + 3]));
                        a2 = max3(a2, __uint_as_float(sv[k + 4]), __uint_as_float(sv[k + 5]));
                        a3 = max3(a3, __uint_as_float(sv[k + 6]), __uint_as_float(sv[k + 7]));
                    }
                    mx = fmaxf(fmaxf(a0, a1), fmaxf(a2, a3)) * sl2;   // sl2 > 0
                }
                // the row max of the pair: exchange with the warp that holds the other 64 columns
                const uint32_t par = (xc++) & 1;
                xch[(par * 2 + s) * 128 + row] = mx;
                named_bar_sync(NB_PAIR + wq, 64);
                const float mt = fmaxf(mx, xch[(par * 2 + (s ^ 1)) * 128 + row]);
                if (__any_sync(0xffffffffu, mt > m_ref + C::RESCALE_THRESHOLD)) {
                    // identical decision in both warps of the pair (same mt, same m_ref per row)
                    const float m_new = fmaxf(m_ref, mt);
                    const float alpha = ex2(m_ref - m_new);   // m_ref = -inf (first pair) -> 0
                    l0 *= alpha;
                    l1 *= alpha;
                    m_ref = m_new;
                    if (j > 0) {
                        // O holds pairs 0..j-1 under the old reference; wait for P V of pair j-1.
                        // (S_FULL of pair g implies P V of pair g-3 is complete, so the barrier of
                        // buffer (g-1) % 3 is at most one phase behind: the parity wait is exact.)
                        mbar_wait(bar(C::B_PV_DONE + (g - 1) % SBUFS), ((g - 1) / SBUFS) & 1);
                        tc_fence_after();
#pragma unroll 1
                        for (int c = 0; c < 2; ++c) {
                            uint32_t o[32];
                            tmem_ld32(tO + c * 32, o);
                            tc_wait_ld();
#pragma unroll
                            for (int k = 0; k < 32; ++k) o[k] = __float_as_uint(__uint_as_float(o[k]) * alpha);
                            tmem_st32(tO + c * 32, o);
                        }
                    }
                }
                if (valid > 0) {
                    // P = exp2(s * sl2 - m_ref + shift).  Element pairs go through packed FFMA2; the
                    // pairs whose bit is set in POLY_MASK (index mod 8) take the polynomial exp2 on
                    // the FMA pipe, the rest the MUFU, so that both pipes finish together.
                    const float2 sl2_2 = make_float2(sl2, sl2);
                    const float2 negm_2 = make_float2(C::P_SHIFT - m_ref, C::P_SHIFT - m_ref);
                    auto exp_pair = [&](int q) -> float2 {     // q: element pair index 0..31
                        const float2 x = ffma2(make_float2(__uint_as_float(sv[2 * q]), __uint_as_float(sv[2 * q + 1])),
                                               sl2_2, negm_2);
                        if ((C::POLY_MASK >> (q & 7)) & 1u) return exp2_poly2<C::POLY_DEG>(x);
                        return make_float2(ex2(x.x), ex2(x.y));
                    };
                    if constexpr (kFp8) {
                        // The denominator sums the e4m3-ROUNDED weights (two f16x2 accumulators per
                        // 32 keys: at most 8 x 2^8 each, exact to 2^-11), i.e. exactly what P V uses.
#pragma unroll
                        for (int c = 0; c < 2; ++c) {            // 32 keys -> 8 columns of 4 e4m3 each
                            uint32_t pk[8];
                            uint32_t h0 = 0u, h1 = 0u;
#pragma unroll
                            for (int k = 0; k < 8; ++k) {
                                const float2 pa = exp_pair(c * 16 + 2 * k), pb = exp_pair(c * 16 + 2 * k + 1);
                                pk[k] = pack_e4m3x4_acc(pa.x, pa.y, pb.x, pb.y, h0, h1);
                            }
                            l0 += f16x2_hsum(h0);
                            l1 += f16x2_hsum(h1);
                            tmem_st8(tS + c * 8, pk);   // P: e4m3 quads over this warp's first 16 S columns
                        }
                    } else {
                        float2 lacc = make_float2(l0, l1);
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            uint32_t pk[8];
#pragma unroll
                            for (int k = 0; k < 8; ++k) {
                                const float2 pp = exp_pair(c * 8 + k);
                                lacc = fadd2(lacc, pp);
                                pk[k] = pack_bf16x2(pp.x, pp.y);
                            }
                            tmem_st8(tS + c * 8, pk);   // P: bf16 pairs over this warp's first 32 S columns
                        }
                        l0 = lacc.x;
                        l1 = lacc.y;
                    }
                }
                tc_wait_st();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(C::B_P_READY + sb));
            }
            // ---------------- epilogue: normalise, convert, store --------------------------------
            const float l = l0 + l1;
            const uint32_t par = (xc++) & 1;
            xch[(par * 2 + s) * 128 + row] = l;
            if (lane == 0 && wq == 0) tma_store_wait_read();   // staging slab s is free again
            named_bar_sync(NB_PAIR + wq, 64);
            const float L = l + xch[(par * 2 + (s ^ 1)) * 128 + row];
            const float inv = (L > 0.f) ? 1.f / L : 0.f;
            named_bar_sync(NB_HALF + s, 128);                  // staging free for the whole warpgroup
            if (it.nt > 0) {
                mbar_wait(bar(C::B_PV_DONE + (g - 1) % SBUFS), ((g - 1) / SBUFS) & 1);
                tc_fence_after();
            }
            const uint32_t srow = sO + s * 16384 + row * 128;
            // FP8: O[:, c] carries V's per-channel scale (R10)
            const float4* vsc = nullptr;
            if constexpr (kFp8)
                vsc = reinterpret_cast<const float4*>(p.v_scale + (static_cast<int64_t>(it.b) * p.H + it.h) * 128 + s * 64);
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                uint32_t o[32];
                if (it.nt > 0) {
                    tmem_ld32(tO + c * 32, o);
                    tc_wait_ld();
                }
                uint32_t pk[16];
#pragma unroll
                for (int k4 = 0; k4 < 8; ++k4) {
                    float4 w = make_float4(inv, inv, inv, inv);
                    if constexpr (kFp8) {
                        const float4 sc = __ldg(vsc + c * 8 + k4);
                        w = make_float4(inv * sc.x, inv * sc.y, inv * sc.z, inv * sc.w);
                    }
                    float x0 = 0.f, x1 = 0.f, x2 = 0.f, x3 = 0.f;
                    if (it.nt > 0) {
                        x0 = __uint_as_float(o[4 * k4]) * w.x;     x1 = __uint_as_float(o[4 * k4 + 1]) * w.y;
                        x2 = __uint_as_float(o[4 * k4 + 2]) * w.z; x3 = __uint_as_float(o[4 * k4 + 3]) * w.w;
                    }
                    pk[2 * k4] = pack_bf16x2(x0, x1);
                    pk[2 * k4 + 1] = pack_bf16x2(x2, x3);
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
                if (lane == 0) mbar_arrive(bar(C::B_O_FREE));
            }
            fence_proxy_async_smem();
            named_bar_sync(NB_HALF + s, 128);
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

template <bool kFp8>
static cudaError_t launch_one(const CUtensorMap& tmQ, const CUtensorMap& tmK, const CUtensorMap& tmV,
                              const CUtensorMap& tmO, const AttnParams& p, cudaStream_t stream) {
    constexpr uint32_t smem = Cfg<kFp8>::SMEM_BYTES;
    cudaError_t e = cudaFuncSetAttribute(attn_fwd_kernel<kFp8>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    int dev = 0, sms = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    const int n_items = p.B * p.H * p.nq;
    const int grid = n_items < sms ? n_items : sms;
    attn_fwd_kernel<kFp8><<<grid, NUM_THREADS, smem, stream>>>(tmQ, tmK, tmV, tmO, p);
    count_launch(1);
    return cudaGetLastError();
}

cudaError_t launch_attn_fwd(const CUtensorMap& tmQ, const CUtensorMap& tmK, const CUtensorMap& tmV,
                            const CUtensorMap& tmO, const AttnParams& p, chorus_dtype dtype,
                            cudaStream_t stream) {
    if (dtype == CHORUS_BF16) return launch_one<false>(tmQ, tmK, tmV, tmO, p, stream);
    if (dtype == CHORUS_FP8_E4M3) return launch_one<true>(tmQ, tmK, tmV, tmO, p, stream);
    return cudaErrorNotSupported;
}

}  // namespace chorus
