// attn_fwd.cu — chorus_block_sparse_attn_fwd for sm_100a ("skip pruned block pairs and
// evaluate only the retained ones in QK^T, softmax, and PV").
//
// Persistent, warp-specialised kernel, one CTA (384 threads) per SM.  A work item is one (batch,
// head, 128-row query block).  Its kept 64-key tiles are taken two at a time ("a pair": any two kept
// tiles, not necessarily adjacent keys) so that QK^T runs at N=128.
//   warp 8        TMA producer: Q tile once per item, then the K / V tiles of every pair into two
//                 rings, 128-byte swizzle
//   warp 9        MMA issuer (one thread): S = Q K^T (M=128, N=128, K=128) into one of THREE S buffers
//                 in tensor memory, up to two pairs ahead of the softmax; O += P V (P the TMEM A
//                 operand, V an MN-major shared-memory B operand) into ONE accumulator
//   warps 0-3     softmax of the even pairs of an item; warps 4-7 of the odd pairs.  Warp w owns TMEM
//                 lanes 32*(w%4).. (one query row per thread) and all 128 score columns of its
//                 pair.  The two warps of an SM sub-partition (w, w+4) therefore work on
//                 consecutive pairs, half a period apart: one's exp phase (MUFU) overlaps the
//                 other's load / max phase.  They share one running reference m_ref per row, handed
//                 from pair j to pair j+1 through shared memory and a 64-thread named barrier
//                 (arrive after the max pass of pair j, sync before the exp pass of pair j+1).
// The 128 scores of a row are streamed from tensor memory twice, 32 columns at a time (max pass,
// then exp pass), so only 64 are live in registers.  P (bf16 / fp16) overwrites the first columns of
// its S buffer behind the read position.  O (fp32, 128 TMEM columns) is rescaled lazily: only when a
// row max grows by more than 2^8 over m_ref.  The epilogue adds the two warps' partial
// row sums, normalises, converts to bf16, stages in shared memory and writes with TMA stores
// (coalesced 128-byte rows; rows beyond N are clipped by the tensor map).
//
// FP16 variant (template kF16; "for the non-quantized (fp16) path"): fp16 Q / K / V, P
// and O; the same pipeline with the kind::f16 operand format switched.
//
// The FP8 (e4m3) path is a kernel of its own: attn_fwd_fp8.cu.
#include <cuda_bf16.h>

#include "attn_common.cuh"

namespace chorus {
namespace {

using namespace ptx;
using namespace attn;

constexpr int SBUFS = 3;

// Geometry.  A "slab" is a [128 rows][128 B] swizzled tile: 64 of the 128 channels of 128 rows (one Q
// block, or the two 64-key tiles of a pair).
struct Cfg {
    static constexpr uint32_t SLABS = 2;                            // slabs per 128-row, 128-channel tile
    static constexpr uint32_t TILE_BYTES = SLABS * 16384;           // Q block, or one K / V pair stage
    static constexpr uint32_t HALF_BYTES = 8192;                    // second tile of a pair inside a slab
    static constexpr int KSTAGES = 2, VSTAGES = 3;
    // shared memory map (bytes from a 1024-aligned base)
    static constexpr uint32_t SQ_OFF = 0;
    static constexpr uint32_t SK_OFF = TILE_BYTES;
    static constexpr uint32_t SV_OFF = SK_OFF + KSTAGES * TILE_BYTES;
    static constexpr uint32_t SO_OFF = SV_OFF + VSTAGES * TILE_BYTES;   // O staging: 2 slabs (bf16 out)
    static constexpr uint32_t XCH_OFF = SO_OFF + 32768;   // f32 [128] m_ref hand-off, [2][2][128] epilogue (m, l)
    static constexpr uint32_t BAR_OFF = XCH_OFF + 2560;
    static constexpr uint32_t SMEM_BYTES = BAR_OFF + 384;
    // mbarrier slots (8 bytes each) from BAR_OFF
    static constexpr uint32_t B_Q_FULL = 0, B_Q_EMPTY = 1, B_K_FULL = 2, B_K_EMPTY = B_K_FULL + KSTAGES,
        B_V_FULL = B_K_EMPTY + KSTAGES, B_V_EMPTY = B_V_FULL + VSTAGES, B_S_FULL = B_V_EMPTY + VSTAGES,
        B_P_READY = B_S_FULL + SBUFS, B_PV_DONE = B_P_READY + SBUFS, B_ITEM_DONE = B_PV_DONE + SBUFS,
        B_O_FREE = B_ITEM_DONE + 1, B_IT_FULL = B_O_FREE + 1, B_IT_EMPTY = B_IT_FULL + ITEM_RING,
        B_COUNT = B_IT_EMPTY + ITEM_RING;
    static_assert(SMEM_BYTES <= 232448, "exceeds the 227 KB per-CTA shared memory of sm_100");
    static_assert(B_COUNT * 8 + 8 + 4 * ITEM_RING <= 384, "barrier area too small");
    // P = exp2(x - m_ref) <= 2^8 under the lazy-rescale threshold of 2^8 (log2 units below)
    static constexpr float RESCALE_THRESHOLD = 8.0f;
    // P V steps per 64-key tile: 16 keys (8 TMEM columns of bf16 / fp16 pairs) per MMA
    static constexpr int PV_STEPS_PER_TILE = 4;
};

// tensor-memory map (columns): three S buffers (each aliased by its P) and the O accumulator
constexpr uint32_t TM_S = 0, TM_O = 384, TM_COLS = 512;

// named barriers: 0 = __syncthreads, 1..4 = warp pair (w, w+4) in the epilogue, 5..6 = column-half
// warpgroup, 7..14 = m_ref hand-off published by parity 0 (7..10) / parity 1 (11..14) of quarter wq
constexpr uint32_t NB_PAIR = 1, NB_HALF = 5, NB_HAND = 7;

// kBeta: first-frame key enhancement (eq. (1)) as a factor on the scores of keys < n_first
// kHalf: col_idx entries carry per-half flags (bit 30 / 31: query rows 0-63 / 64-127 of the block do NOT keep the
// tile), as chorus_mask_to_index_64x128 writes them for masks in the paper's 64 x 128 geometry
template <bool kF16, bool kBeta, bool kHalf>   // fp16 inputs and output (else bf16)
__global__ void __launch_bounds__(NUM_THREADS, 1)
attn_fwd_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmO,
                const AttnParams p) {
    using C = Cfg;
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
    const ItemRing ring{bar(C::B_IT_FULL), bar(C::B_IT_EMPTY),
                        reinterpret_cast<volatile int*>(gbase + C::BAR_OFF + 8 * C::B_COUNT + 8)};

    if (threadIdx.x == 0) {
        mbar_init(bar(C::B_Q_FULL), 1);
        mbar_init(bar(C::B_Q_EMPTY), 1);
        for (int i = 0; i < KSTAGES; ++i) { mbar_init(bar(C::B_K_FULL + i), 1); mbar_init(bar(C::B_K_EMPTY + i), 1); }
        for (int i = 0; i < VSTAGES; ++i) { mbar_init(bar(C::B_V_FULL + i), 1); mbar_init(bar(C::B_V_EMPTY + i), 1); }
        for (int i = 0; i < SBUFS; ++i) {
            mbar_init(bar(C::B_S_FULL + i), 1);
            mbar_init(bar(C::B_P_READY + i), 4);
            mbar_init(bar(C::B_PV_DONE + i), 1);
        }
        mbar_init(bar(C::B_ITEM_DONE), 1);
        mbar_init(bar(C::B_O_FREE), 8);
        for (int i = 0; i < ITEM_RING; ++i) { mbar_init(bar(C::B_IT_FULL + i), 1); mbar_init(bar(C::B_IT_EMPTY + i), 9); }   // MMA warp + 8 softmax warps
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
        // Both roles run with the WHOLE warp converged (all lanes wait on the barriers and keep the
        // same loop state); one elected lane issues the TMA / tcgen05 instructions.  Everything an
        // issue needs is made warp-uniform with a shuffle first, so that the compiler keeps the
        // descriptors and coordinates in uniform registers instead of wrapping every issue in a
        // per-lane loop (which made the single-thread issue stream the bottleneck of the kernel).
        if (warp == PRODUCER_WARP) {
            // one 128-row, 128-channel box = SLABS loads of [rows][128 B]
            auto load_tile = [&](uint32_t dst, const CUtensorMap* tm, uint32_t b, int row0, int h, int bb) {
                tma_load_4d(dst, tm, b, 0, row0, h, bb);
                tma_load_4d(dst + 16384, tm, b, 64, row0, h, bb);
            };
            uint32_t g = 0, icnt = 0;   // pairs and non-empty items issued so far
            for (uint32_t kit = 0;; ++kit) {
                const int idx = item_draw(ring, kit, n_items, p.ticket_slot);
                if (idx < 0) break;
                const Item it = get_item_uniform(p, idx);
                if (it.nt == 0) continue;   // empty rows touch no barrier
                mbar_wait(bar(C::B_Q_EMPTY), (icnt & 1) ^ 1);
                if (elect_one()) {
                    mbar_arrive_expect_tx(bar(C::B_Q_FULL), TILE);
                    load_tile(sQ, &tmQ, bar(C::B_Q_FULL), it.qb * BQ, it.h, it.b);
                }
                __syncwarp();
                // the key-block indices of 16 pairs are fetched with one coalesced load
                for (int j0 = 0; j0 < it.np; j0 += 16) {
                    const int t = 2 * j0 + lane;
                    int mine = (t < it.nt) ? ld_col(p, it.r0 + t) : 0;
                    if constexpr (kHalf) mine &= 0x3fffffff;
                    const int jn = min(16, it.np - j0);
                    for (int jl = 0; jl < jn; ++jl, ++g) {
                        const int ntile = (2 * (j0 + jl) + 1 < it.nt) ? 2 : 1;
                        const int kb0 = __shfl_sync(0xffffffffu, mine, 2 * jl);
                        const int kb1 = __shfl_sync(0xffffffffu, mine, 2 * jl + 1);
                        {
                            const uint32_t st = g % KSTAGES, ph = (g / KSTAGES) & 1;
                            mbar_wait(bar(C::B_K_EMPTY + st), ph ^ 1);
                            if (elect_one()) {
                                mbar_arrive_expect_tx(bar(C::B_K_FULL + st), ntile * (TILE / 2));
                                const uint32_t dst = sK + st * TILE;
                                load_tile(dst, &tmK, bar(C::B_K_FULL + st), kb0 * BK, it.h, it.b);
                                if (ntile == 2) load_tile(dst + HALF, &tmK, bar(C::B_K_FULL + st), kb1 * BK, it.h, it.b);
                            }
                            __syncwarp();
                        }
                        {
                            const uint32_t st = g % VSTAGES, ph = (g / VSTAGES) & 1;
                            mbar_wait(bar(C::B_V_EMPTY + st), ph ^ 1);
                            if (elect_one()) {
                                mbar_arrive_expect_tx(bar(C::B_V_FULL + st), ntile * (TILE / 2));
                                const uint32_t dst = sV + st * TILE;
                                load_tile(dst, &tmV, bar(C::B_V_FULL + st), kb0 * BK, it.h, it.b);
                                if (ntile == 2) load_tile(dst + HALF, &tmV, bar(C::B_V_FULL + st), kb1 * BK, it.h, it.b);
                            }
                            __syncwarp();
                        }
                    }
                }
                ++icnt;
            }
        } else if (warp == MMA_WARP) {
            // kind::f16: format 1 = bf16; kind::f8f6f4: format 0 = e4m3.  PV: B (= V) is MN-major.
            constexpr uint32_t FMT = kF16 ? 0u : 1u;   // kind::f16: 0 = fp16, 1 = bf16
            constexpr uint32_t IDESC_S128 = make_idesc(FMT, FMT, 128, 128, 0, 0);
            constexpr uint32_t IDESC_S64 = make_idesc(FMT, FMT, 128, 64, 0, 0);
            constexpr uint32_t IDESC_PV = make_idesc(FMT, FMT, 128, 128, 0, 1);   // A and B formats must agree in kind::f16
            const uint64_t dQ = smem_desc_sw128(sQ, 16, 1024);
            const uint64_t dK = smem_desc_sw128(sK, 16, 1024);
            const uint64_t dV = smem_desc_sw128(sV, 16384, 1024);
            uint32_t g0 = 0, icnt = 0;      // pairs before this item, non-empty items so far
            for (uint32_t kit = 0;; ++kit) {
                const int idx = item_take(ring, kit);
                if (idx < 0) break;
                const Item it = get_item_uniform(p, idx);
                if (it.nt == 0) continue;
                mbar_wait(bar(C::B_Q_FULL), icnt & 1);
                for (int jj = 0; jj < it.np + 2; ++jj) {
                    if (jj < it.np) {   // S[g % 3] = Q K^T of pair jj (runs up to two pairs ahead)
                        const uint32_t g = g0 + jj;
                        const uint32_t st = g % KSTAGES, ph = (g / KSTAGES) & 1, sb = g % SBUFS;
                        const bool two = 2 * jj + 1 < it.nt;
                        mbar_wait(bar(C::B_K_FULL + st), ph);
                        tc_fence_after();
                        if (elect_one()) {
                            const uint32_t tS = tmem + TM_S + sb * 128;
                            const uint32_t idesc = two ? IDESC_S128 : IDESC_S64;
                            const uint64_t dKs = dK + ((st * TILE) >> 4);
#pragma unroll
                            for (int ks = 0; ks < 8; ++ks) {     // 16 channels = 32 B per step, 2 slabs
                                const uint32_t off = ((ks >> 2) * 16384 + (ks & 3) * 32) >> 4;
                                mma_f16_ss(tS, dQ + off, dKs + off, idesc, ks > 0);
                            }
                            tc_commit(bar(C::B_K_EMPTY + st));
                            tc_commit(bar(C::B_S_FULL + sb));
                            if (jj == it.np - 1) tc_commit(bar(C::B_Q_EMPTY));
                        }
                        __syncwarp();
                    }
                    if (jj >= 2) {      // O += P V of pair jj - 2
                        const int jp = jj - 2;
                        const uint32_t g = g0 + jp;
                        const uint32_t st = g % VSTAGES, ph = (g / VSTAGES) & 1, sb = g % SBUFS;
                        const bool two = 2 * jp + 1 < it.nt;
                        mbar_wait(bar(C::B_P_READY + sb), (g / SBUFS) & 1);
                        mbar_wait(bar(C::B_V_FULL + st), ph);
                        if (jp == 0) mbar_wait(bar(C::B_O_FREE), (icnt & 1) ^ 1);
                        tc_fence_after();
                        if (elect_one()) {
                            const uint32_t tP = tmem + TM_S + sb * 128, tO = tmem + TM_O;
                            const uint64_t dVs = dV + ((st * TILE) >> 4);
                            constexpr uint32_t KBYTES = 2048u;   // 16 keys x 128 B per step
                            constexpr int STEPS = C::PV_STEPS_PER_TILE;
#pragma unroll
                            for (int ks = 0; ks < STEPS; ++ks) {
                                const uint32_t acc = (jp > 0) || (ks > 0);
                                mma_f16_ts(tO, tP + ks * 8, dVs + ((ks * KBYTES) >> 4), IDESC_PV, acc);
                            }
                            if (two) {
#pragma unroll
                                for (int ks = STEPS; ks < 2 * STEPS; ++ks) {
                                    mma_f16_ts(tO, tP + ks * 8, dVs + ((ks * KBYTES) >> 4), IDESC_PV, 1u);
                                }
                            }
                            tc_commit(bar(C::B_V_EMPTY + st));
                            tc_commit(bar(C::B_PV_DONE + sb));
                            if (jp == it.np - 1) tc_commit(bar(C::B_ITEM_DONE));
                        }
                        __syncwarp();
                    }
                }
                g0 += it.np;
                ++icnt;
            }
        }
    } else {
        // ======================= softmax warps ======================================================
        setmaxnreg_inc_216();
        const int sm = warp >> 2;                // parity: pairs sm, sm + 2, ... of every item
        const int wq = warp & 3;                 // TMEM lane quarter
        const int row = wq * 32 + lane;          // query row inside the block == TMEM lane
        const uint32_t tlane = tmem + (static_cast<uint32_t>(wq * 32) << 16);
        const uint32_t tOs = tlane + TM_O;       // the O accumulator (all 128 columns of this row)
        volatile float* xm = xch;                // [128] m_ref hand-off between the two parities
        volatile float* xe = xch + 128;          // [2 parity][m, l][128] epilogue exchange
        uint32_t g0 = 0;                         // pairs of all previous items (S buffer / phase)
        uint32_t icnt = 0;                       // non-empty items so far
        for (uint32_t kit = 0;; ++kit) {
            const int idx = item_take(ring, kit);
            if (idx < 0) break;
            const Item it = get_item(p, idx);
            float m_ref = -INFINITY, l0 = 0.f, l1 = 0.f;
            // FP8 (R10): scores are (q8 . k8) * s_q[qb] * s_k[kb / 2]; the per-tile factor is
            // folded into the exp2 FMA constant.  The key-block indices of the stream's NEXT pair are
            // fetched one pair ahead so that the loads are off the critical path.
            float sl2a = p.scale_log2, sl2b = p.scale_log2;
            int kba_next = 0, kbb_next = 0;
            if constexpr (kBeta || kHalf) {
                if (2 * sm < it.nt) kba_next = ld_col(p, it.r0 + 2 * sm);
                if (2 * sm + 1 < it.nt) kbb_next = ld_col(p, it.r0 + 2 * sm + 1);
            }
            for (int j = sm; j < it.np; j += 2) {
                const uint32_t g = g0 + j, sb = g % SBUFS;
                const uint32_t tS = tlane + TM_S + sb * 128;     // this pair's S, overwritten by its P
                int va = BK, vb = BK;            // valid keys in the two tiles of the pair
                int kba = 0, kbb = 0;
                if constexpr (kBeta || kHalf) {
                    kba = kba_next;
                    kbb = kbb_next;
                    if (2 * (j + 2) < it.nt) kba_next = ld_col(p, it.r0 + 2 * (j + 2));
                    if (2 * (j + 2) + 1 < it.nt) kbb_next = ld_col(p, it.r0 + 2 * (j + 2) + 1);
                }
                uint32_t skip_a = 0u, skip_b = 0u;   // kHalf: this warp's rows do not keep tile a / b
                if constexpr (kHalf) {
                    const int hb = 30 + (wq >> 1);
                    skip_a = (static_cast<uint32_t>(kba) >> hb) & 1u;
                    skip_b = (static_cast<uint32_t>(kbb) >> hb) & 1u;
                    kba &= 0x3fffffff;
                    kbb &= 0x3fffffff;
                }
                // kBeta: a tile inside the first frame takes beta in its scale factor; the one tile
                // that straddles n_first takes it per column (fa / fb leading columns) in the masked body
                int fa = 0, fb = 0;
                if constexpr (kBeta) {
                    sl2a = sl2b = p.scale_log2;
                    fa = min(BK, max(0, p.n_first - kba * BK));
                    fb = (2 * j + 1 < it.nt) ? min(BK, max(0, p.n_first - kbb * BK)) : 0;
                    if (fa == BK) { sl2a *= p.beta; fa = 0; }
                    if (fb == BK) { sl2b *= p.beta; fb = 0; }
                }
                if (j == it.np - 1) {            // only the last pair can be odd or hold the ragged key block
                    if constexpr (!(kBeta || kHalf)) {
                        kba = ld_col(p, it.r0 + 2 * j);
                        if (2 * j + 1 < it.nt) kbb = ld_col(p, it.r0 + 2 * j + 1);
                    }
                    va = min(BK, p.N - kba * BK);
                    vb = (2 * j + 1 < it.nt) ? min(BK, p.N - kbb * BK) : 0;
                }
                if constexpr (kHalf) {           // a tile the rows of this warp do not keep: all -inf
                    if (skip_a) va = 0;
                    if (skip_b) vb = 0;
                }
                mbar_wait(bar(C::B_S_FULL + sb), (g / SBUFS) & 1);
                tc_fence_after();
                // The 128 scores of a row are streamed from tensor memory twice, 32 columns at a time
                // with the next chunk's load in flight (pass 1: row max; pass 2: exp, pack, store P
                // behind the read position), so that only 64 of them are ever live in registers.
                const bool ragged = (va < BK) || (vb < BK) || (fa | fb) != 0;   // warp-uniform and rare
                // The body is instantiated twice (with / without tail masking) so that the common
                // case carries no branch: the compiler can then schedule across the chunks.
                auto pair_body = [&](auto rag_tag) {
                constexpr bool RAG = decltype(rag_tag)::value;
                auto mask_chunk = [&](uint32_t (&r)[32], int c) {
                    const int valid = ((c >> 1) ? vb : va) - 32 * (c & 1);
#pragma unroll
                    for (int k = 0; k < 32; ++k)
                        if (k >= valid) r[k] = 0xff800000u;   // -inf
                    if constexpr (kBeta) {
                        const int nf = ((c >> 1) ? fb : fa) - 32 * (c & 1);
#pragma unroll
                        for (int k = 0; k < 32; ++k)
                            if (k < nf) r[k] = __float_as_uint(__uint_as_float(r[k]) * p.beta);
                    }
                };
                auto max32 = [](const uint32_t (&r)[32]) {
                    float a0 = -INFINITY, a1 = -INFINITY;
#pragma unroll
                    for (int k = 0; k < 32; k += 4) {
                        a0 = max3(a0, __uint_as_float(r[k]), __uint_as_float(r[k + 1]));
                        a1 = max3(a1, __uint_as_float(r[k + 2]), __uint_as_float(r[k + 3]));
                    }
                    return fmaxf(a0, a1);
                };
                uint32_t ra[32], rb[32];
                float mxa, mxb;
                {
                    tmem_ld32(tS, ra);
                    tc_wait_ld();
                    tmem_ld32(tS + 32, rb);
                    if constexpr (RAG) mask_chunk(ra, 0);
                    mxa = max32(ra);
                    tc_wait_ld();
                    tmem_ld32(tS + 64, ra);
                    if constexpr (RAG) mask_chunk(rb, 1);
                    mxa = fmaxf(mxa, max32(rb));
                    tc_wait_ld();
                    tmem_ld32(tS + 96, rb);
                    if constexpr (RAG) mask_chunk(ra, 2);
                    mxb = max32(ra);
                    tc_wait_ld();
                    tmem_ld32(tS, ra);                       // first chunk of pass 2
                    if constexpr (RAG) mask_chunk(rb, 3);
                    mxb = fmaxf(mxb, max32(rb));
                }
                const float mt = fmaxf(mxa * sl2a, mxb * sl2b);   // sl2 > 0; va > 0
                // m_ref hand-off: the other parity published the reference it used for pair j - 1
                // (and under which O now stands) after ITS max pass.
                if (j > 0) {
                    named_bar_sync(NB_HAND + (sm ^ 1) * 4 + wq, 64);
                    const float m_in = xm[row];
                    if (m_in != m_ref) {             // also covers m_ref = -inf (this warp's first pair)
                        const float a = ex2(m_ref - m_in);
                        l0 *= a;
                        l1 *= a;
                        m_ref = m_in;
                    }
                }
                const bool grow = __any_sync(0xffffffffu, mt > m_ref + C::RESCALE_THRESHOLD);
                float alpha = 1.f;
                if (grow) {
                    const float m_new = fmaxf(m_ref, mt);
                    alpha = ex2(m_ref - m_new);      // m_ref = -inf (first pair of the item) -> 0
                    l0 *= alpha;
                    l1 *= alpha;
                    m_ref = m_new;
                }
                if (j + 1 < it.np) {                 // publish before the (rare) rescale: P V of pair j + 1
                    xm[row] = m_ref;                 // cannot be issued before this pair's P is ready
                    named_bar_arrive(NB_HAND + sm * 4 + wq, 64);
                }
                if (grow && j > 0) {
                    // O holds pairs 0..j-1 under the old reference; wait for P V of pair j-1.
                    // (S_FULL of pair g implies P V of pair g-3 is complete, so the barrier of
                    // buffer (g-1) % 3 is at most one phase behind: the parity wait is exact.)
                    mbar_wait(bar(C::B_PV_DONE + (g - 1) % SBUFS), ((g - 1) / SBUFS) & 1);
                    tc_fence_after();
#pragma unroll 1
                    for (int c = 0; c < 4; ++c) {
                        tc_wait_ld();
                        tmem_ld32(tOs + c * 32, rb);
                        tc_wait_ld();
#pragma unroll
                        for (int k = 0; k < 32; ++k) rb[k] = __float_as_uint(__uint_as_float(rb[k]) * alpha);
                        tmem_st32(tOs + c * 32, rb);
                    }
                }
                {
                    // P = exp2(s * sl2 - m_ref + shift).  Element pairs go through packed FFMA2; the
                    // pairs whose bit is set in POLY_MASK (index mod 8) take the polynomial exp2 on
                    // the FMA pipe, the rest the MUFU.
                    // kHalf: a row that has kept nothing so far has m_ref = -inf and only -inf scores
                    const float negm = (kHalf && m_ref == -INFINITY) ? 0.f : -m_ref;
                    const float2 negm_2 = make_float2(negm, negm);
                    const float2 sl2a_2 = make_float2(sl2a, sl2a), sl2b_2 = make_float2(sl2b, sl2b);
                    float2 lacc = make_float2(l0, l1);
                    // 32 scores -> 16 (bf16) / 8 (e4m3) TMEM columns of P at chunk position c
                    auto exp_chunk = [&](const uint32_t (&r)[32], int c) {
                        const float2 sl2_2 = (c >> 1) ? sl2b_2 : sl2a_2;
                        auto exp_pair = [&](int q) -> float2 {     // q: element pair index 0..15
                            const float2 x = ffma2(make_float2(__uint_as_float(r[2 * q]), __uint_as_float(r[2 * q + 1])),
                                                   sl2_2, negm_2);
                            return make_float2(ex2(x.x), ex2(x.y));   // all on the MUFU: a polynomial share never paid here
                        };
                        {
                            uint32_t pk[16];
#pragma unroll
                            for (int k = 0; k < 16; ++k) {
                                const float2 pp = exp_pair(k);
                                lacc = fadd2(lacc, pp);
                                pk[k] = kF16 ? pack_f16x2(pp.x, pp.y) : pack_bf16x2(pp.x, pp.y);
                            }
                            tmem_st16(tS + c * 16, pk);      // P: bf16 pairs over the first 64 S columns
                        }
                    };
                    tc_wait_ld();
                    tmem_ld32(tS + 32, rb);
                    if constexpr (RAG) mask_chunk(ra, 0);
                    exp_chunk(ra, 0);
                    tc_wait_ld();
                    tmem_ld32(tS + 64, ra);
                    if constexpr (RAG) mask_chunk(rb, 1);
                    exp_chunk(rb, 1);
                    tc_wait_ld();
                    tmem_ld32(tS + 96, rb);
                    if constexpr (RAG) mask_chunk(ra, 2);
                    exp_chunk(ra, 2);
                    tc_wait_ld();
                    if constexpr (RAG) mask_chunk(rb, 3);
                    exp_chunk(rb, 3);
                    l0 = lacc.x;
                    l1 = lacc.y;
                }
                };
                // kHalf: the rows of this warp keep neither tile of the pair (the other half of the block
                // does): no pass over S, P = 0, the reference is handed on unchanged
                auto skip_body = [&]() {
                    if (j > 0) {
                        named_bar_sync(NB_HAND + (sm ^ 1) * 4 + wq, 64);
                        const float m_in = xm[row];
                        if (m_in != m_ref) {
                            const float a = ex2(m_ref - m_in);
                            l0 *= a;
                            l1 *= a;
                            m_ref = m_in;
                        }
                    }
                    if (j + 1 < it.np) {
                        xm[row] = m_ref;
                        named_bar_arrive(NB_HAND + sm * 4 + wq, 64);
                    }
                    uint32_t z[16];
#pragma unroll
                    for (int k = 0; k < 16; ++k) z[k] = 0u;
#pragma unroll
                    for (int c = 0; c < 4; ++c) tmem_st16(tS + c * 16, z);
                };
                if (kHalf && va == 0 && vb == 0) skip_body();
                else if (ragged) pair_body(BoolTag<true>{});
                else pair_body(BoolTag<false>{});
                tc_wait_st();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(C::B_P_READY + sb));
            }
            g0 += it.np;
            // ---------------- epilogue: add the partial row sums, normalise, convert, store ------
            // Warp (sm, wq) finalises O columns [64 sm, 64 sm + 64) of its 32 rows.  The parity that
            // handled the last pair holds the final m_ref; the other one may be one update behind.
            const float l_mine = l0 + l1;
            xe[(sm * 2 + 0) * 128 + row] = m_ref;
            xe[(sm * 2 + 1) * 128 + row] = l_mine;
            if (lane == 0 && wq == 0) tma_store_wait_read();   // staging slab sm is free again
            named_bar_sync(NB_PAIR + wq, 64);
            const float m_oth = xe[((sm ^ 1) * 2 + 0) * 128 + row];
            const float l_oth = xe[((sm ^ 1) * 2 + 1) * 128 + row];
            named_bar_sync(NB_PAIR + wq, 64);                  // both have read: the slots may be rewritten
            const float m_all = fmaxf(m_ref, m_oth);
            // a parity without pairs has m = -inf, l = 0
            const float a_mine = (m_ref == -INFINITY) ? 0.f : ex2(m_ref - m_all);
            const float a_oth = (m_oth == -INFINITY) ? 0.f : ex2(m_oth - m_all);
            const float L = l_mine * a_mine + l_oth * a_oth;
            const float inv = (L > 0.f) ? 1.f / L : 0.f;
            // optional row log-sum-exp (natural log of sum_j exp(scale * q . k_j) over the retained
            // keys; -inf for an empty row): what a later block-mass pass needs
            if (p.lse != nullptr && sm == 0 && it.qb * BQ + row < p.N)
                p.lse[(static_cast<int64_t>(it.b) * p.H + it.h) * p.N + it.qb * BQ + row] =
                    (L > 0.f) ? (m_all + lg2(L)) * 0.6931471805599453f : -INFINITY;
            named_bar_sync(NB_HALF + sm, 128);                 // staging free for the whole warpgroup
            if (it.nt > 0) {
                mbar_wait(bar(C::B_ITEM_DONE), icnt & 1);      // every P V of the item has completed
                tc_fence_after();
            }
            const uint32_t srow = sO + sm * 16384 + row * 128;
            const uint32_t tO = tOs + sm * 64;
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
                    const float4 w = make_float4(inv, inv, inv, inv);
                    float x0 = 0.f, x1 = 0.f, x2 = 0.f, x3 = 0.f;
                    if (it.nt > 0) {
                        x0 = __uint_as_float(o[4 * k4]) * w.x;     x1 = __uint_as_float(o[4 * k4 + 1]) * w.y;
                        x2 = __uint_as_float(o[4 * k4 + 2]) * w.z; x3 = __uint_as_float(o[4 * k4 + 3]) * w.w;
                    }
                    pk[2 * k4] = kF16 ? pack_f16x2(x0, x1) : pack_bf16x2(x0, x1);
                    pk[2 * k4 + 1] = kF16 ? pack_f16x2(x2, x3) : pack_bf16x2(x2, x3);
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
                ++icnt;
            }
            fence_proxy_async_smem();
            named_bar_sync(NB_HALF + sm, 128);
            if (lane == 0 && wq == 0) {
                tma_store_4d(&tmO, sO + sm * 16384, sm * 64, it.qb * BQ, it.h, it.b);
                tma_store_commit();
            }
        }
        if (lane == 0 && wq == 0) tma_store_wait_all();
    }
    tc_fence_before();
    __syncthreads();
    if (warp == MMA_WARP) tmem_dealloc(tmem, TM_COLS);
    if (threadIdx.x == 0) item_ticket_release(p.ticket_slot);
}

}  // namespace

template <bool kF16, bool kBeta, bool kHalf>
static cudaError_t launch_one(const CUtensorMap& tmQ, const CUtensorMap& tmK, const CUtensorMap& tmV,
                              const CUtensorMap& tmO, const AttnParams& p, cudaStream_t stream) {
    constexpr uint32_t smem = Cfg::SMEM_BYTES;
    cudaError_t e = cudaFuncSetAttribute(attn_fwd_kernel<kF16, kBeta, kHalf>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    int dev = 0, sms = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    const int n_items = p.B * p.H * p.nq;
    const int grid = n_items < sms ? n_items : sms;
    AttnParams pl = p;
    pl.ticket_slot = next_ticket_slot();
    attn_fwd_kernel<kF16, kBeta, kHalf><<<grid, NUM_THREADS, smem, stream>>>(tmQ, tmK, tmV, tmO, pl);
    count_launch(1);
    return cudaGetLastError();
}

cudaError_t launch_attn_fwd(const CUtensorMap& tmQ, const CUtensorMap& tmK, const CUtensorMap& tmV,
                            const CUtensorMap& tmO, const AttnParams& p, chorus_dtype dtype,
                            cudaStream_t stream) {
    const bool beta = p.n_first > 0 && p.beta != 1.f;
    auto go = [&](auto f16) -> cudaError_t {
        constexpr bool F16 = decltype(f16)::value;
        if (beta && p.half_flags) return launch_one<F16, true, true>(tmQ, tmK, tmV, tmO, p, stream);
        if (beta) return launch_one<F16, true, false>(tmQ, tmK, tmV, tmO, p, stream);
        if (p.half_flags) return launch_one<F16, false, true>(tmQ, tmK, tmV, tmO, p, stream);
        return launch_one<F16, false, false>(tmQ, tmK, tmV, tmO, p, stream);
    };
    if (dtype == CHORUS_BF16) return go(BoolTag<false>{});
    if (dtype == CHORUS_FP8_E4M3) return launch_attn_fwd_fp8(tmQ, tmK, tmV, tmO, p, stream);   // attn_fwd_fp8.cu
    if (dtype == CHORUS_FP16) return go(BoolTag<true>{});
    return cudaErrorNotSupported;
}

}  // namespace chorus
