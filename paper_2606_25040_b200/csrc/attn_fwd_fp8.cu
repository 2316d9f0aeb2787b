// attn_fwd_fp8.cu — chorus_block_sparse_attn_fwd for dtype CHORUS_FP8_E4M3 on sm_100a (row a-3; PAPER.md:L97
// "FP8 quantization ... low-precision matrix multiplication with high-precision accumulation", the paper's
// default backend; R10-R12).
//
// Same persistent, warp-specialised structure as the 16-bit kernel (attn_fwd.cu): one CTA of 384 threads per SM,
// a work item is one (batch, head, 128-row query block), its kept 64-key tiles are taken two at a time ("a pair",
// any two kept tiles) so that QK^T runs at N = 128.  What differs is everything around the softmax, which is what
// bounds the FP8 kernel (its MMAs are half as long):
//   * S is read from tensor memory ONCE: a thread takes the 128 fp32 scores of its query row into registers, frees
//     the S buffer at once (two S buffers suffice and QK^T of the next pairs never waits for a P V), takes the row
//     maximum, joins the m_ref hand-off and exponentiates from registers.
//   * P (e4m3) has its own three 32-column buffers in tensor memory, so a pair's S, P and the O accumulator never
//     alias and the MMA warp issues P V two pairs behind QK^T.
//   * The softmax denominator is not summed by the softmax warps at all: V's shared-memory tile is extended by a
//     constant slab of ones (16 extra B columns reached through the descriptor's leading-dimension offset), so
//     P V runs at N = 144 and O[:, 128] accumulates sum_j P_ij in fp32 on the tensor cores, of exactly the
//     e4m3-rounded weights that multiply V (so a row dominated by one key does not inherit the 2^-4 rounding of its
//     weight), rescaled together with O on the lazy-rescale path.  This removes the e4m3 -> f16 unpack, the HADD2
//     accumulation and the (m, l) exchange between the two softmax parities of the epilogue.
//   warp 8        TMA producer: Q tile once per item, K / V pairs into two rings of four 16 KB stages; the pair's
//                 col_idx entries and K scales into a small ring for the softmax warps
//   warp 9        issues S = Q K^T (kind::f8f6f4, M 128, N 128, K 128) into S[g % 2], as soon as the buffer is free
//   warp 10       issues O += P V (P the TMEM A operand, V an MN-major B operand, N = 144 with the ones columns).
//                 Two issuing warps on two schedulers: either one's ~80 instructions per pair share a scheduler
//                 with two softmax warps, and the slowest of the four lane quarters sets the pace of a pair
//   warps 0-3     softmax of the even pairs of an item; warps 4-7 of the odd pairs (one query row per thread)
// TMEM (512 columns): O 0..143 (128 channels + 16 copies of the row sum), S0 160.., S1 288.., P0 416, P1 448,
// P2 480.  O is rescaled lazily: only when a row maximum exceeds the reference by more than 2^3.
#include <cuda_bf16.h>

#include "attn_common.cuh"

namespace chorus {
namespace {

using namespace ptx;
using namespace attn;

constexpr int KSTAGES = 4, VSTAGES = 4, SBUFS = 2, PBUFS = 3;
// What the softmax warps need to know about a pair - its two col_idx entries and the K scales of its two key blocks -
// is fetched ONCE, by the producer warp (which has the entries anyway), and handed over in shared memory: entry
// g % PAIR_RING, written before the pair's K tiles are requested.  The producer is at most KSTAGES pairs ahead of the
// Q K^T issue and that at most SBUFS pairs ahead of the last softmax warp's read of S, which follows its read of the
// entry: 8 > 4 + 2 entries are never overwritten early.
constexpr uint32_t PAIR_RING = 8;
constexpr uint32_t TILE = 16384;        // one pair stage: [128 keys][128 B] = two 64-key tiles of 128 e4m3 channels
constexpr uint32_t HALF = 8192;         // the second tile of a pair
// shared memory map (bytes from a 1024-aligned base).  The ones slab lies ABOVE every V stage: the B descriptor of
// a P V step reaches it as the second 128-byte column block of its operand (leading-dimension byte offset).
constexpr uint32_t SQ_OFF = 0, SK_OFF = TILE, SV_OFF = SK_OFF + KSTAGES * TILE, ONES_OFF = SV_OFF + VSTAGES * TILE,
                   ONES_BYTES = 4096,   // [32 keys][128 B] of e4m3 1.0: one K = 32 MMA step's worth
                   SO_OFF = ONES_OFF + ONES_BYTES, XCH_OFF = SO_OFF + 32768, PR_OFF = XCH_OFF + 512,
                   BAR_OFF = PR_OFF + PAIR_RING * 16,
                   SMEM_BYTES = BAR_OFF + 384;
static_assert(SMEM_BYTES <= 232448, "exceeds the 227 KB per-CTA shared memory of sm_100");
// mbarrier slots
constexpr uint32_t B_Q_FULL = 0, B_Q_EMPTY = 1, B_K_FULL = 2, B_K_EMPTY = B_K_FULL + KSTAGES,
                   B_V_FULL = B_K_EMPTY + KSTAGES, B_V_EMPTY = B_V_FULL + VSTAGES, B_S_FULL = B_V_EMPTY + VSTAGES,
                   B_S_FREE = B_S_FULL + SBUFS, B_P_READY = B_S_FREE + SBUFS, B_PV_DONE = B_P_READY + PBUFS,
                   B_ITEM_DONE = B_PV_DONE + PBUFS, B_O_FREE = B_ITEM_DONE + 1, B_IT_FULL = B_O_FREE + 1,
                   B_IT_EMPTY = B_IT_FULL + ITEM_RING, B_COUNT = B_IT_EMPTY + ITEM_RING;
static_assert(B_COUNT * 8 + 8 + 4 * ITEM_RING <= 384, "barrier area too small");
// tensor-memory map (columns)
constexpr uint32_t TM_O = 0, TM_L = 128, TM_S = 160, TM_P = 416, TM_COLS = 512;
constexpr uint32_t PV_N = 144;          // 128 channels + 16 ones columns (M = 128 needs N % 16 == 0)
// P = exp2(x - m_ref + 5): e4m3 (max 448, smallest normal 2^-6) keeps probabilities down to 2^-11 of the row
// maximum as normal numbers while P <= 2^8 holds under the lazy-rescale threshold of 2^3.
constexpr float P_SHIFT = 5.0f, RESCALE_THRESHOLD = 3.0f;
// The exponentials of a pair are split between two units, by element pair (index mod 8):
//   LIN_MASK   every other pair: the piecewise-linear 2^x read off the score's own bits on the ALU / FMA pipes.
//              t = x + 1.5 * 2^15 leaves round(x * 2^8) in the low mantissa bits of t, and (bits(t) << 15) + LIN_K is
//              the float 2^floor(x) * (1 + frac(x) - d): one FMNMX (clamp at 2^-126) and one integer shift-add per
//              element after the FFMA2 that every path needs.  d = 0.0564 makes the error -3.8 % .. +2.1 % with
//              mean 0 over frac(x), next to the +-3.1 % of the e4m3 rounding that follows; the row sums are taken by
//              the tensor cores from the same P, so numerator and denominator stay consistent and unbiased.
//   the rest   MUFU.EX2, one warp instruction per 8 cycles and scheduler: the unit that bounded the kernel
// (4 of 8 is the measured optimum: DESIGN.md section 6.5)
constexpr uint32_t LIN_MASK = 0x55u;
constexpr float LIN_C = 49152.0f;                                  // 1.5 * 2^15: ulp 2^-8
constexpr float LIN_LO = LIN_C - 126.0f;                           // 2^-126: rounds to the e4m3 code 0
constexpr int LIN_K = static_cast<int>((127u << 23) - 473118u - (0x47400000u << 15));
// named barriers: 0 = __syncthreads, 5..6 = parity warpgroup (epilogue staging), 7..14 = m_ref hand-off published
// by parity 0 (7..10) / parity 1 (11..14) of lane quarter wq
constexpr uint32_t NB_HALF = 5, NB_HAND = 7;

// four floats -> four e4m3 codes, a in the lowest byte (RNE, saturating)
__device__ __forceinline__ uint32_t pack4(float a, float b, float c, float d) { return pack_e4m3x4(a, b, c, d); }

template <bool kBeta, bool kHalf>
__global__ void __launch_bounds__(NUM_THREADS, 1)
attn_fwd_fp8_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                    const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmO,
                    const AttnParams p) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t base = smem_u32(smem_raw);
    if (base & 1023u) __trap();
    uint8_t* gbase = smem_raw;
    const uint32_t sQ = base + SQ_OFF, sK = base + SK_OFF, sV = base + SV_OFF, sOnes = base + ONES_OFF, sO = base + SO_OFF;
    const uint32_t bars = base + BAR_OFF;
    auto bar = [&](uint32_t i) { return bars + 8u * i; };
    volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(gbase + BAR_OFF + 8 * B_COUNT);
    volatile float* xm = reinterpret_cast<volatile float*>(gbase + XCH_OFF);   // [128] m_ref hand-off
    const uint32_t pair_ring = base + PR_OFF;                                   // [PAIR_RING] {entry a, entry b, k scale a, b}

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_items = p.B * p.H * p.nq;
    const ItemRing ring{bar(B_IT_FULL), bar(B_IT_EMPTY), reinterpret_cast<volatile int*>(gbase + BAR_OFF + 8 * B_COUNT + 8)};

    if (threadIdx.x == 0) {
        mbar_init(bar(B_Q_FULL), 1);
        mbar_init(bar(B_Q_EMPTY), 1);
        for (int i = 0; i < KSTAGES; ++i) { mbar_init(bar(B_K_FULL + i), 1); mbar_init(bar(B_K_EMPTY + i), 1); }
        for (int i = 0; i < VSTAGES; ++i) { mbar_init(bar(B_V_FULL + i), 1); mbar_init(bar(B_V_EMPTY + i), 1); }
        for (int i = 0; i < SBUFS; ++i) { mbar_init(bar(B_S_FULL + i), 1); mbar_init(bar(B_S_FREE + i), 4); }
        for (int i = 0; i < PBUFS; ++i) { mbar_init(bar(B_P_READY + i), 4); mbar_init(bar(B_PV_DONE + i), 1); }
        mbar_init(bar(B_ITEM_DONE), 1);
        mbar_init(bar(B_O_FREE), 8);
        for (int i = 0; i < ITEM_RING; ++i) { mbar_init(bar(B_IT_FULL + i), 1); mbar_init(bar(B_IT_EMPTY + i), 10); }   // two MMA warps + 8 softmax warps
        fence_mbar_init();
    }
    // the ones slab: e4m3 1.0 = 0x38 in every byte (constant, so the 128-byte swizzle does not matter)
    for (uint32_t i = threadIdx.x; i < ONES_BYTES / 16; i += NUM_THREADS)
        reinterpret_cast<uint4*>(gbase + ONES_OFF)[i] = make_uint4(0x38383838u, 0x38383838u, 0x38383838u, 0x38383838u);
    fence_proxy_async_smem();            // generic-proxy stores -> visible to the tensor core's reads
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
        // Both roles run with the WHOLE warp converged; one elected lane issues the TMA / tcgen05 instructions and
        // everything an issue needs is made warp-uniform first (see attn_fwd.cu).
        if (warp == PRODUCER_WARP) {
            uint32_t g = 0, icnt = 0;   // pairs and non-empty items issued so far
            for (uint32_t kit = 0;; ++kit) {
                const int idx = item_draw(ring, kit, n_items, p.ticket_slot);
                if (idx < 0) break;
                const Item it = get_item_uniform(p, idx);
                if (it.nt == 0) continue;   // empty rows touch no barrier
                mbar_wait(bar(B_Q_EMPTY), (icnt & 1) ^ 1);
                if (elect_one()) {
                    mbar_arrive_expect_tx(bar(B_Q_FULL), TILE);
                    tma_load_4d(sQ, &tmQ, bar(B_Q_FULL), 0, it.qb * BQ, it.h, it.b);
                }
                __syncwarp();
                const float* ksc = p.k_scale + (static_cast<int64_t>(it.b) * p.H + it.h) * ((p.N + 127) >> 7);
                // the key-block indices of 16 pairs are fetched with one coalesced load, their K scales with a second
                for (int j0 = 0; j0 < it.np; j0 += 16) {
                    const int t = 2 * j0 + lane;
                    const int raw = (t < it.nt) ? ld_col(p, it.r0 + t) : 0;     // kHalf: with the per-half flags
                    const int mine = kHalf ? (raw & 0x3fffffff) : raw;
                    const float mysc = (t < it.nt) ? __ldg(ksc + (mine >> 1)) : 0.f;
                    const int jn = min(16, it.np - j0);
                    for (int jl = 0; jl < jn; ++jl, ++g) {
                        const int ntile = (2 * (j0 + jl) + 1 < it.nt) ? 2 : 1;
                        const int kb0 = __shfl_sync(0xffffffffu, mine, 2 * jl);
                        const int kb1 = __shfl_sync(0xffffffffu, mine, 2 * jl + 1);
                        const int raw0 = kHalf ? __shfl_sync(0xffffffffu, raw, 2 * jl) : kb0;
                        const int raw1 = kHalf ? __shfl_sync(0xffffffffu, raw, 2 * jl + 1) : kb1;
                        const float sc0 = __shfl_sync(0xffffffffu, mysc, 2 * jl);
                        const float sc1 = __shfl_sync(0xffffffffu, mysc, 2 * jl + 1);
                        {
                            const uint32_t st = g % KSTAGES, ph = (g / KSTAGES) & 1;
                            mbar_wait(bar(B_K_EMPTY + st), ph ^ 1);
                            if (elect_one()) {
                                asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(pair_ring + (g % PAIR_RING) * 16),
                                             "r"(raw0), "r"(raw1), "r"(__float_as_int(sc0)), "r"(__float_as_int(sc1)) : "memory");
                                mbar_arrive_expect_tx(bar(B_K_FULL + st), ntile * HALF);
                                const uint32_t dst = sK + st * TILE;
                                tma_load_4d(dst, &tmK, bar(B_K_FULL + st), 0, kb0 * BK, it.h, it.b);
                                if (ntile == 2) tma_load_4d(dst + HALF, &tmK, bar(B_K_FULL + st), 0, kb1 * BK, it.h, it.b);
                            }
                            __syncwarp();
                        }
                        {
                            const uint32_t st = g % VSTAGES, ph = (g / VSTAGES) & 1;
                            mbar_wait(bar(B_V_EMPTY + st), ph ^ 1);
                            if (elect_one()) {
                                mbar_arrive_expect_tx(bar(B_V_FULL + st), ntile * HALF);
                                const uint32_t dst = sV + st * TILE;
                                tma_load_4d(dst, &tmV, bar(B_V_FULL + st), 0, kb0 * BK, it.h, it.b);
                                if (ntile == 2) tma_load_4d(dst + HALF, &tmV, bar(B_V_FULL + st), 0, kb1 * BK, it.h, it.b);
                            }
                            __syncwarp();
                        }
                    }
                }
                ++icnt;
            }
        } else if (warp == MMA_WARP) {
            // kind::f8f6f4, format 0 = e4m3.  P V: B (= V and the ones slab) is MN-major, N = 144.
            constexpr uint32_t IDESC_S128 = make_idesc(0, 0, 128, 128, 0, 0);
            constexpr uint32_t IDESC_S64 = make_idesc(0, 0, 128, 64, 0, 0);
            const uint64_t dQ = smem_desc_sw128(sQ, 16, 1024);
            const uint64_t dK = smem_desc_sw128(sK, 16, 1024);
            uint32_t g0 = 0, icnt = 0;      // pairs before this item, non-empty items so far
            for (uint32_t kit = 0;; ++kit) {
                const int idx = item_take(ring, kit);
                if (idx < 0) break;
                const Item it = get_item_uniform(p, idx);
                if (it.nt == 0) continue;
                mbar_wait(bar(B_Q_FULL), icnt & 1);
                for (int jj = 0; jj < it.np; ++jj) {
                    {   // S[g % 2] = Q K^T of pair jj
                        const uint32_t g = g0 + jj;
                        const uint32_t st = g % KSTAGES, ph = (g / KSTAGES) & 1, sb = g % SBUFS;
                        const bool two = 2 * jj + 1 < it.nt;
                        mbar_wait(bar(B_K_FULL + st), ph);
                        mbar_wait(bar(B_S_FREE + sb), ((g / SBUFS) & 1) ^ 1);   // pair g - 2 is in registers
                        tc_fence_after();
                        if (elect_one()) {
                            const uint32_t tS = tmem + TM_S + sb * 128;
                            const uint32_t idesc = two ? IDESC_S128 : IDESC_S64;
                            const uint64_t dKs = dK + ((st * TILE) >> 4);
#pragma unroll
                            for (int ks = 0; ks < 4; ++ks)       // 32 e4m3 channels = 32 B per step
                                mma_f8_ss(tS, dQ + ((ks * 32) >> 4), dKs + ((ks * 32) >> 4), idesc, ks > 0);
                            tc_commit(bar(B_K_EMPTY + st));
                            tc_commit(bar(B_S_FULL + sb));
                            if (jj == it.np - 1) tc_commit(bar(B_Q_EMPTY));
                        }
                        __syncwarp();
                    }
                }
                g0 += it.np;
                ++icnt;
            }
        } else if (warp == MMA_WARP + 1) {
            constexpr uint32_t IDESC_PV = make_idesc(0, 0, 128, PV_N, 0, 1);
            uint32_t g0 = 0, icnt = 0;
            for (uint32_t kit = 0;; ++kit) {
                const int idx = item_take(ring, kit);
                if (idx < 0) break;
                const Item it = get_item_uniform(p, idx);
                if (it.nt == 0) continue;
                for (int jp = 0; jp < it.np; ++jp) {
                    {      // O += P V of pair jp
                        const uint32_t g = g0 + jp;
                        const uint32_t st = g % VSTAGES, ph = (g / VSTAGES) & 1, pb = g % PBUFS;
                        const bool two = 2 * jp + 1 < it.nt;
                        mbar_wait(bar(B_P_READY + pb), (g / PBUFS) & 1);
                        mbar_wait(bar(B_V_FULL + st), ph);
                        if (jp == 0) mbar_wait(bar(B_O_FREE), (icnt & 1) ^ 1);
                        tc_fence_after();
                        if (elect_one()) {
                            const uint32_t tP = tmem + TM_P + pb * 32, tO = tmem + TM_O;
                            const uint32_t vst = sV + st * TILE;
                            const int steps = two ? 4 : 2;           // 32 keys x 128 B per step
                            // columns 128..143 of B come from the ones slab: leading-dimension offset = its distance.
                            // A step further down the tile adds 4096 B to the start address and takes them off the
                            // offset: one 64-bit constant on the descriptor (both fields stay inside their bits).
                            const uint64_t dV0 = smem_desc_sw128(vst, sOnes - vst, 1024);
                            constexpr uint64_t DV_STEP = static_cast<uint64_t>(256) - (static_cast<uint64_t>(256) << 16);
#pragma unroll
                            for (int ks = 0; ks < 4; ++ks)
                                if (ks < steps)
                                    mma_f8_ts(tO, tP + ks * 8, dV0 + static_cast<uint64_t>(ks) * DV_STEP, IDESC_PV, (jp > 0) || (ks > 0));
                            tc_commit(bar(B_V_EMPTY + st));
                            tc_commit(bar(B_PV_DONE + pb));
                            if (jp == it.np - 1) tc_commit(bar(B_ITEM_DONE));
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
        const uint32_t tOs = tlane + TM_O;       // the O accumulator (128 channels, then the row sum)
        const int nsb = (p.N + 127) >> 7;        // Q/K scale blocks of 128 tokens
        uint32_t g0 = 0;                         // pairs of all previous items
        uint32_t icnt = 0;                       // non-empty items so far
        for (uint32_t kit = 0;; ++kit) {
            const int idx = item_take(ring, kit);
            if (idx < 0) break;
            const Item it = get_item(p, idx);
            float m_ref = -INFINITY;
            // scores are (q8 . k8) * s_q[qb] * s_k[kb / 2] (R10); the per-tile factor is folded into the
            // exp2 FMA constant.  The pair's entries and K scales come from the producer warp (pair ring).
            const int64_t sbase = (static_cast<int64_t>(it.b) * p.H + it.h) * nsb;
            const float qsl2 = p.scale_log2 * __ldg(p.q_scale + sbase + it.qb);
            for (int j = sm; j < it.np; j += 2) {
                const uint32_t g = g0 + j, sb = g % SBUFS, pb = g % PBUFS;
                const uint32_t tS = tlane + TM_S + sb * 128, tP = tlane + TM_P + pb * 32;
                int va = BK, vb = BK;            // valid keys in the two tiles of the pair
                // S of the pair is complete; its ring entry was written before its K tiles were even requested
                mbar_wait(bar(B_S_FULL + sb), (g / SBUFS) & 1);
                tc_fence_after();
                int kba, kbb;
                float ska, skb;
                asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(kba), "=r"(kbb), "=f"(ska), "=f"(skb)
                             : "r"(pair_ring + (g % PAIR_RING) * 16) : "memory");
                uint32_t skip_a = 0u, skip_b = 0u;   // kHalf: this warp's rows do not keep tile a / b
                if constexpr (kHalf) {
                    const int hb = 30 + (wq >> 1);
                    skip_a = (static_cast<uint32_t>(kba) >> hb) & 1u;
                    skip_b = (static_cast<uint32_t>(kbb) >> hb) & 1u;
                    kba &= 0x3fffffff;
                    kbb &= 0x3fffffff;
                }
                float sl2a = qsl2 * ska;
                float sl2b = qsl2 * skb;
                // kBeta: a tile inside the first frame takes beta in its scale factor; the one tile that straddles
                // n_first takes it per column (fa / fb leading columns) in the masked body
                int fa = 0, fb = 0;
                if constexpr (kBeta) {
                    fa = min(BK, max(0, p.n_first - kba * BK));
                    fb = (2 * j + 1 < it.nt) ? min(BK, max(0, p.n_first - kbb * BK)) : 0;
                    if (fa == BK) { sl2a *= p.beta; fa = 0; }
                    if (fb == BK) { sl2b *= p.beta; fb = 0; }
                }
                if (j == it.np - 1) {            // only the last pair can be odd or hold the ragged key block
                    va = min(BK, p.N - kba * BK);
                    vb = (2 * j + 1 < it.nt) ? min(BK, p.N - kbb * BK) : 0;
                }
                if constexpr (kHalf) {           // a tile the rows of this warp do not keep: all -inf
                    if (skip_a) va = 0;
                    if (skip_b) vb = 0;
                }
                // ---- the 128 scores of the row into registers; the S buffer is free again at once ----
                uint32_t s[128];
                tmem_ld32(tS, reinterpret_cast<uint32_t(&)[32]>(s[0]));
                tmem_ld32(tS + 32, reinterpret_cast<uint32_t(&)[32]>(s[32]));
                tmem_ld32(tS + 64, reinterpret_cast<uint32_t(&)[32]>(s[64]));
                tmem_ld32(tS + 96, reinterpret_cast<uint32_t(&)[32]>(s[96]));
                tc_wait_ld();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(B_S_FREE + sb));
                const bool ragged = (va < BK) || (vb < BK) || (fa | fb) != 0;   // warp-uniform and rare
                if (ragged) {
#pragma unroll
                    for (int k = 0; k < 64; ++k) {
                        if (k >= va) s[k] = 0xff800000u;            // -inf
                        if (k >= vb) s[64 + k] = 0xff800000u;
                    }
                    if constexpr (kBeta) {
#pragma unroll
                        for (int k = 0; k < 64; ++k) {
                            if (k < fa) s[k] = __float_as_uint(__uint_as_float(s[k]) * p.beta);
                            if (k < fb) s[64 + k] = __float_as_uint(__uint_as_float(s[64 + k]) * p.beta);
                        }
                    }
                }
                const bool none = kHalf && va == 0 && vb == 0;      // the rows of this warp keep neither tile
                float mt = -INFINITY;
                if (!none) {
                    const float mxa = max64(s), mxb = max64(s + 64);
                    // sl2 > 0 (scale and the block scales are positive); a tile without valid keys has max -inf
                    mt = fmaxf(mxa * sl2a, vb > 0 ? mxb * sl2b : -INFINITY);
                }
                // m_ref hand-off: the other parity published the reference it used for pair j - 1 (and under which
                // O now stands) after ITS max pass.
                if (j > 0) {
                    named_bar_sync(NB_HAND + (sm ^ 1) * 4 + wq, 64);
                    m_ref = xm[row];
                }
                const bool grow = __any_sync(0xffffffffu, mt > m_ref + RESCALE_THRESHOLD);
                float alpha = 1.f;
                if (grow) {
                    const float m_new = fmaxf(m_ref, mt);
                    alpha = ex2(m_ref - m_new);      // m_ref = -inf (nothing kept so far) -> 0
                    if (m_new == -INFINITY) alpha = 1.f;
                    m_ref = m_new;
                }
                if (j + 1 < it.np) {                 // publish before the (rare) rescale: P V of pair j + 1
                    xm[row] = m_ref;                 // cannot be issued before this pair's P is ready
                    named_bar_arrive(NB_HAND + sm * 4 + wq, 64);
                }
                if (grow && j > 0) {
                    // O (and its row-sum column) hold pairs 0..j-1 under the old reference: wait for P V of pair
                    // j - 1.  P V of pair g + 2 cannot complete before this pair's P is ready, so the barrier of
                    // buffer (g - 1) % 3 is at most one phase ahead and the parity wait is exact.
                    mbar_wait(bar(B_PV_DONE + (g - 1) % PBUFS), ((g - 1) / PBUFS) & 1);
                    tc_fence_after();
                    uint32_t o[32];
#pragma unroll 1
                    for (int c = 0; c < 4; ++c) {
                        tmem_ld32(tOs + c * 32, o);
                        tc_wait_ld();
#pragma unroll
                        for (int k = 0; k < 32; ++k) o[k] = __float_as_uint(__uint_as_float(o[k]) * alpha);
                        tmem_st32(tOs + c * 32, o);
                    }
                    uint32_t l1[1];
                    tmem_ld1(tOs + TM_L, l1);
                    tc_wait_ld();
                    l1[0] = __float_as_uint(__uint_as_float(l1[0]) * alpha);
                    tmem_st1(tOs + TM_L, l1);
                }
                // ---- P = exp2(s * sl2 - m_ref + shift) -> e4m3, 4 codes per register -----------------------------
                uint32_t pk[32];
                if (none) {
#pragma unroll
                    for (int k = 0; k < 32; ++k) pk[k] = 0u;
                } else {
                    // a row that has kept nothing so far has m_ref = -inf and only -inf scores: constant 0, not NaN
                    const float negm = (kHalf && m_ref == -INFINITY) ? 0.f : P_SHIFT - m_ref;
                    const float2 negm_2 = make_float2(negm, negm);
                    const float2 negmc_2 = make_float2(negm + LIN_C, negm + LIN_C);
                    const float2 sl2a_2 = make_float2(sl2a, sl2a), sl2b_2 = make_float2(sl2b, sl2b);
                    auto exp_pair = [&](int q) -> float2 {     // q: element pair index 0..63
                        const float2 sv = make_float2(__uint_as_float(s[2 * q]), __uint_as_float(s[2 * q + 1]));
                        if ((LIN_MASK >> (q & 7)) & 1u) {
                            const float2 t = ffma2(sv, q < 32 ? sl2a_2 : sl2b_2, negmc_2);
                            const int ix = __float_as_int(fmaxf(t.x, LIN_LO)), iy = __float_as_int(fmaxf(t.y, LIN_LO));
                            return make_float2(__int_as_float((ix << 15) + LIN_K), __int_as_float((iy << 15) + LIN_K));
                        }
                        const float2 x = ffma2(sv, q < 32 ? sl2a_2 : sl2b_2, negm_2);
                        return make_float2(ex2(x.x), ex2(x.y));
                    };
#pragma unroll
                    for (int k = 0; k < 32; ++k) {
                        const float2 pa = exp_pair(2 * k), pb2 = exp_pair(2 * k + 1);
                        pk[k] = pack4(pa.x, pa.y, pb2.x, pb2.y);
                    }
                }
                // the P buffer is free once P V of pair g - 3 has completed
                mbar_wait(bar(B_PV_DONE + pb), ((g / PBUFS) & 1) ^ 1);
                tc_fence_after();
                tmem_st32(tP, pk);
                tc_wait_st();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(B_P_READY + pb));
            }
            g0 += it.np;
            // ---------------- epilogue: normalise by the accumulated row sum, convert, store ------------------
            // Warp (sm, wq) finalises O columns [64 sm, 64 sm + 64) of its 32 rows.  The row sum stands in column
            // 128 of the accumulator under the same reference as O.
            if (lane == 0 && wq == 0) tma_store_wait_read();   // staging slab sm is free again
            named_bar_sync(NB_HALF + sm, 128);                 // staging free for the whole warpgroup
            float inv = 0.f, L = 0.f;
            if (it.nt > 0) {
                mbar_wait(bar(B_ITEM_DONE), icnt & 1);         // every P V of the item has completed
                tc_fence_after();
                uint32_t l1[1];
                tmem_ld1(tOs + TM_L, l1);
                tc_wait_ld();
                L = __uint_as_float(l1[0]);
                inv = (L > 0.f) ? 1.f / L : 0.f;
            }
            // optional row log-sum-exp (natural log; -inf for an empty row): the parity that handled the last pair
            // holds the reference under which O and L stand
            if (p.lse != nullptr && it.qb * BQ + row < p.N && sm == (it.nt > 0 ? ((it.np - 1) & 1) : 0))
                p.lse[(static_cast<int64_t>(it.b) * p.H + it.h) * p.N + it.qb * BQ + row] =
                    (L > 0.f) ? (m_ref + lg2(L) - P_SHIFT) * 0.6931471805599453f : -INFINITY;
            const uint32_t srow = sO + sm * 16384 + row * 128;
            const uint32_t tO = tOs + sm * 64;
            // O[:, c] carries V's per-channel scale (R10)
            const float4* vsc = reinterpret_cast<const float4*>(p.v_scale + (static_cast<int64_t>(it.b) * p.H + it.h) * 128 + sm * 64);
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
                    const float4 sc = __ldg(vsc + c * 8 + k4);
                    float x0 = 0.f, x1 = 0.f, x2 = 0.f, x3 = 0.f;
                    if (it.nt > 0) {
                        x0 = __uint_as_float(o[4 * k4]) * (inv * sc.x);     x1 = __uint_as_float(o[4 * k4 + 1]) * (inv * sc.y);
                        x2 = __uint_as_float(o[4 * k4 + 2]) * (inv * sc.z); x3 = __uint_as_float(o[4 * k4 + 3]) * (inv * sc.w);
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
                if (lane == 0) mbar_arrive(bar(B_O_FREE));
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

template <bool kBeta, bool kHalf>
cudaError_t launch_one(const CUtensorMap& tmQ, const CUtensorMap& tmK, const CUtensorMap& tmV,
                       const CUtensorMap& tmO, const AttnParams& p, cudaStream_t stream) {
    cudaError_t e = cudaFuncSetAttribute(attn_fwd_fp8_kernel<kBeta, kHalf>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    if (e != cudaSuccess) return e;
    int dev = 0, sms = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    const int n_items = p.B * p.H * p.nq;
    const int grid = n_items < sms ? n_items : sms;
    AttnParams pl = p;
    pl.ticket_slot = next_ticket_slot();
    attn_fwd_fp8_kernel<kBeta, kHalf><<<grid, NUM_THREADS, SMEM_BYTES, stream>>>(tmQ, tmK, tmV, tmO, pl);
    count_launch(1);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_attn_fwd_fp8(const CUtensorMap& tmQ, const CUtensorMap& tmK, const CUtensorMap& tmV,
                                const CUtensorMap& tmO, const AttnParams& p, cudaStream_t stream) {
    const bool beta = p.n_first > 0 && p.beta != 1.f;
    if (beta && p.half_flags) return launch_one<true, true>(tmQ, tmK, tmV, tmO, p, stream);
    if (beta) return launch_one<true, false>(tmQ, tmK, tmV, tmO, p, stream);
    if (p.half_flags) return launch_one<false, true>(tmQ, tmK, tmV, tmO, p, stream);
    return launch_one<false, false>(tmQ, tmK, tmV, tmO, p, stream);
}

}  // namespace chorus
