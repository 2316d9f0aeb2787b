// mask_build.cu — the historical request's side of sparsity reuse ("in the dense case
// we select a block-level mask from its attention map via top-p with a top-k floor", L93 (2)
// min_top_k, L73 coverage):
//   chorus_block_mass      dense QK^T on the tensor cores, two passes over the keys of a query block
//                          (row log-sum-exp, then normalised probabilities summed per 128 x 64 block)
//   chorus_mask_from_mass  per row: integer masses, bitonic sort, prefix sums, top-p prefix with a
//                          top-k floor -> packed bitmask (the layout chorus_mask_to_index reads)
//   chorus_mask_coverage   per head: kept mass / total mass
#include <cuda_bf16.h>

#include "chorus_internal.h"
#include "sm100_ptx.cuh"

namespace chorus {
namespace {

using namespace ptx;

// =================================================================================================
// block mass
// =================================================================================================
// Persistent kernel, one CTA (576 threads) per SM, work item = one (batch, head, 256-row query
// block): TWO 128-row query tiles share every key tile that is brought in.  Keys are taken 128 at a
// time ("a pair" of 64-key blocks); an item makes 2 * P steps over its P pairs: steps 0..P-1 give
// every row its running maximum and sum (-> log-sum-exp), steps P..2P-1 recompute the same scores and
// sum exp2(s - lse) over the rows and the 64 columns of each block.  Recomputing QK^T costs a second
// MMA pass, but nothing of size N x N is ever stored.  When the caller hands in the rows' log-sum-exp
// (an output of the dense attention call that the historical request makes anyway), the
// first pass is skipped (template kLse).
//   warp 16     TMA producer: the two Q tiles once per item, then the K pair of every step (ring of KST stages)
//   warp 17     MMA issuer: per step S_q = Q_q K^T (M=128, N=128, K=128, bf16 -> fp32) for q = 0, 1 into
//               two of four S buffers in tensor memory, one step ahead of the readers
//   warps 0-15  four groups of four: group (q, parity) reads query tile q on the steps of that parity, i.e.
//               it owns S buffer 2 * parity + q; warp w owns TMEM lanes 32*(w%4).. (one query row per
//               thread); an S buffer is released as soon as it is in registers.  Four reader warps per
//               scheduler (at <= 112 registers) keep its MUFU busy: one warp's exponential pass is paced
//               by ptxas at one MUFU.EX2 per 8 cycles, the pipe's own rate, and every stall of a lone warp
//               is a stall of the pipe (80 % MUFU utilisation with four warps, 54 % with two).
constexpr int MB_THREADS = 576, MB_READERS = 16, MB_PRODUCER = 16, MB_MMA = 17;
constexpr int KST = 4, SB = 4;
constexpr uint32_t MASS_POLY = 0x49u;                  // element pairs 0, 3, 6 of every 8: polynomial exp2
constexpr uint32_t TILE = 32768;                       // 128 rows x 128 bf16 channels (two slabs)
constexpr uint32_t M_SQ = 0, M_SK = 2 * TILE, M_XCH = M_SK + KST * TILE, M_BAR = M_XCH + 4096 + 512,
                   M_SMEM = M_BAR + 256;
// mbarrier slots
constexpr uint32_t B_Q_FULL = 0, B_Q_EMPTY = 1, B_K_FULL = 2, B_K_EMPTY = B_K_FULL + KST,
                   B_S_FULL = B_K_EMPTY + KST, B_S_FREE = B_S_FULL + SB, B_CNT = B_S_FREE + SB;
static_assert(B_CNT * 8 + 8 <= 256, "barrier area too small");

struct MassParams {
    float* mass;
    const float* lse;   // optional [B][H][N] natural-log row log-sum-exp of the SAME dense attention
    int B, H, N, nq, nk;
    float scale_log2;
    int geo64;          // 1: output in the paper's 64 x 128 geometry, [B][H][ceil(N/64)][ceil(N/128)]
};

template <bool kLse>   // the rows' log-sum-exp is given: one pass over the keys instead of two
__global__ void __launch_bounds__(MB_THREADS, 1)
block_mass_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                  const MassParams p) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t base = smem_u32(smem_raw);
    if (base & 1023u) __trap();
    const uint32_t sQ = base + M_SQ, sK = base + M_SK, bars = base + M_BAR;
    auto bar = [&](uint32_t i) { return bars + 8u * i; };
    volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem_raw + M_BAR + 8 * B_CNT);
    volatile float* xst = reinterpret_cast<volatile float*>(smem_raw + M_XCH);            // [2 tiles][2 parities][m, l][128]
    volatile float* xpart = reinterpret_cast<volatile float*>(smem_raw + M_XCH + 4096);   // [4 groups][2 bufs][4 warps][2]

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nq2 = (p.nq + 1) >> 1;     // 256-row items per head
    const int n_items = p.B * p.H * nq2;
    const int P = (p.nk + 1) >> 1;       // pairs per item
    // With the rows' log-sum-exp given (an output of the dense attention call) the first pass is
    // skipped: P steps instead of 2 P, one exponential per score instead of two.
    const int T = kLse ? P : 2 * P;       // steps per item
    if (threadIdx.x == 0) {
        mbar_init(bar(B_Q_FULL), 1);
        mbar_init(bar(B_Q_EMPTY), 1);
        for (int i = 0; i < KST; ++i) { mbar_init(bar(B_K_FULL + i), 1); mbar_init(bar(B_K_EMPTY + i), 1); }
        for (int i = 0; i < SB; ++i) { mbar_init(bar(B_S_FULL + i), 1); mbar_init(bar(B_S_FREE + i), 4); }
        fence_mbar_init();
    }
    if (warp == MB_MMA) tmem_alloc(bars + 8 * B_CNT, 512);
    if (warp == MB_PRODUCER && lane == 0) { prefetch_tmap(&tmQ); prefetch_tmap(&tmK); }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp == MB_PRODUCER) {
        uint32_t st = 0, ph = 0, icnt = 0;
        for (int idx = blockIdx.x; idx < n_items; idx += gridDim.x, ++icnt) {
            const int qb2 = idx % nq2, bh = idx / nq2, h = bh % p.H, b = bh / p.H;
            mbar_wait(bar(B_Q_EMPTY), (icnt & 1) ^ 1);
            if (elect_one()) {
                // rows >= N (the second tile of an odd last item included) arrive as zeros
                mbar_arrive_expect_tx(bar(B_Q_FULL), 2 * TILE);
                for (int q = 0; q < 2; ++q) {
                    tma_load_4d(sQ + q * TILE, &tmQ, bar(B_Q_FULL), 0, (2 * qb2 + q) * 128, h, b);
                    tma_load_4d(sQ + q * TILE + 16384, &tmQ, bar(B_Q_FULL), 64, (2 * qb2 + q) * 128, h, b);
                }
            }
            __syncwarp();
            for (int t = 0; t < T; ++t) {
                const int j = t < P ? t : t - P;
                mbar_wait(bar(B_K_EMPTY + st), ph ^ 1);
                if (elect_one()) {
                    mbar_arrive_expect_tx(bar(B_K_FULL + st), TILE);
                    const uint32_t dst = sK + st * TILE;
                    tma_load_4d(dst, &tmK, bar(B_K_FULL + st), 0, j * 128, h, b);       // keys >= N: zeros
                    tma_load_4d(dst + 16384, &tmK, bar(B_K_FULL + st), 64, j * 128, h, b);
                }
                __syncwarp();
                if (++st == KST) { st = 0; ph ^= 1; }
            }
        }
    } else if (warp == MB_MMA) {
        constexpr uint32_t IDESC = make_idesc(1u, 1u, 128, 128, 0, 0);    // bf16 x bf16 -> fp32
        const uint64_t dQ = smem_desc_sw128(sQ, 16, 1024);
        const uint64_t dK = smem_desc_sw128(sK, 16, 1024);
        uint32_t st = 0, ph = 0, icnt = 0, g = 0;      // g: steps so far; step g writes S buffers 2 (g & 1) + q
        for (int idx = blockIdx.x; idx < n_items; idx += gridDim.x, ++icnt) {
            mbar_wait(bar(B_Q_FULL), icnt & 1);
            for (int t = 0; t < T; ++t, ++g) {
                mbar_wait(bar(B_K_FULL + st), ph);
                for (int q = 0; q < 2; ++q) {
                    const uint32_t sb = 2 * (g & 1) + q;
                    if (g >= 2) mbar_wait(bar(B_S_FREE + sb), ((g >> 1) - 1) & 1);
                    tc_fence_after();
                    if (elect_one()) {
                        const uint32_t tS = tmem + sb * 128;
                        const uint64_t dQq = dQ + ((q * TILE) >> 4);
                        const uint64_t dKs = dK + ((st * TILE) >> 4);
#pragma unroll
                        for (int ks = 0; ks < 8; ++ks) {     // 16 bf16 channels = 32 B per step, 2 slabs
                            const uint32_t off = ((ks >> 2) * 16384 + (ks & 3) * 32) >> 4;
                            mma_f16_ss(tS, dQq + off, dKs + off, IDESC, ks > 0);
                        }
                        tc_commit(bar(B_S_FULL + sb));
                        if (q == 1) {
                            tc_commit(bar(B_K_EMPTY + st));
                            if (t == T - 1) tc_commit(bar(B_Q_EMPTY));
                        }
                    }
                    __syncwarp();
                }
                if (++st == KST) { st = 0; ph ^= 1; }
            }
        }
    } else if (warp < MB_READERS) {
        // group = (query tile of the item, parity of the steps it reads): it owns S buffer 2 * parity + tile
        const int grp = warp >> 2, tile = grp & 1, par = grp >> 1, wq = warp & 3, row = wq * 32 + lane;
        const uint32_t tlane = tmem + (static_cast<uint32_t>(wq * 32) << 16);
        const float sl2 = p.scale_log2;
        uint32_t g0 = 0;                        // steps of all previous items
        uint32_t own = 0;                       // mass steps of this group so far (xpart buffer)
        for (int idx = blockIdx.x; idx < n_items; idx += gridDim.x) {
            const int qb = 2 * (idx % nq2) + tile;          // this group's 128-row query block
            const int64_t bh = idx / nq2;
            const bool tile_ok = qb < p.nq;                 // the second tile of an odd last item does not exist
            const bool row_ok = qb * 128 + row < p.N;
            float m = -INFINITY, l = 0.f, lse2 = 0.f;
            if (kLse && row_ok)                 // natural log -> the log2 domain of the scores
                lse2 = __ldg(p.lse + bh * p.N + qb * 128 + row) * 1.4426950408889634f;
            bool second = kLse;                  // the mass pass has begun (with an LSE given: from the start)
            // pass boundary: the two groups of a tile combine their (m, l) into the row's log-sum-exp
            auto boundary = [&]() {
                second = true;
                xst[((tile * 2 + par) * 2 + 0) * 128 + row] = m;
                xst[((tile * 2 + par) * 2 + 1) * 128 + row] = l;
                named_bar_sync(6 + tile, 256);
                const float mo = xst[((tile * 2 + (par ^ 1)) * 2 + 0) * 128 + row];
                const float lo = xst[((tile * 2 + (par ^ 1)) * 2 + 1) * 128 + row];
                const float M = fmaxf(m, mo);               // finite: every row sees at least one key
                const float L = (m == -INFINITY ? 0.f : l * ex2(m - M)) + (mo == -INFINITY ? 0.f : lo * ex2(mo - M));
                lse2 = M + lg2(L);
                named_bar_sync(6 + tile, 256);               // both have read: the slots may be rewritten
            };
            // this group's steps: those whose number g0 + t has its parity
            for (int t = (par ^ static_cast<int>(g0 & 1u)); t < T; t += 2) {
                if (!second && t >= P) boundary();
                const uint32_t g = g0 + t;
                const uint32_t sb = 2 * par + tile;
                const int j = t < P ? t : t - P;
                const int valid = min(128, p.N - j * 128);   // keys of this pair that exist
                mbar_wait(bar(B_S_FULL + sb), (g >> 1) & 1);
                tc_fence_after();
                const uint32_t tS = tlane + sb * 128;
                float sum_a = 0.f, sum_b = 0.f;
                if ((kLse || t >= P) && valid == 128) {
                    // ---- the common step (mass pass, all 128 keys exist): the four 32-column chunks are streamed
                    // with the next chunk's load in flight, packed FFMA2 / FADD2, and three of every 8 element
                    // pairs (MASS_POLY) take their exponential from the degree-3 polynomial on the FMA pipe
                    // (relative error 1e-4; tolerance of the masses 2e-3)
                    const float2 sl2_2 = make_float2(sl2, sl2), nlse_2 = make_float2(-lse2, -lse2);
                    auto chunk = [&](const uint32_t (&r)[32], float2& acc) {
#pragma unroll
                        for (int q = 0; q < 16; ++q) {
                            const float2 x = ffma2(make_float2(__uint_as_float(r[2 * q]), __uint_as_float(r[2 * q + 1])),
                                                   sl2_2, nlse_2);
                            const float2 e = ((MASS_POLY >> (q & 7)) & 1u) ? exp2_poly2<3>(x)
                                                                           : make_float2(ex2(x.x), ex2(x.y));
                            acc = fadd2(acc, e);
                        }
                    };
                    uint32_t ra[32], rb[32];
                    float2 acc_a = make_float2(0.f, 0.f), acc_b = make_float2(0.f, 0.f);
                    tmem_ld32(tS, ra);
                    tc_wait_ld();
                    tmem_ld32(tS + 32, rb);
                    chunk(ra, acc_a);
                    tc_wait_ld();
                    tmem_ld32(tS + 64, ra);
                    chunk(rb, acc_a);
                    tc_wait_ld();
                    tmem_ld32(tS + 96, rb);
                    chunk(ra, acc_b);
                    tc_wait_ld();
                    tc_fence_before();                       // the buffer is in registers: hand it back
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar(B_S_FREE + sb));
                    chunk(rb, acc_b);
                    sum_a = acc_a.x + acc_a.y;
                    sum_b = acc_b.x + acc_b.y;
                } else if (!kLse && t < P && valid == 128) {
                    // ---- the common step of the first pass: online maximum and sum per 32-column chunk, streamed
                    // and packed like the mass pass
                    const float2 sl2_2 = make_float2(sl2, sl2);
                    auto chunk1 = [&](const uint32_t (&r)[32]) {
                        float a0 = -INFINITY, a1 = -INFINITY;
#pragma unroll
                        for (int k = 0; k < 32; k += 4) {
                            a0 = fmaxf(fmaxf(a0, __uint_as_float(r[k])), __uint_as_float(r[k + 1]));
                            a1 = fmaxf(fmaxf(a1, __uint_as_float(r[k + 2])), __uint_as_float(r[k + 3]));
                        }
                        const float mn = fmaxf(m, fmaxf(a0, a1) * sl2);      // sl2 > 0
                        l *= ex2(m - mn);                                    // m = -inf: l is 0 and stays 0
                        m = mn;
                        const float2 nm_2 = make_float2(-m, -m);
                        float2 acc = make_float2(0.f, 0.f);
#pragma unroll
                        for (int q = 0; q < 16; ++q) {
                            const float2 x = ffma2(make_float2(__uint_as_float(r[2 * q]), __uint_as_float(r[2 * q + 1])),
                                                   sl2_2, nm_2);
                            const float2 e = ((MASS_POLY >> (q & 7)) & 1u) ? exp2_poly2<3>(x)
                                                                           : make_float2(ex2(x.x), ex2(x.y));
                            acc = fadd2(acc, e);
                        }
                        l += acc.x + acc.y;
                    };
                    uint32_t ra[32], rb[32];
                    tmem_ld32(tS, ra);
                    tc_wait_ld();
                    tmem_ld32(tS + 32, rb);
                    chunk1(ra);
                    tc_wait_ld();
                    tmem_ld32(tS + 64, ra);
                    chunk1(rb);
                    tc_wait_ld();
                    tmem_ld32(tS + 96, rb);
                    chunk1(ra);
                    tc_wait_ld();
                    tc_fence_before();                       // the buffer is in registers: hand it back
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar(B_S_FREE + sb));
                    chunk1(rb);
                } else
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    uint32_t r[32];
                    tmem_ld32(tS + 32 * c, r);
                    tc_wait_ld();
                    if (c == 3) {                            // the buffer is in registers: hand it back
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive(bar(B_S_FREE + sb));
                    }
                    const int vc = valid - 32 * c;           // valid columns of this chunk
                    if (!kLse && t < P) {
                        float cm = -INFINITY;
#pragma unroll
                        for (int k = 0; k < 32; ++k)
                            if (k < vc) cm = fmaxf(cm, __uint_as_float(r[k]));
                        if (cm > -INFINITY) {
                            const float mn = fmaxf(m, cm * sl2);
                            l *= ex2(m - mn);                // m = -inf: l is 0 and stays 0
                            m = mn;
                            float acc = 0.f;
#pragma unroll
                            for (int k = 0; k < 32; ++k)
                                if (k < vc) acc += ex2(fmaf(__uint_as_float(r[k]), sl2, -m));
                            l += acc;
                        }
                    } else {
                        float acc = 0.f;
#pragma unroll
                        for (int k = 0; k < 32; ++k)
                            if (k < vc) acc += ex2(fmaf(__uint_as_float(r[k]), sl2, -lse2));
                        if (c < 2) sum_a += acc; else sum_b += acc;
                    }
                }
                if (kLse || t >= P) {
                    // ---- sums over the 128 rows: lanes, then the four warps in a fixed order ------
                    if (!row_ok) { sum_a = 0.f; sum_b = 0.f; }
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) {
                        sum_a += __shfl_xor_sync(0xffffffffu, sum_a, o);
                        sum_b += __shfl_xor_sync(0xffffffffu, sum_b, o);
                    }
                    volatile float* part = xpart + ((grp * 2 + (own & 1)) * 4) * 2;
                    if (lane == 0) { part[wq * 2] = sum_a; part[wq * 2 + 1] = sum_b; }
                    named_bar_sync(2 + grp, 128);
                    if (wq == 0 && lane == 0 && tile_ok) {
                        const float a = ((part[0] + part[2]) + part[4]) + part[6];
                        const float bsum = ((part[1] + part[3]) + part[5]) + part[7];
                        if (p.geo64) {
                            // 64 x 128 geometry: step j is key block j; warps 0-1 / 2-3 hold rows 0-63 / 64-127
                            const int nq64 = (p.N + 63) >> 6, nk128 = p.nq;
                            float* out = p.mass + (bh * nq64 + 2 * qb) * nk128 + j;
                            out[0] = (part[0] + part[2]) + (part[1] + part[3]);
                            if (2 * qb + 1 < nq64) out[nk128] = (part[4] + part[6]) + (part[5] + part[7]);
                        } else {
                            float* out = p.mass + (bh * p.nq + qb) * p.nk + 2 * j;
                            out[0] = a;
                            if (2 * j + 1 < p.nk) out[1] = bsum;
                        }
                    }
                    ++own;
                }
            }
            if (!second) boundary();             // (a single pair: this group had no step in the mass pass)
            g0 += T;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == MB_MMA) tmem_dealloc(tmem, 512);
}

// =================================================================================================
// top-p with a top-k floor
// =================================================================================================
constexpr int SEL_THREADS = 256;

// One CTA per row.  Key of block k: ((q + 1) << 11) | (2047 - k) with q = floor(mass * 2^24): sorting
// the keys in DESCENDING order ranks by q descending, ties by index ascending; padding keys are 0.
__global__ void __launch_bounds__(SEL_THREADS)
mask_from_mass_kernel(const float* __restrict__ mass, int nk, int words, int n_sort, double top_p,
                      int n_floor, uint32_t* __restrict__ bitmask, int32_t* __restrict__ kept) {
    extern __shared__ unsigned long long keys[];       // [n_sort]
    __shared__ unsigned long long s_red[SEL_THREADS / 32];
    __shared__ unsigned long long s_total;
    __shared__ uint32_t s_words[64];
    __shared__ int s_np;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const float* mr = mass + static_cast<int64_t>(blockIdx.x) * nk;

    unsigned long long mine = 0;
    for (int k = tid; k < n_sort; k += SEL_THREADS) {
        unsigned long long key = 0;
        if (k < nk) {
            const unsigned long long q = static_cast<unsigned long long>(floor(static_cast<double>(mr[k]) * 16777216.0));
            mine += q;
            key = ((q + 1ull) << 11) | static_cast<unsigned long long>(2047 - k);
        }
        keys[k] = key;
    }
    if (tid < 64) s_words[tid] = 0u;
    if (tid == 0) s_np = nk;
    // total of q (integers: any order gives the same sum)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mine += __shfl_xor_sync(0xffffffffu, mine, o);
    if (lane == 0) s_red[warp] = mine;
    __syncthreads();
    if (tid == 0) {
        unsigned long long t = 0;
        for (int w = 0; w < SEL_THREADS / 32; ++w) t += s_red[w];
        s_total = t;
    }
    // bitonic sort, descending
    for (int size = 2; size <= n_sort; size <<= 1) {
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            __syncthreads();
            for (int i = tid; i < (n_sort >> 1); i += SEL_THREADS) {
                const int lo = ((i / stride) * stride << 1) + (i % stride), hi = lo + stride;
                const bool desc = ((lo & size) == 0);
                const unsigned long long a = keys[lo], b = keys[hi];
                if ((a < b) == desc) { keys[lo] = b; keys[hi] = a; }
            }
        }
    }
    __syncthreads();
    const unsigned long long total = s_total;
    const unsigned long long target = static_cast<unsigned long long>(ceil(top_p * static_cast<double>(total)));
    // shortest prefix (in sorted order) whose q-sum reaches the target: contiguous chunk per thread,
    // exclusive scan of the chunk sums over the block, then a walk inside the chunk
    const int per = n_sort / SEL_THREADS > 0 ? n_sort / SEL_THREADS : 1;
    const int p0 = tid * per;
    unsigned long long csum = 0;
    if (p0 < n_sort)
        for (int i = 0; i < per; ++i) {
            const unsigned long long key = keys[p0 + i];
            csum += key ? (key >> 11) - 1ull : 0ull;
        }
    unsigned long long inc = csum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long u = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += u;
    }
    __syncthreads();                 // s_red is free again
    if (lane == 31) s_red[warp] = inc;
    __syncthreads();
    unsigned long long before = inc - csum;
    for (int w = 0; w < warp; ++w) before += s_red[w];
    if (total > 0 && target > 0 && p0 < n_sort && before < target && before + csum >= target) {
        unsigned long long acc = before;
        for (int i = 0; i < per; ++i) {
            const unsigned long long key = keys[p0 + i];
            acc += key ? (key >> 11) - 1ull : 0ull;
            if (acc >= target) { s_np = p0 + i + 1; break; }     // exactly one thread gets here
        }
    }
    __syncthreads();
    const int n_p = (total > 0 && target > 0) ? s_np : 0;
    const int n = n_p > n_floor ? n_p : n_floor;
    for (int i = tid; i < n; i += SEL_THREADS) {
        const int k = 2047 - static_cast<int>(keys[i] & 2047ull);
        atomicOr(&s_words[k >> 5], 1u << (k & 31));
    }
    __syncthreads();
    if (tid < words) bitmask[static_cast<int64_t>(blockIdx.x) * words + tid] = s_words[tid];
    if (kept && tid == 0) kept[blockIdx.x] = n;
}

// One CTA per head; fp64 sums, fixed order.
__global__ void __launch_bounds__(256)
mask_coverage_kernel(const float* __restrict__ mass, const uint32_t* __restrict__ bitmask, int nq,
                     int nk, int words, float* __restrict__ coverage) {
    __shared__ double s_in[256], s_all[256];
    const int h = blockIdx.x;
    const int64_t n = static_cast<int64_t>(nq) * nk;
    double in = 0.0, all = 0.0;
    for (int64_t e = threadIdx.x; e < n; e += 256) {
        const int64_t r = static_cast<int64_t>(h) * nq + e / nk;
        const int kb = static_cast<int>(e % nk);
        const double m = static_cast<double>(mass[static_cast<int64_t>(h) * n + e]);
        all += m;
        if ((bitmask[r * words + (kb >> 5)] >> (kb & 31)) & 1u) in += m;
    }
    s_in[threadIdx.x] = in;
    s_all[threadIdx.x] = all;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) {
            s_in[threadIdx.x] += s_in[threadIdx.x + o];
            s_all[threadIdx.x] += s_all[threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) coverage[h] = s_all[0] > 0.0 ? static_cast<float>(s_in[0] / s_all[0]) : 0.f;
}

}  // namespace

cudaError_t launch_block_mass(const CUtensorMap& tmQ, const CUtensorMap& tmK, const float* lse, float* mass,
                              int B, int H, int N, float scale_log2, bool geo64, cudaStream_t stream) {
    cudaError_t e = lse ? cudaFuncSetAttribute(block_mass_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, M_SMEM)
                        : cudaFuncSetAttribute(block_mass_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, M_SMEM);
    if (e != cudaSuccess) return e;
    int dev = 0, sms = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    MassParams p;
    p.mass = mass;
    p.lse = lse;
    p.B = B; p.H = H; p.N = N;
    p.nq = (N + 127) / 128;
    p.nk = (N + 63) / 64;
    p.scale_log2 = scale_log2;
    p.geo64 = geo64 ? 1 : 0;
    const int n_items = B * H * ((p.nq + 1) / 2);
    const int grid = n_items < sms ? n_items : sms;
    if (lse) block_mass_kernel<true><<<grid, MB_THREADS, M_SMEM, stream>>>(tmQ, tmK, p);
    else block_mass_kernel<false><<<grid, MB_THREADS, M_SMEM, stream>>>(tmQ, tmK, p);
    count_launch(1);
    return cudaGetLastError();
}

cudaError_t launch_mask_from_mass(const float* mass, int64_t rows, int nk, double top_p, double min_top_k,
                                  uint32_t* bitmask, int32_t* kept, cudaStream_t stream) {
    int n_sort = 64;
    while (n_sort < nk) n_sort <<= 1;
    int n_floor = static_cast<int>(ceil(min_top_k * static_cast<double>(nk)));
    n_floor = n_floor < 0 ? 0 : (n_floor > nk ? nk : n_floor);
    if (n_sort < SEL_THREADS) n_sort = SEL_THREADS;     // one key per thread at least
    mask_from_mass_kernel<<<static_cast<unsigned>(rows), SEL_THREADS, n_sort * sizeof(unsigned long long), stream>>>(
        mass, nk, (nk + 31) / 32, n_sort, top_p, n_floor, bitmask, kept);
    count_launch(1);
    return cudaGetLastError();
}

cudaError_t launch_mask_coverage(const float* mass, const uint32_t* bitmask, int heads, int nq, int nk,
                                 float* coverage, cudaStream_t stream) {
    mask_coverage_kernel<<<heads, 256, 0, stream>>>(mass, bitmask, nq, nk, (nk + 31) / 32, coverage);
    count_launch(1);
    return cudaGetLastError();
}

}  // namespace chorus
