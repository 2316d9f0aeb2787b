// chorus_oracle.cpp — CPU oracle for the Chorus II sparsity-reuse hot path.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no code,
// header, table or helper with the CUDA path under paper_2606_25040_b200/csrc/, and the CUDA path
// never calls it.
//
// Plain, slow, obviously-correct fp64 restatement of what the path computes, written from
// /root/reference/PAPER.md (cited as PAPER.md:L<n>) and the readings listed in DESIGN.md §3
// ("R<k>").  No blocking, fusion or reordering beyond what the definitions state; OpenMP only
// distributes independent (head, query-block) items over host cores.
//
// Pin status (tests/test_oracle_*.py, all `-m "not gpu"`):
//   oracle_mask_to_index        pinned (brute force, popcount total, round trip, word-boundary cases)
//   oracle_block_sparse_attn    pinned (numpy dense fp64 softmax for full/diagonal/single-block masks,
//                               long-double brute force with materialised -inf scores, closed forms,
//                               hand-derived golden fixture, permutation invariance, padded tail);
//                               first-frame key scaling (eq. 1): numpy dense attention on hand-scaled
//                               keys, closed form; 64 x 128 geometry: numpy token-level masked softmax
//   oracle_mask_to_index_64x128 pinned (brute-force restatement, round trip to the token-level keep
//                               matrix of the mask, ascending / no duplicates)
//   oracle_mask_to_index_u16, oracle_mask_to_index_64x128_u16
//                               pinned (independent per-bit Python loops, agreement with the 32-bit forms
//                               entry by entry, flag positions, the does-not-fit refusals)
//   oracle_quantize_fp8         pinned (torch.float8_e4m3fn cast as an independent library routine,
//                               error bound, exact round trip of {0, +-amax}); the FORMAT itself
//                               (granularity, amax/448) is reading R10/R11 — the paper only says
//                               "FP8 quantization", so that choice is "parity unpinned"
//                               by the paper and pinned only by BASELINE.json cfg3.
//   oracle_retrieve_top1        pinned (planted neighbour, numpy argmax)
//   oracle_visit_refresh        pinned (brute force per bit, every pair visited once per group)
//   oracle_block_mass           pinned (numpy dense softmax summed per block, rows sum to 1, uniform
//                               attention closed form; 64 x 128 geometry: numpy, and agreement of
//                               the two geometries on 128 x 128 super-blocks)
//   oracle_mask_from_mass       pinned (exact-rational brute force on tiny rows, minimality of the
//                               kept prefix, floor count, ties by index, hand-worked golden row)
//   oracle_mask_coverage        pinned (numpy; full mask = 1, top-p mask >= p)
//
// Build: g++ -O3 -march=native -fopenmp -shared -fPIC (see oracle/build.py).

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---- exact input conversions (the oracle's own; nothing shared with the CUDA side) -------------

// bf16 -> double: a bf16 is the top 16 bits of an IEEE binary32.
inline double bf16_to_double(uint16_t b) {
    uint32_t u = static_cast<uint32_t>(b) << 16;
    float f;
    std::memcpy(&f, &u, 4);
    return static_cast<double>(f);
}

// IEEE binary16 -> double: 1 sign, 5 exponent (bias 15), 10 mantissa; subnormals m/1024 * 2^-14.
inline double f16_to_double(uint16_t hbits) {
    const int sign = (hbits >> 15) & 1, e = (hbits >> 10) & 0x1F, m = hbits & 0x3FF;
    double v;
    if (e == 0x1F) v = m ? std::numeric_limits<double>::quiet_NaN() : std::numeric_limits<double>::infinity();
    else if (e == 0) v = std::ldexp(static_cast<double>(m) / 1024.0, -14);
    else v = std::ldexp(1.0 + static_cast<double>(m) / 1024.0, e - 15);
    return sign ? -v : v;
}

// e4m3fn -> double.  1 sign, 4 exponent (bias 7), 3 mantissa; no infinities; S.1111.111 is NaN;
// largest finite 448 = 1.75 * 2^8; subnormals m/8 * 2^-6.
inline double e4m3_to_double(uint8_t c) {
    const int sign = (c >> 7) & 1;
    const int e = (c >> 3) & 0xF;
    const int m = c & 0x7;
    double v;
    if (e == 0xF && m == 0x7) {
        v = std::numeric_limits<double>::quiet_NaN();
    } else if (e == 0) {
        v = std::ldexp(static_cast<double>(m) / 8.0, -6);
    } else {
        v = std::ldexp(1.0 + static_cast<double>(m) / 8.0, e - 7);
    }
    return sign ? -v : v;
}

// float -> e4m3fn code, round-to-nearest-even, saturating to +-448 (reading R11).  Written as a
// search over the 127 non-negative finite codes so that it is checkable by eye: pick the nearest
// representable magnitude, ties to the even code.
inline uint8_t float_to_e4m3_rne_sat(float x) {
    if (std::isnan(x)) return 0x7F;
    const uint8_t sign = std::signbit(x) ? 0x80 : 0x00;
    const double a = std::fabs(static_cast<double>(x));
    if (a >= 448.0) return sign | 0x7E;  // saturate (0x7E = 448)
    // codes 0x00..0x7E are monotonically increasing in magnitude
    int lo = 0, hi = 0x7E;
    while (hi - lo > 1) {  // invariant: value(lo) <= a < value(hi)
        const int mid = (lo + hi) / 2;
        if (e4m3_to_double(static_cast<uint8_t>(mid)) <= a) lo = mid; else hi = mid;
    }
    const double vlo = e4m3_to_double(static_cast<uint8_t>(lo));
    const double vhi = e4m3_to_double(static_cast<uint8_t>(hi));
    int pick;
    if (a - vlo < vhi - a) pick = lo;
    else if (a - vlo > vhi - a) pick = hi;
    else pick = (lo % 2 == 0) ? lo : hi;  // tie -> even mantissa LSB == even code
    return sign | static_cast<uint8_t>(pick);
}

inline bool mask_bit(const uint32_t* row_words, int kb) {
    return (row_words[kb >> 5] >> (kb & 31)) & 1u;  // LSB-first packing, reading R1
}

constexpr int BQ = 128;  // query rows per block  (BASELINE.json north_star; reading R3)
constexpr int BK = 64;   // keys per block

}  // namespace

extern "C" {

// -------------------------------------------------------------------------------------------------
// a-1  Mask decode.  PAPER.md:L81 (mask stored per layer/head), L93 (binary per
// (head, q-block, k-block)), L97 (kernel visits only retained pairs).  Rows are visited in
// (l, h, qb) order; each row lists its set key blocks in ascending order; row_ptr is the running
// count.  One bit tested at a time, nothing clever.  Bits >= nk in the last word are ignored (R1).
// col_idx may be null (count only).  Returns nnz.
// -------------------------------------------------------------------------------------------------
int64_t oracle_mask_to_index(const uint32_t* bitmask, int L, int H, int nq, int nk,
                             int32_t* row_ptr, int32_t* col_idx) {
    const int words = (nk + 31) / 32;
    int64_t nnz = 0;
    int64_t r = 0;
    row_ptr[0] = 0;
    for (int l = 0; l < L; ++l)
        for (int h = 0; h < H; ++h)
            for (int qb = 0; qb < nq; ++qb, ++r) {
                const uint32_t* row = bitmask + r * words;
                for (int kb = 0; kb < nk; ++kb) {
                    if (mask_bit(row, kb)) {
                        if (col_idx) col_idx[nnz] = kb;
                        ++nnz;
                    }
                }
                row_ptr[r + 1] = static_cast<int32_t>(nnz);
            }
    return nnz;
}

// -------------------------------------------------------------------------------------------------
// f-4  Decode of a mask in the paper's own geometry (64 query rows x 128 keys per
// block) into the index the 128 x 64 kernel walks (R26).  bitmask is
// [L][H][nq64][words], nq64 = ceil(N/64), bit kb of a row = key block kb (keys 128 kb .. 128 kb + 127)
// of nk128 = ceil(N/128).  Output row R = (l, h, qb128) covers mask rows 2 qb128 ("upper", query
// rows 0-63 of the 128) and 2 qb128 + 1 ("lower", if it exists).  For every key block kept by
// EITHER of them, ascending, and for each of its two 64-key tiles t = 2 kb, 2 kb + 1 with
// 64 t < N, one entry:  t | (upper does not keep kb) << 30 | (lower does not keep kb) << 31.
// Returns the number of entries; col_idx may be null (count only).
// -------------------------------------------------------------------------------------------------
int64_t oracle_mask_to_index_64x128(const uint32_t* bitmask, int L, int H, int N,
                                    int32_t* row_ptr, uint32_t* col_idx) {
    const int nq64 = (N + 63) / 64, nk128 = (N + 127) / 128, nq128 = (N + 127) / 128;
    const int words = (nk128 + 31) / 32;
    int64_t nnz = 0, R = 0;
    row_ptr[0] = 0;
    for (int l = 0; l < L; ++l)
        for (int h = 0; h < H; ++h)
            for (int qb = 0; qb < nq128; ++qb, ++R) {
                const uint32_t* up = bitmask + ((static_cast<int64_t>(l) * H + h) * nq64 + 2 * qb) * words;
                const uint32_t* lo = (2 * qb + 1 < nq64) ? up + words : nullptr;
                for (int kb = 0; kb < nk128; ++kb) {
                    const bool ku = mask_bit(up, kb), kl = lo != nullptr && mask_bit(lo, kb);
                    if (!ku && !kl) continue;
                    for (int t = 2 * kb; t <= 2 * kb + 1; ++t) {
                        if (64 * t >= N) continue;
                        if (col_idx)
                            col_idx[nnz] = static_cast<uint32_t>(t) | (ku ? 0u : 1u << 30) | (kl ? 0u : 1u << 31);
                        ++nnz;
                    }
                }
                row_ptr[R + 1] = static_cast<int32_t>(nnz);
            }
    return nnz;
}

// -------------------------------------------------------------------------------------------------
// f-4  The same two decodes with 16-bit entries (SURVEY section 8 f-4 "uint16 col_idx"; the index is
// what the mask decode writes and the attention kernel reads, "loaded and used
// directly": at 25 % density the entries are 5.24 of the 5.9 MB a 480p layer's decode moves, and a
// key-block index of the paper's shapes (512 / 1182) fits 16 bits).  Written out on their own, one
// bit at a time like the 32-bit forms.  Plain geometry: entry = kb, nk <= 65536.  64 x 128 geometry:
// entry = t | (upper does not keep kb) << 14 | (lower does not keep kb) << 15, tiles t < 16384.
// Return -1 (nothing written) when an index does not fit.
// -------------------------------------------------------------------------------------------------
int64_t oracle_mask_to_index_u16(const uint32_t* bitmask, int L, int H, int nq, int nk,
                                 int32_t* row_ptr, uint16_t* col_idx) {
    if (nk > 65536) return -1;
    const int words = (nk + 31) / 32;
    int64_t nnz = 0, r = 0;
    row_ptr[0] = 0;
    for (int l = 0; l < L; ++l)
        for (int h = 0; h < H; ++h)
            for (int qb = 0; qb < nq; ++qb, ++r) {
                for (int kb = 0; kb < nk; ++kb) {
                    const uint32_t word = bitmask[r * words + kb / 32];
                    if ((word >> (kb % 32)) & 1u) {
                        if (col_idx) col_idx[nnz] = static_cast<uint16_t>(kb);
                        ++nnz;
                    }
                }
                row_ptr[r + 1] = static_cast<int32_t>(nnz);
            }
    return nnz;
}

int64_t oracle_mask_to_index_64x128_u16(const uint32_t* bitmask, int L, int H, int N,
                                        int32_t* row_ptr, uint16_t* col_idx) {
    const int nq64 = (N + 63) / 64, nk128 = (N + 127) / 128, nq128 = (N + 127) / 128;
    if ((N + 63) / 64 > 16384) return -1;
    const int words = (nk128 + 31) / 32;
    int64_t nnz = 0, R = 0;
    row_ptr[0] = 0;
    for (int l = 0; l < L; ++l)
        for (int h = 0; h < H; ++h)
            for (int qb = 0; qb < nq128; ++qb, ++R) {
                const int64_t upper = ((static_cast<int64_t>(l) * H + h) * nq64 + 2 * qb) * words;
                const bool has_lower = 2 * qb + 1 < nq64;
                for (int kb = 0; kb < nk128; ++kb) {
                    const bool ku = (bitmask[upper + kb / 32] >> (kb % 32)) & 1u;
                    const bool kl = has_lower && ((bitmask[upper + words + kb / 32] >> (kb % 32)) & 1u);
                    if (!ku && !kl) continue;
                    for (int t = 2 * kb; t <= 2 * kb + 1; ++t) {
                        if (64 * t >= N) continue;
                        if (col_idx)
                            col_idx[nnz] = static_cast<uint16_t>(t | (ku ? 0 : 1 << 14) | (kl ? 0 : 1 << 15));
                        ++nnz;
                    }
                }
                row_ptr[R + 1] = static_cast<int32_t>(nnz);
            }
    return nnz;
}

// -------------------------------------------------------------------------------------------------
// a-2 / a-3  Block-sparse attention.  PAPER.md:L97: "skip pruned block pairs and
// evaluate only the retained ones in QK^T, softmax, and PV" => the softmax is normalised over the
// retained keys only (R5).  For head h and query i (qb = i / 128):
//     J(i) = { j < N : bit(h, qb, j / 64) = 1 }           keys >= N are masked (R6)
//     s_j  = scale * sum_c Q[i,h,c] K[j,h,c]
//     m = max_j s_j ;  p_j = exp(s_j - m) ;  l = sum_j p_j
//     O[i,h,:] = (sum_j p_j V[j,h,:]) / l                  J(i) empty => O = 0 (R7)
// Everything in fp64 on the exact values of the input bytes.  dtype 0: bf16 bits; dtype 2: IEEE
// binary16 bits (the paper's non-quantised path); dtype 1: e4m3
// codes dequantised as code * scale (q_scale[b][h][i/128], k_scale[b][h][j/128], v_scale[b][h][c];
// R10).  The oracle reads the BITMASK, never a CSR, so a decode bug cannot hide.
//
// Items: item t computes batch item_b[t], head item_h[t], query block item_qb[t] and writes
// out[t][r][c] (r < 128, c < d) as doubles; rows with 128*qb + r >= N are written as 0.
// bitmask is one layer: [H][nq][words].  Strides are in elements; the last dim is contiguous.
// If weight_sum != null, weight_sum[t][r] receives sum_j p_j / l (must be 1; 0 for an empty row).
// If lse != null, lse[t][r] receives the row's log-sum-exp m + log(l) = log sum_{j in J} exp(s_j)
// (natural log; -inf for an empty row or a row >= N).
// -------------------------------------------------------------------------------------------------
void oracle_block_sparse_attn(const void* Q, const void* K, const void* V, int dtype,
                              int B, int H, int N, int d,
                              int64_t q_sb, int64_t q_sn, int64_t q_sh,
                              int64_t k_sb, int64_t k_sn, int64_t k_sh,
                              int64_t v_sb, int64_t v_sn, int64_t v_sh,
                              const float* q_scale, const float* k_scale, const float* v_scale,
                              const uint32_t* bitmask, double scale,
                              int n_items, const int32_t* item_b, const int32_t* item_h,
                              const int32_t* item_qb, double* out, double* weight_sum,
                              double* lse, int n_threads, int n_first, double beta, int bq, int bk) {
    (void)B;
    // block geometry: 128 x 64 (BASELINE.json north_star) unless the caller asks for the paper's own
    // 64 x 128; it only decides which keys a query row retains
    const int BQ = bq > 0 ? bq : ::BQ, BK = bk > 0 ? bk : ::BK;
    const int nq = (N + BQ - 1) / BQ;
    const int nk = (N + BK - 1) / BK;
    const int words = (nk + 31) / 32;
    const int nsb = (N + 127) / 128;  // scale blocks of 128 tokens (R10)

#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel
    {
        std::vector<double> q(d), s, acc(d), Kd, Vd;
        std::vector<int> js;
#pragma omp for schedule(dynamic, 1)
        for (int t = 0; t < n_items; ++t) {
            const int b = item_b[t], h = item_h[t], qb = item_qb[t];
            const uint32_t* mrow = bitmask + (static_cast<int64_t>(h) * nq + qb) * words;
            // exact value of one input element as a double (dequantised for FP8, R10)
            auto load = [&](const void* base, int64_t off, double sc) -> double {
                if (dtype == 0) return bf16_to_double(static_cast<const uint16_t*>(base)[off]);
                if (dtype == 2) return f16_to_double(static_cast<const uint16_t*>(base)[off]);
                return e4m3_to_double(static_cast<const uint8_t*>(base)[off]) * sc;
            };
            // J = retained, valid keys of this query block (the same set for its 128 rows)
            js.clear();
            for (int kb = 0; kb < nk; ++kb)
                if (mask_bit(mrow, kb))
                    for (int j = kb * BK; j < (kb + 1) * BK && j < N; ++j) js.push_back(j);
            const size_t nj = js.size();
            // the K and V rows of J, converted to fp64 once (a conversion, not a reordering)
            Kd.resize(nj * d);
            Vd.resize(nj * d);
            for (size_t x = 0; x < nj; ++x) {
                const int j = js[x];
                const double ks = dtype == 1 ? static_cast<double>(
                    k_scale[(static_cast<int64_t>(b) * H + h) * nsb + j / 128]) : 1.0;
                for (int c = 0; c < d; ++c) {
                    const double vs = dtype == 1 ? static_cast<double>(
                        v_scale[(static_cast<int64_t>(b) * H + h) * d + c]) : 1.0;
                    // first-frame key enhancement, eq. (1): K[:, 0:N0] <- beta K[:, 0:N0]
                    const double kf = j < n_first ? beta : 1.0;
                    Kd[x * d + c] = kf * load(K, b * k_sb + j * k_sn + h * k_sh + c, ks);
                    Vd[x * d + c] = load(V, b * v_sb + j * v_sn + h * v_sh + c, vs);
                }
            }
            s.resize(nj);

            for (int r = 0; r < BQ; ++r) {
                double* o = out + (static_cast<int64_t>(t) * BQ + r) * d;
                const int i = qb * BQ + r;
                for (int c = 0; c < d; ++c) o[c] = 0.0;
                if (weight_sum) weight_sum[static_cast<int64_t>(t) * BQ + r] = 0.0;
                if (lse) lse[static_cast<int64_t>(t) * BQ + r] = -std::numeric_limits<double>::infinity();
                if (i >= N || nj == 0) continue;

                const double qs = dtype == 1 ? static_cast<double>(
                    q_scale[(static_cast<int64_t>(b) * H + h) * nsb + i / 128]) : 1.0;
                for (int c = 0; c < d; ++c) q[c] = load(Q, b * q_sb + i * q_sn + h * q_sh + c, qs);

                double m = -std::numeric_limits<double>::infinity();
                for (size_t x = 0; x < nj; ++x) {
                    double dot = 0.0;
                    for (int c = 0; c < d; ++c) dot += q[c] * Kd[x * d + c];
                    s[x] = scale * dot;
                    if (s[x] > m) m = s[x];
                }
                double l = 0.0;
                for (int c = 0; c < d; ++c) acc[c] = 0.0;
                for (size_t x = 0; x < nj; ++x) {
                    const double p = std::exp(s[x] - m);
                    l += p;
                    for (int c = 0; c < d; ++c) acc[c] += p * Vd[x * d + c];
                }
                for (int c = 0; c < d; ++c) o[c] = acc[c] / l;
                if (lse) lse[static_cast<int64_t>(t) * BQ + r] = m + std::log(l);
                if (weight_sum) {
                    double w = 0.0;
                    for (size_t x = 0; x < nj; ++x) w += std::exp(s[x] - m) / l;
                    weight_sum[static_cast<int64_t>(t) * BQ + r] = w;
                }
            }
        }
    }
}

// -------------------------------------------------------------------------------------------------
// a-4  FP8 quantisation pre-pass (readings R10/R11; PAPER.md:L97 says only "FP8
// quantization").  Q and K: one fp32 scale per (b, h, block of 128 tokens) over all d channels;
// V: one fp32 scale per (b, h, channel) over all tokens.  amax over valid tokens only.
//     s  = max(amax, 1e-12f) / 448.0f              (fp32 division)
//     x8 = e4m3_rne_sat( x / s )                   (fp32 division, then RNE, saturate at 448)
// The decision arithmetic is fp32 on both sides (the kernel's precision), so codes are bit-exact.
// Inputs are bf16 bits [B][N][H][d] with element strides; outputs are packed [B][N][H][d] codes.
// -------------------------------------------------------------------------------------------------
void oracle_quantize_fp8(const uint16_t* Q, const uint16_t* K, const uint16_t* V,
                         int B, int H, int N, int d,
                         int64_t q_sb, int64_t q_sn, int64_t q_sh,
                         int64_t k_sb, int64_t k_sn, int64_t k_sh,
                         int64_t v_sb, int64_t v_sn, int64_t v_sh,
                         uint8_t* q8, uint8_t* k8, uint8_t* v8,
                         float* q_scale, float* k_scale, float* v_scale) {
    const int nsb = (N + 127) / 128;
    auto f = [](uint16_t b) { return static_cast<float>(bf16_to_double(b)); };
    auto out_off = [&](int b, int n, int h, int c) {
        return ((static_cast<int64_t>(b) * N + n) * H + h) * d + c;
    };
    for (int which = 0; which < 2; ++which) {  // 0: Q, 1: K
        const uint16_t* X = which ? K : Q;
        const int64_t sb = which ? k_sb : q_sb, sn = which ? k_sn : q_sn, sh = which ? k_sh : q_sh;
        uint8_t* X8 = which ? k8 : q8;
        float* S = which ? k_scale : q_scale;
#pragma omp parallel for collapse(2) schedule(static)
        for (int bh = 0; bh < B * H; ++bh)
            for (int blk = 0; blk < nsb; ++blk) {
                const int b = bh / H, h = bh % H;
                float amax = 0.f;
                for (int n = blk * 128; n < (blk + 1) * 128 && n < N; ++n)
                    for (int c = 0; c < d; ++c)
                        amax = std::fmax(amax, std::fabs(f(X[b * sb + n * sn + h * sh + c])));
                const float s = std::fmax(amax, 1e-12f) / 448.0f;
                S[static_cast<int64_t>(bh) * nsb + blk] = s;
                for (int n = blk * 128; n < (blk + 1) * 128 && n < N; ++n)
                    for (int c = 0; c < d; ++c)
                        X8[out_off(b, n, h, c)] =
                            float_to_e4m3_rne_sat(f(X[b * sb + n * sn + h * sh + c]) / s);
            }
    }
#pragma omp parallel for collapse(2) schedule(static)
    for (int bh = 0; bh < B * H; ++bh)
        for (int c = 0; c < d; ++c) {
            const int b = bh / H, h = bh % H;
            float amax = 0.f;
            for (int n = 0; n < N; ++n)
                amax = std::fmax(amax, std::fabs(f(V[b * v_sb + n * v_sn + h * v_sh + c])));
            const float s = std::fmax(amax, 1e-12f) / 448.0f;
            v_scale[static_cast<int64_t>(bh) * d + c] = s;
            for (int n = 0; n < N; ++n)
                v8[out_off(b, n, h, c)] =
                    float_to_e4m3_rne_sat(f(V[b * v_sb + n * v_sn + h * v_sh + c]) / s);
        }
}

// Element-wise helpers exposed so the tests can pin the two conversions on their own.
double oracle_e4m3_to_double(uint8_t code) { return e4m3_to_double(code); }
double oracle_f16_to_double(uint16_t bits) { return f16_to_double(bits); }
uint8_t oracle_float_to_e4m3(float x) { return float_to_e4m3_rne_sat(x); }

// -------------------------------------------------------------------------------------------------
// a-0  Retrieval (reading R15).  PAPER.md:L87: k-NN under cosine similarity over the
// request embeddings; if the top neighbour's similarity reaches the threshold tau its masks are
// used (tau = 0.4), else fall back.  Embeddings are unit-norm, so cosine = dot
// product.  fp64 dot products; ties -> lowest index; hit = (best_sim >= tau).
// -------------------------------------------------------------------------------------------------
void oracle_retrieve_top1(const float* bank, int n, int dim, const float* query, double tau,
                          int32_t* best_idx, double* best_sim, int32_t* hit) {
    int best = -1;
    double bs = -std::numeric_limits<double>::infinity();
    for (int j = 0; j < n; ++j) {
        double dot = 0.0;
        for (int c = 0; c < dim; ++c)
            dot += static_cast<double>(bank[static_cast<int64_t>(j) * dim + c]) *
                   static_cast<double>(query[c]);
        if (dot > bs) { bs = dot; best = j; }
    }
    *best_idx = best;
    *best_sim = bs;
    *hit = (bs >= tau) ? 1 : 0;
}

// -------------------------------------------------------------------------------------------------
// NEXT row f-1  Block-pair visit refreshing (PAPER.md:L93 (1), L153 layer_flash = 8; reading R17).
// A visited map V[h,q,k] records whether the pair was activated by the mask in the current layer
// group of `group` consecutive layers; "when executing the last layer of the group, any block pair
// that is still unvisited is forced into the sparse mask"; the map is reset at the start of the next
// group.  Followed step by step: walk the layers in order, keep an explicit visited map, and at
// the last layer of each COMPLETE group force the unvisited pairs.  (A trailing partial group has
// no "last layer of the group" and is left unchanged.)  mask is [L][H][nq][words], updated in
// place; pad bits (kb >= nk) of forced words are left as they were.
// -------------------------------------------------------------------------------------------------
void oracle_visit_refresh(uint32_t* mask, int L, int H, int nq, int nk, int group) {
    const int words = (nk + 31) / 32;
    const int64_t per_layer = static_cast<int64_t>(H) * nq * words;
    std::vector<uint8_t> visited(static_cast<size_t>(H) * nq * nk);
    for (int l = 0; l < L; ++l) {
        const int pos = l % group;
        if (pos == 0) std::fill(visited.begin(), visited.end(), 0);
        uint32_t* ml = mask + l * per_layer;
        const bool last = (pos == group - 1);
        for (int h = 0; h < H; ++h)
            for (int qb = 0; qb < nq; ++qb) {
                uint32_t* row = ml + (static_cast<int64_t>(h) * nq + qb) * words;
                uint8_t* vis = visited.data() + (static_cast<size_t>(h) * nq + qb) * nk;
                for (int kb = 0; kb < nk; ++kb) {
                    if (mask_bit(row, kb)) vis[kb] = 1;
                    if (last && !vis[kb]) {
                        row[kb >> 5] |= (1u << (kb & 31));
                        vis[kb] = 1;
                    }
                }
            }
    }
}

// -------------------------------------------------------------------------------------------------
// Mask construction from a dense pass ("in the dense case we select a block-level mask
// from its attention map via top-p with a top-k floor"; L73 "coverage: the fraction of the target's
// true token-level attention mass that falls within the blocks it selects"; L93 (2) min_top_k: "every
// head retains at least a fraction k_min of its key blocks"; L153 defaults top_p 0.95 / 0.9,
// min_top_k 0.1 / 0.0).  Readings R21-R23 in DESIGN.md section 3.
// -------------------------------------------------------------------------------------------------

// Block mass of the TRUE (dense) attention: mass[h][qb][kb] = sum over queries i of q-block qb and
// keys j of k-block kb of softmax_j(scale * q_i . k_j), all N keys retained, fp64, two-pass softmax.
// Q, K: bf16 bits [B][N][H][d] (element strides); mass: double [B][H][nq][nk].  Each row of a
// q-block contributes exactly 1, so a q-block's masses sum to its number of valid rows.
void oracle_block_mass(const uint16_t* Q, const uint16_t* K, int B, int H, int N, int d,
                       int64_t q_sb, int64_t q_sn, int64_t q_sh, int64_t k_sb, int64_t k_sn,
                       int64_t k_sh, double scale, double* mass, int n_sel, const int32_t* sel_qb,
                       int n_threads, int bq, int bk) {
    // n_sel > 0: only the query blocks listed in sel_qb are computed (the others stay as they are)
    // block geometry bq x bk: 128 x 64 (default, bq <= 0) or the paper's 64 x 128
    const int BQ = bq > 0 ? bq : 128, BK = bk > 0 ? bk : 64;
    const int nq = (N + BQ - 1) / BQ, nk = (N + BK - 1) / BK;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
    const int64_t total = static_cast<int64_t>(B) * H * nq;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t it = 0; it < total; ++it) {
        const int qb = static_cast<int>(it % nq);
        const int h = static_cast<int>((it / nq) % H);
        const int b = static_cast<int>(it / (static_cast<int64_t>(nq) * H));
        if (n_sel > 0) {
            bool wanted = false;
            for (int t = 0; t < n_sel; ++t) wanted = wanted || sel_qb[t] == qb;
            if (!wanted) continue;
        }
        double* out = mass + it * nk;
        for (int kb = 0; kb < nk; ++kb) out[kb] = 0.0;
        std::vector<double> kd(static_cast<size_t>(N) * d), s(N), q(d);
        for (int j = 0; j < N; ++j)
            for (int c = 0; c < d; ++c) kd[static_cast<size_t>(j) * d + c] = bf16_to_double(K[b * k_sb + j * k_sn + h * k_sh + c]);
        for (int i = qb * BQ; i < N && i < qb * BQ + BQ; ++i) {
            for (int c = 0; c < d; ++c) q[c] = bf16_to_double(Q[b * q_sb + i * q_sn + h * q_sh + c]);
            double m = -std::numeric_limits<double>::infinity();
            for (int j = 0; j < N; ++j) {
                double acc = 0.0;
                for (int c = 0; c < d; ++c) acc += q[c] * kd[static_cast<size_t>(j) * d + c];
                s[j] = scale * acc;
                if (s[j] > m) m = s[j];
            }
            double l = 0.0;
            for (int j = 0; j < N; ++j) {
                s[j] = std::exp(s[j] - m);
                l += s[j];
            }
            for (int j = 0; j < N; ++j) out[j / BK] += s[j] / l;
        }
    }
}

// Top-p with a top-k floor, one row of nk block masses at a time (R22): the masses (fp32, >= 0) are
// taken in units of 2^-24 (q = floor(mass * 2^24), an exact integer), so that sums do not depend on
// the order of addition; blocks are ranked by q descending, ties by index ascending; the row keeps
// the shortest prefix of that ranking whose q-sum reaches ceil(top_p * total q), and never fewer
// than ceil(min_top_k * nk) blocks.  A row without any mass keeps only the floor.
// mass: float [rows][nk] -> bitmask uint32 [rows][words] (pad bits 0), kept[rows] = blocks kept.
void oracle_mask_from_mass(const float* mass, int64_t rows, int nk, double top_p, double min_top_k,
                           uint32_t* bitmask, int32_t* kept) {
    const int words = (nk + 31) / 32;
    int n_floor = static_cast<int>(std::ceil(min_top_k * static_cast<double>(nk)));
    if (n_floor < 0) n_floor = 0;
    if (n_floor > nk) n_floor = nk;
    std::vector<uint64_t> q(nk);
    std::vector<int> order(nk);
    for (int64_t r = 0; r < rows; ++r) {
        const float* mr = mass + r * nk;
        uint64_t total = 0;
        for (int k = 0; k < nk; ++k) {
            q[k] = static_cast<uint64_t>(std::floor(static_cast<double>(mr[k]) * 16777216.0));
            total += q[k];
            order[k] = k;
        }
        // selection sort into (q descending, index ascending): plain and obviously right
        for (int a = 0; a < nk; ++a) {
            int best = a;
            for (int c = a + 1; c < nk; ++c) {
                const int x = order[c], y = order[best];
                if (q[x] > q[y] || (q[x] == q[y] && x < y)) best = c;
            }
            const int t = order[a];
            order[a] = order[best];
            order[best] = t;
        }
        const uint64_t target = static_cast<uint64_t>(std::ceil(top_p * static_cast<double>(total)));
        int n_p = 0;
        if (total > 0) {
            uint64_t acc = 0;
            while (n_p < nk && acc < target) acc += q[order[n_p++]];
        }
        const int n = n_p > n_floor ? n_p : n_floor;
        uint32_t* br = bitmask + r * words;
        for (int w = 0; w < words; ++w) br[w] = 0u;
        for (int a = 0; a < n; ++a) br[order[a] >> 5] |= (1u << (order[a] & 31));
        if (kept) kept[r] = n;
    }
}

// Coverage of a mask on a mass map, per head: sum of the masses of the kept blocks
// over the sum of all masses.  mass: float [heads][nq][nk], bitmask [heads][nq][words].
void oracle_mask_coverage(const float* mass, const uint32_t* bitmask, int heads, int nq, int nk,
                          double* coverage) {
    const int words = (nk + 31) / 32;
    for (int h = 0; h < heads; ++h) {
        double in = 0.0, all = 0.0;
        for (int qb = 0; qb < nq; ++qb) {
            const int64_t r = static_cast<int64_t>(h) * nq + qb;
            for (int kb = 0; kb < nk; ++kb) {
                const double m = static_cast<double>(mass[r * nk + kb]);
                all += m;
                if (mask_bit(bitmask + r * words, kb)) in += m;
            }
        }
        coverage[h] = all > 0.0 ? in / all : 0.0;
    }
}

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
