/* chorus.h — C ABI of libchorus.so: the B200-native (sm_100a) hot path of Chorus II's
 * cross-request sparsity reuse (arxiv/paper_2606_25040).
 *
 * The path: a new request looks up the most similar historical request; if it is
 * similar enough, that request's cached block masks "are loaded and used directly by the current
 * block sparse attention", whose kernels "skip pruned block pairs and evaluate only the retained
 * ones in QK^T, softmax, and PV".  This library is that path on one GPU:
 *
 *   chorus_retrieve_top1          cosine top-1 over stored request embeddings, threshold tau   (L87, L149)
 *   chorus_visit_refresh          block-pair visit refreshing over groups of layers            (L93 (1), L153)
 *   chorus_mask_to_index          stored block bitmask  ->  CSR of kept key blocks per query block (L81, L87)
 *   chorus_quantize_fp8           bf16 Q/K/V -> e4m3 + scales for the FP8 backend              (L97)
 *   chorus_block_sparse_attn_fwd  block-sparse attention forward, BF16, FP16 or FP8 e4m3       (L97)
 *   chorus_block_sparse_attn_fwd_lse   the same, also writing the rows' log-sum-exp            (L87)
 *   chorus_block_sparse_attn_fwd_first_frame   the same with first-frame key enhancement  (L109-114 eq. 1)
 *   chorus_mask_to_index_64x128 / chorus_block_sparse_attn_fwd_64x128
 *                                 the same path for masks in the paper's own 64 x 128 block geometry (L153)
 * and, for the historical request whose masks get cached, and for sequence-parallel groups:
 *   chorus_block_mass / chorus_mask_from_mass / chorus_mask_coverage
 *                                 dense attention mass per block -> top-p mask with a top-k floor
 *                                 -> coverage                                                  (L73, L81, L93 (2))
 *   chorus_head_costs / chorus_schedule_heads   per-head cost and greedy head -> rank schedule (L95, appendix A)
 *   chorus_gather_heads / chorus_scatter_heads  the local copies around the Ulysses all-to-all   (L95, appendix A)
 *
 * Conventions (all entry points)
 *   - Plain C: pointers and sizes only.  "device" = pointer into CUDA device memory of the current
 *     device; "host" = ordinary host memory.  Every buffer is owned by the caller; the library
 *     allocates nothing that outlives a call, keeps no global state (beyond cached device attributes),
 *     and never frees caller memory.
 *   - All work is enqueued on `cuda_stream` (a cudaStream_t passed as void*; NULL = default stream)
 *     and the call returns without synchronising.
 *   - Errors: an integer status, never an exception.  Argument errors are detected on the host
 *     before anything is launched.  chorus_last_error() gives a thread-local message.
 *   - The kernels' tile is fixed: 128 query rows x 64 keys, head_dim 128 (BASELINE.json north_star).
 *     Masks in the paper's own 64 x 128 block geometry go through the *_64x128
 *     entry points, which serve them exactly on the same tiles.
 *   - There is no CPU fallback: without a CUDA device every compute entry point returns
 *     CHORUS_ERR_CUDA.
 */
#ifndef CHORUS_H_
#define CHORUS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CHORUS_BLOCK_Q 128 /* query rows per mask block */
#define CHORUS_BLOCK_K 64  /* keys per mask block       */
#define CHORUS_HEAD_DIM 128

typedef enum {
    CHORUS_OK = 0,
    CHORUS_ERR_INVALID_ARG = 1, /* null / misaligned pointer, inconsistent sizes            */
    CHORUS_ERR_UNSUPPORTED = 2, /* valid request the library does not implement (d != 128)  */
    CHORUS_ERR_CAPACITY = 3,    /* a size does not fit (nnz > INT32_MAX, workspace too small) */
    CHORUS_ERR_CUDA = 4         /* a CUDA call failed; see chorus_last_error()              */
} chorus_status;

typedef enum { CHORUS_BF16 = 0, CHORUS_FP8_E4M3 = 1, CHORUS_FP16 = 2 } chorus_dtype;

/* ---------------------------------------------------------------------------------------------
 * Mask decode ("stored, indexed by denoising step, transformer layer, and attention
 * head"; L87 "loaded and used directly by the current block sparse attention"; L93: the mask is
 * binary per (head, q-block, k-block)).
 *
 * bitmask   device, uint32 [L][H][nq_blk][words], words = ceil(nk_blk / 32), 4-byte aligned.
 *           Key block kb is bit (kb & 31) (bit 0 = LSB) of word kb >> 5.  Bits >= nk_blk of the
 *           last word are ignored (they need not be zero).
 * row_ptr   device, int32 [L*H*nq_blk + 1].  row_ptr[0] = 0; row r = (l*H + h)*nq_blk + qb owns
 *           col_idx[row_ptr[r] .. row_ptr[r+1]).  Offsets are absolute over the whole mask set.
 * col_idx   device, int32 [col_cap], kept key-block indices, ascending within each row.
 *           NULL = count only (row_ptr is still filled).  Entries beyond col_cap are never
 *           written; the caller sizes col_idx either at an upper bound or from a count-only call
 *           followed by one 4-byte read of row_ptr[L*H*nq_blk].
 * workspace device scratch.  Call with workspace == NULL to get the required size in
 *           *workspace_bytes (nothing is launched); otherwise *workspace_bytes is the size given.
 * Result is unique (ascending order), so it is compared bit-exactly with the oracle.
 * Errors: INVALID_ARG (null bitmask/row_ptr/workspace_bytes, L/H/nq_blk/nk_blk <= 0, col_cap < 0),
 *         CAPACITY (L*H*nq_blk*nk_blk > INT32_MAX, or workspace too small), CUDA.
 * ------------------------------------------------------------------------------------------- */
chorus_status chorus_mask_to_index(const uint32_t* bitmask, int L, int H, int nq_blk, int nk_blk,
                                   int32_t* row_ptr, int32_t* col_idx, int64_t col_cap,
                                   void* workspace, size_t* workspace_bytes, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * chorus_mask_to_index_static: chorus_mask_to_index (same operation; same bitmask,
 * row_ptr, col_idx, col_cap and result, bit for bit) for callers that cannot allocate or hand in a
 * workspace: code under CUDA graph capture, serving loops and harnesses that forbid cudaMalloc.
 * The call allocates nothing (no cudaMalloc / cudaFree, no allocating library routine): the kernel's
 * scratch - one 8-byte status word per tile of the mask - is a file-scope device array of
 * CHORUS_STATIC_DECODE_MAX_TILES + 1 words (128 KB), which every GPU that loads the library holds until
 * exit.  Limit: the mask set may have at most CHORUS_STATIC_DECODE_MAX_WORDS = 2^24 32-bit words
 * (L*H*nq_blk*ceil(nk_blk/32); 64 MiB of bitmask: 2.5 mask sets of 40 layers x 40 heads at 480p);
 * larger sets are rejected with CHORUS_ERR_CAPACITY and nothing is launched.
 * All calls on a device share the array: calls that overlap on the GPU (different streams, or
 * different threads without ordering) RACE; calls ordered on one stream are fine.  The array keeps the
 * previous call's contents; each call clears the words it uses on its own stream first.
 * Errors: INVALID_ARG (null bitmask/row_ptr, sizes <= 0, col_cap < 0, misaligned pointers),
 *         CAPACITY (L*H*nq_blk*nk_blk > INT32_MAX, or more words than the limit), CUDA.
 * ------------------------------------------------------------------------------------------- */
#define CHORUS_STATIC_DECODE_MAX_TILES 16384
#define CHORUS_STATIC_DECODE_MAX_WORDS (1 << 24)
chorus_status chorus_mask_to_index_static(const uint32_t* bitmask, int L, int H, int nq_blk, int nk_blk,
                                          int32_t* row_ptr, int32_t* col_idx, int64_t col_cap,
                                          void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Block-pair visit refreshing (PAPER.md:L93 (1); layer_flash = 8 at L153).  Within each group of
 * `group` consecutive layers a visited map V[h,q,k] records the block pairs activated so far;
 * "when executing the last layer of the group, any block pair that is still unvisited is forced
 * into the sparse mask"; the map is reset at the start of the next group.  In place:
 *     mask[g*group + group-1] |= ~(mask[g*group] | ... | mask[g*group + group-2])
 * for every complete group g; a trailing partial group is left unchanged.  Pad bits (>= nk_blk)
 * of the forced layer are left as they were.
 * bitmask   device, uint32 [L][H][nq_blk][words], updated in place.
 * Errors: INVALID_ARG (null, sizes <= 0, group < 1), CUDA.
 * ------------------------------------------------------------------------------------------- */
chorus_status chorus_visit_refresh(uint32_t* bitmask, int L, int H, int nq_blk, int nk_blk,
                                   int group, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Block-sparse attention forward.  For batch b, head h, query i (qb = i / 128):
 *     J(i)   = { j < N : key block j/64 is in CSR row (h, qb) }        keys >= N are masked
 *     O[i,:] = sum_{j in J(i)} softmax_j(scale * <Q[i], K[j]>) V[j,:]   softmax over J(i) only
 * A row with no kept block gives O = 0.  Query rows >= N are not written.
 *
 * Shapes/strides: Q, K, V, O are [B][N][H][d]-indexed tensors with arbitrary element strides for
 * B, N, H (so [B][H][N][d] storage also works); the last dimension (d = 128) is contiguous.
 * ------------------------------------------------------------------------------------------- */
typedef struct {
    int B, H, N, d; /* d must be 128 */
    int64_t q_stride_b, q_stride_n, q_stride_h; /* in elements */
    int64_t k_stride_b, k_stride_n, k_stride_h;
    int64_t v_stride_b, v_stride_n, v_stride_h;
    int64_t o_stride_b, o_stride_n, o_stride_h;
} chorus_attn_shape;

/* FP8 scales (device, float).  Dequantised values are code * scale:
 *   Q^[i,c] = q8[i,c] * q_scale[b][h][i/128]     K^[j,c] = k8[j,c] * k_scale[b][h][j/128]
 *   V^[j,c] = v8[j,c] * v_scale[b][h][c]
 * (per-128x128-block Q/K scales, per-channel V scales: BASELINE.json configs[2]). */
typedef struct {
    const float* q_scale; /* [B][H][ceil(N/128)] */
    const float* k_scale; /* [B][H][ceil(N/128)] */
    const float* v_scale; /* [B][H][d]           */
} chorus_fp8_scales;

/* Q, K, V   device; dtype BF16: bf16 elements; dtype FP16: IEEE half elements (the paper's
 *           non-quantised path); dtype FP8_E4M3: e4m3 (fn) codes.  Base pointers
 *           16-byte aligned; strides multiples of 8 (bf16) / 16 (fp8) elements (TMA rules).
 * row_ptr   device, int32, points at THIS layer's first row: H*nq_blk + 1 readable entries,
 *           nq_blk = ceil(N/128); the same mask is used for every b.
 * col_idx   device, the base pointer that row_ptr's absolute offsets index into.  Indices must
 *           lie in [0, ceil(N/64)) and ascend within a row (what chorus_mask_to_index produces);
 *           anything else is undefined behaviour (an index with the per-half flag bits of
 *           chorus_mask_to_index_64x128 belongs to chorus_block_sparse_attn_fwd_64x128 only).
 * scale     multiplies QK^T before the softmax (1/sqrt(128) in all workloads).  Must be positive and
 *           finite (the row maximum is taken on the raw scores): anything else is INVALID_ARG, here
 *           and in chorus_block_mass.
 * O         device, bf16 for dtype BF16 and FP8_E4M3, fp16 for dtype FP16; 16-byte aligned, strides
 *           multiples of 8 elements.
 * fp8       non-NULL iff dtype == CHORUS_FP8_E4M3.
 * Accuracy against the fp64 oracle on the same input bytes (BASELINE.json north_star):
 *           BF16 and FP16: max|err| <= 2e-2, mean|err| <= 2e-3;  FP8: max|err| <= 8e-2, cosine >= 0.995.
 * Errors: INVALID_ARG (null pointer, misalignment, bad strides, N/H/B <= 0, fp8/dtype mismatch),
 *         UNSUPPORTED (d != 128, unknown dtype), CUDA.
 */
chorus_status chorus_block_sparse_attn_fwd(const void* Q, const void* K, const void* V,
                                           const int32_t* row_ptr, const int32_t* col_idx,
                                           float scale, chorus_dtype dtype, void* O,
                                           const chorus_attn_shape* shape,
                                           const chorus_fp8_scales* fp8, void* cuda_stream);

/* The same call with one more output: lse[b][h][i] = log sum_{j in J(i)} exp(scale * <Q[i], K[j]>)
 * (natural log, fp32, PACKED [B][H][N]; -inf for a row with no kept block).  With a full mask this
 * is the row statistic of the dense attention that chorus_block_mass can reuse (the
 * historical request records its mask "as a by-product" of its own attention).  For FP8 inputs the
 * scores are those of the dequantised Q and K.  lse == NULL behaves like the call above.
 * Accuracy against the fp64 oracle: |err| <= 2e-3 (bf16), 2e-2 (fp8). */
chorus_status chorus_block_sparse_attn_fwd_lse(const void* Q, const void* K, const void* V,
                                               const int32_t* row_ptr, const int32_t* col_idx,
                                               float scale, chorus_dtype dtype, void* O,
                                               const chorus_attn_shape* shape,
                                               const chorus_fp8_scales* fp8, float* lse,
                                               void* cuda_stream);

/* The same call with first-frame key enhancement fused in (eq. (1):
 * "K[:, 0:N0] <- beta_step K[:, 0:N0] ... leaving Q and V unchanged", N0 = tokens of the first
 * frame): the scores of keys 0 .. n_first-1 are multiplied by beta inside the kernel (the scale
 * factor of a key tile that lies in the first frame, a per-column factor in the one tile that
 * straddles n_first), so K is neither rewritten nor re-rounded: the result is that of the plain call
 * on keys scaled in exact arithmetic (R25).  lse, if given, is that of the scaled scores.
 *   n_first  >= 0 (values above N act as N; 0 = no scaling);  beta  > 0 and finite.
 * n_first == 0 or beta == 1 runs the plain kernel.  Same accuracy bounds as the plain call.
 * Errors: as above, plus INVALID_ARG for n_first < 0 or beta not positive and finite. */
chorus_status chorus_block_sparse_attn_fwd_first_frame(const void* Q, const void* K, const void* V,
                                                       const int32_t* row_ptr, const int32_t* col_idx,
                                                       float scale, chorus_dtype dtype, void* O,
                                                       const chorus_attn_shape* shape,
                                                       const chorus_fp8_scales* fp8, float* lse,
                                                       int n_first, float beta, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Masks in the paper's own block geometry ("block size for sparse attention 64 x 128":
 * 64 query rows x 128 keys per mask block; R26).  The kernel keeps its 128 x 64 tiles:
 *
 * chorus_mask_to_index_64x128
 *   bitmask   device, uint32 [L][H][ceil(N/64)][words], words = ceil(ceil(N/128) / 32); bit kb of a
 *             row = key block kb (keys 128 kb .. 128 kb + 127); pad bits are ignored.
 *   row_ptr   device, int32 [L*H*ceil(N/128) + 1]: row (l, h, qb) covers mask rows 2 qb ("upper":
 *             query rows 0-63 of the 128) and 2 qb + 1 ("lower", if it exists).
 *   col_idx   device, int32 [col_cap] or NULL (count only).  For every key block kept by EITHER mask
 *             row, ascending, and each of its two 64-key tiles t = 2 kb, 2 kb + 1 with 64 t < N, one
 *             entry  t | (upper does not keep kb) << 30 | (lower does not keep kb) << 31.
 *             An entry without flag bits is a plain chorus_mask_to_index entry.
 *   workspace as for chorus_mask_to_index (NULL = size query), 16-byte aligned.
 *   Unique result, compared bit-exactly with the oracle.  One launch: the decode kernel forms the tile
 *   mask of a row pair on the fly and never stores it.
 *
 * chorus_block_sparse_attn_fwd_64x128
 *   The attention call (arguments as chorus_block_sparse_attn_fwd_first_frame; n_first = 0 or beta = 1
 *   for no first-frame scaling) on such an index: query row i
 *   attends the keys of the key blocks its own 64-row mask row keeps, exactly; the tiles a 128-row
 *   block's other half alone keeps are computed and masked (up to 2x the tile work of the mask when
 *   the two halves share nothing, none when they agree).  Same accuracy bounds as the plain call.
 * Errors: as the plain calls.
 * ------------------------------------------------------------------------------------------- */
chorus_status chorus_mask_to_index_64x128(const uint32_t* bitmask, int L, int H, int N,
                                          int32_t* row_ptr, int32_t* col_idx, int64_t col_cap,
                                          void* workspace, size_t* workspace_bytes, void* cuda_stream);
chorus_status chorus_block_sparse_attn_fwd_64x128(const void* Q, const void* K, const void* V,
                                                  const int32_t* row_ptr, const int32_t* col_idx,
                                                  float scale, chorus_dtype dtype, void* O,
                                                  const chorus_attn_shape* shape,
                                                  const chorus_fp8_scales* fp8, float* lse,
                                                  int n_first, float beta, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * 16-bit index entries (the decoded index is what the attention
 * kernel "loads and uses directly", and at 25 % density its entries are 5.24 of the 5.9 MB that the
 * decode of a 480p layer moves: 16-bit entries halve that, and the key-block indices of the
 * paper's shapes, 512 and 1182, fit).
 *
 * chorus_mask_to_index_u16, chorus_mask_to_index_64x128_u16: the two decodes above with
 *   col_idx   device, uint16 [col_cap] (2-byte aligned) or NULL (count only).  Plain geometry: the
 *             key-block index (nk_blk <= 65536).  64 x 128 geometry: t | (upper does not keep kb) << 14
 *             | (lower does not keep kb) << 15 (ceil(N/64) <= 16384).
 *   row_ptr, workspace, order of the entries: exactly as in the 32-bit calls; compared bit-exactly
 *   with the oracle's 16-bit forms.
 * chorus_block_sparse_attn_fwd_idx16: the attention call on such an index.  Arguments as
 *   chorus_block_sparse_attn_fwd_first_frame plus geometry_64x128 (non-zero: the entries carry the two
 *   per-half flags, as chorus_block_sparse_attn_fwd_64x128 takes them in 32 bits).  The result is
 *   bit-identical to the call on the 32-bit index of the same mask.
 * Errors: as the 32-bit calls, and UNSUPPORTED when an index does not fit (nk_blk > 65536, or more
 *         than 16384 tiles with the flags).
 * ------------------------------------------------------------------------------------------- */
chorus_status chorus_mask_to_index_u16(const uint32_t* bitmask, int L, int H, int nq_blk, int nk_blk,
                                       int32_t* row_ptr, uint16_t* col_idx, int64_t col_cap,
                                       void* workspace, size_t* workspace_bytes, void* cuda_stream);
chorus_status chorus_mask_to_index_64x128_u16(const uint32_t* bitmask, int L, int H, int N,
                                              int32_t* row_ptr, uint16_t* col_idx, int64_t col_cap,
                                              void* workspace, size_t* workspace_bytes, void* cuda_stream);
chorus_status chorus_block_sparse_attn_fwd_idx16(const void* Q, const void* K, const void* V,
                                                 const int32_t* row_ptr, const uint16_t* col_idx,
                                                 float scale, chorus_dtype dtype, void* O,
                                                 const chorus_attn_shape* shape,
                                                 const chorus_fp8_scales* fp8, float* lse,
                                                 int n_first, float beta, int geometry_64x128,
                                                 void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * FP8 quantisation pre-pass for dtype = CHORUS_FP8_E4M3 (PAPER.md:L97 says only "FP8
 * quantization"; granularity and formula are BASELINE.json configs[2] / DESIGN.md R10-R11):
 *     s  = max(amax, 1e-12) / 448      x8 = e4m3_rne_saturate(x / s)       (fp32 arithmetic)
 * with amax over one (b, h, 128-token block) for Q and K, and over all tokens of one
 * (b, h, channel) for V; only tokens < N count.
 * Q, K, V   device, bf16, [B][N][H][d] with the strides in `shape` (o_stride_* ignored).
 * q8,k8,v8  device, uint8 e4m3 codes, PACKED [B][N][H][d] (stride_n = H*d, stride_h = d).
 * q_scale, k_scale  device float [B][H][ceil(N/128)];  v_scale  device float [B][H][d].
 * Errors: INVALID_ARG, UNSUPPORTED (d != 128), CUDA.
 * ------------------------------------------------------------------------------------------- */
chorus_status chorus_quantize_fp8(const void* Q, const void* K, const void* V,
                                  const chorus_attn_shape* shape, void* q8, void* k8, void* v8,
                                  float* q_scale, float* k_scale, float* v_scale,
                                  void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Retrieval ("k-nearest-neighbor search under cosine similarity over the joint text
 * and image embeddings; if the similarity to the top neighbor exceeds a threshold tau, its cached
 * sparse masks are loaded"; tau = 0.4 at L149).  Embeddings are unit-norm, so cosine = dot.
 * bank      device, float [n][dim], row-major, 16-byte aligned, dim % 4 == 0.
 * query     device, float [dim].
 * best_idx  device int32: argmax_j <bank[j], query>, ties -> lowest j.
 * best_sim  device float: that dot product (fp32 accumulation).
 * hit       device int32: 1 if best_sim >= tau else 0 (0 => caller falls back, L87/L149).
 * workspace device scratch, same query protocol as chorus_mask_to_index.
 * Errors: INVALID_ARG, CAPACITY (workspace too small), CUDA.
 * ------------------------------------------------------------------------------------------- */
chorus_status chorus_retrieve_top1(const float* bank, int n, int dim, const float* query, float tau,
                                   int32_t* best_idx, float* best_sim, int32_t* hit,
                                   void* workspace, size_t* workspace_bytes, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Mask construction from a dense pass (the historical request's side of sparsity reuse,
 * "in the dense case we select a block-level mask from its attention map via top-p
 * with a top-k floor"; L93 (2) min_top_k; L73 coverage; defaults at L153: top_p 0.95 / 0.9,
 * min_top_k 0.1 / 0.0).  Three calls: block mass -> mask -> (optionally) coverage.
 *
 * chorus_block_mass: mass[b][h][qb][kb] = sum over queries i of query block qb and keys j of key
 *   block kb of softmax_j(scale * <Q[i], K[j]>), the softmax taken over ALL N keys (the true, dense
 *   attention).  Every valid query row contributes exactly 1.
 *   Q, K     device, bf16, [B][N][H][d] with the q_/k_ strides of `shape` (v_/o_ strides ignored);
 *            16-byte aligned, strides multiples of 8 elements, d = 128.
 *   lse      device, float [B][H][N] or NULL: the rows' log-sum-exp (natural log) of the SAME dense
 *            attention, as written by chorus_block_sparse_attn_fwd_lse with a full mask.  Given, the
 *            kernel makes one pass over the keys instead of two (half the MMAs and exponentials).
 *   mass     device, float [B][H][ceil(N/128)][ceil(N/64)], fully overwritten.
 *   Accuracy against the fp64 oracle: |err| <= 2e-3 * max(mass, 1e-3) + 1e-5 per block (bf16
 *   products, fp32 sums, ex2.approx); the result is deterministic (fixed summation order).
 *
 * chorus_mask_from_mass: one row of nk_blk masses at a time (R22): masses are taken in
 *   units of 2^-24 (q = floor(mass * 2^24)), ranked by q descending with ties by index ascending;
 *   the row keeps the shortest prefix whose q-sum reaches ceil(top_p * sum q) (double product) and
 *   never fewer than ceil(min_top_k * nk_blk) blocks (double product).  Integer decisions: the
 *   result is compared bit-exactly with the oracle on the same masses.
 *   mass     device, float [rows][nk_blk], finite and >= 0;  nk_blk <= 2048.
 *   bitmask  device, uint32 [rows][ceil(nk_blk/32)], fully overwritten, pad bits 0 (the layout
 *            chorus_mask_to_index reads).
 *   kept     device, int32 [rows] or NULL: number of blocks kept per row.
 *
 * chorus_mask_coverage: coverage[h] = sum of the masses of the kept blocks of head h / sum of all
 *   its masses (0 if a head has no mass); fp64 accumulation, fixed order.
 *   mass [heads][nq_blk][nk_blk] float, bitmask [heads][nq_blk][words], coverage float [heads].
 * Errors: INVALID_ARG (null, sizes <= 0, top_p / min_top_k outside [0, 1], misalignment),
 *         UNSUPPORTED (d != 128, nk_blk > 2048), CUDA.
 * ------------------------------------------------------------------------------------------- */
chorus_status chorus_block_mass(const void* Q, const void* K, float scale,
                                const chorus_attn_shape* shape, const float* lse, float* mass,
                                void* cuda_stream);
/* chorus_block_mass with its output in the paper's 64 x 128 geometry (R26):
 * mass is float [B][H][ceil(N/64)][ceil(N/128)], mass[b][h][qb][kb] = sum of the token-level
 * probabilities of query rows 64 qb .. 64 qb + 63 over keys 128 kb .. 128 kb + 127.  Everything else
 * as chorus_block_mass; chorus_mask_from_mass (rows = B*H*ceil(N/64), nk_blk = ceil(N/128)) then
 * gives the bitmask chorus_mask_to_index_64x128 reads. */
chorus_status chorus_block_mass_64x128(const void* Q, const void* K, float scale,
                                       const chorus_attn_shape* shape, const float* lse, float* mass,
                                       void* cuda_stream);
chorus_status chorus_mask_from_mass(const float* mass, int64_t rows, int nk_blk, double top_p,
                                    double min_top_k, uint32_t* bitmask, int32_t* kept,
                                    void* cuda_stream);
chorus_status chorus_mask_coverage(const float* mass, const uint32_t* bitmask, int heads, int nq_blk,
                                   int nk_blk, float* coverage, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Head-level scheduling for load balance (PAPER.md:L95 and appendix A): with a reused
 * mask the cost of every head is known before the attention runs, so heads are re-partitioned over
 * the ranks of a sequence-parallel (Ulysses) group before the all-to-all.
 *
 * chorus_head_costs: cost[h] = kept tiles of head h = row_ptr[(h+1)*nq_blk] - row_ptr[h*nq_blk].
 *   row_ptr  device, int32, this layer's H*nq_blk + 1 entries;  cost  device, int64 [H].
 * chorus_schedule_heads (HOST function, no device work): heads in order of decreasing cost (ties:
 *   lower head first) go to the rank with the lightest current load among the ranks that still have
 *   room (ties: lower rank); a rank takes at most cap = ceil(H / n_ranks) heads (R24).
 *   cost     host, int64 [H], >= 0.
 *   order    host, int32 [n_ranks * cap]: order[r*cap + i] = i-th head of rank r (ascending inside a
 *            rank), -1 in unused slots.  n_ranks == 1 gives 0, 1, ..., H-1 (a no-op, Table 4).
 *   load     host, int64 [n_ranks] or NULL: summed cost per rank.
 * Errors: INVALID_ARG (null, H/n_ranks/nq_blk <= 0, negative cost), CUDA (head_costs only).
 * ------------------------------------------------------------------------------------------- */
chorus_status chorus_head_costs(const int32_t* row_ptr, int H, int nq_blk, int64_t* cost,
                                void* cuda_stream);
chorus_status chorus_schedule_heads(const int64_t* cost, int H, int n_ranks, int32_t* order,
                                    int64_t* load);

/* ---------------------------------------------------------------------------------------------
 * The two local copies around the Ulysses all-to-all (appendix A: the heads
 * are "re-partitioned (reordered) across ranks before the all-to-all communication").  A rank of a
 * sequence-parallel group holds n_tokens tokens of all H heads; the exchange hands rank p the heads
 * order[p * slots .. (p + 1) * slots), slots = H / n_ranks, of every rank's tokens.
 *   chorus_gather_heads    packed[p][i][s][:] = X[i][order[p * slots + s]][:]      (before the exchange)
 *   chorus_scatter_heads   X[i][order[p * slots + s]][:] = packed[p][i][s][:]      (after it, for O)
 * X        device, [n_tokens][H][d] with element strides stride_n, stride_h (last dim contiguous).
 * packed   device, contiguous [n_ranks][n_tokens][slots][d]: chunk p is what goes to / came from rank p.
 * order    HOST, H head indices, a permutation of 0..H-1 (chorus_schedule_heads' `order` when
 *          H % n_ranks == 0); validated on the host.
 * elem_bytes 1, 2 or 4; d * elem_bytes and the strides in bytes must be multiples of 16; X and packed
 *          16-byte aligned.  The exchange itself is the caller's (NCCL all-to-all with equal splits;
 *          paper_2606_25040_b200/ulysses.py); with one rank both calls are a head permutation.
 * Bit-exact copies.  Errors: INVALID_ARG, UNSUPPORTED (H > 256), CUDA.
 * ------------------------------------------------------------------------------------------- */
chorus_status chorus_gather_heads(const void* X, int n_tokens, int H, int d, int elem_bytes, int64_t stride_n,
                                  int64_t stride_h, const int32_t* order, int n_ranks, void* packed,
                                  void* cuda_stream);
chorus_status chorus_scatter_heads(const void* packed, int n_tokens, int H, int d, int elem_bytes,
                                   int64_t stride_n, int64_t stride_h, const int32_t* order, int n_ranks,
                                   void* X, void* cuda_stream);

/* Thread-local description of the last error returned on this thread ("" if none). */
const char* chorus_last_error(void);

/* Library/ABI version and build info, static storage. */
const char* chorus_version(void);

/* Number of kernel launches enqueued by this library on the calling thread since the last
 * chorus_reset_launch_count() (bench.py reports it as gpu_launches). */
int64_t chorus_launch_count(void);
void chorus_reset_launch_count(void);

/* TMA tensor maps are cached per thread, keyed by (pointer, element size, shape, strides, box): a call with
 * tensors seen before encodes nothing.  Number of cuTensorMapEncodeTiled calls made on this thread so far. */
int64_t chorus_tensor_map_encodes(void);

#ifdef __cplusplus
}
#endif
#endif /* CHORUS_H_ */
