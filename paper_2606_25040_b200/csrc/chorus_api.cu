// chorus_api.cu — the C ABI of libchorus.so (include/chorus.h): argument validation, TMA tensor-map
// construction and kernel launches.  No torch types, no allocation, no synchronisation.
#include <cstdarg>
#include <cstdio>
#include <cstring>

#include "chorus_internal.h"

namespace chorus {
namespace {

thread_local char g_err[512] = "";
thread_local int64_t g_launches = 0;

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (fn) return fn;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
        return nullptr;
    fn = reinterpret_cast<EncodeTiledFn>(p);
    return fn;
}

// Tensor map over a [B][N][H][d]-indexed tensor with element strides (d contiguous):
// dims (innermost first) = {d, N, H, B}; box = {box_cols, box_rows, 1, 1}; 128-byte swizzle.
// Encoded maps are kept in a small per-thread cache keyed by everything that goes into the encoding
// (SURVEY section 8(b)): a serving loop calls with the same few tensors over and over, and
// cuTensorMapEncodeTiled costs a few microseconds of host time per map.
struct TmapKey {
    const void* base;
    int elem_bytes, B, H, N, d, box_cols, box_rows;
    int64_t sb, sn, sh;
    bool operator==(const TmapKey& o) const {
        return base == o.base && elem_bytes == o.elem_bytes && B == o.B && H == o.H && N == o.N && d == o.d &&
               box_cols == o.box_cols && box_rows == o.box_rows && sb == o.sb && sn == o.sn && sh == o.sh;
    }
};
constexpr int TMAP_CACHE = 1024, TMAP_PROBES = 8;     // hashed, 8-way probing, the first probe is the victim
struct TmapCache {
    TmapKey key[TMAP_CACHE];
    CUtensorMap map[TMAP_CACHE];
    bool used[TMAP_CACHE];
};
thread_local TmapCache* g_tmaps = nullptr;
thread_local int64_t g_tmap_encodes = 0;

uint32_t tmap_hash(const TmapKey& k) {
    uint64_t h = reinterpret_cast<uintptr_t>(k.base) * 0x9E3779B97F4A7C15ull;
    h ^= (static_cast<uint64_t>(k.box_rows) << 40) ^ (static_cast<uint64_t>(k.elem_bytes) << 32) ^ static_cast<uint64_t>(k.sn) ^
         (static_cast<uint64_t>(k.N) << 13);
    h *= 0xC2B2AE3D27D4EB4Full;
    return static_cast<uint32_t>(h >> 40);
}

chorus_status make_tmap(CUtensorMap* tm, const void* base, int elem_bytes, int B, int H, int N,
                        int d, int64_t sb, int64_t sn, int64_t sh, int box_cols, int box_rows,
                        const char* name) {
    // a size-1 dimension never advances; give it a harmless, valid stride
    const int64_t row = static_cast<int64_t>(d);
    if (N == 1) sn = row;
    if (H == 1) sh = row;
    if (B == 1) sb = row;
    const TmapKey k{base, elem_bytes, B, H, N, d, box_cols, box_rows, sb, sn, sh};
    if (!g_tmaps) g_tmaps = new TmapCache();          // zero-initialised: nothing used
    const uint32_t h0 = tmap_hash(k);
    int slot = static_cast<int>(h0 % TMAP_CACHE);
    for (int i = 0; i < TMAP_PROBES; ++i) {
        const int s = static_cast<int>((h0 + i) % TMAP_CACHE);
        if (!g_tmaps->used[s]) { slot = s; break; }
        if (g_tmaps->key[s] == k) {
            *tm = g_tmaps->map[s];
            return CHORUS_OK;
        }
    }
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) return set_error(CHORUS_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
    const CUtensorMapDataType dt =
        elem_bytes == 2 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_UINT8;
    cuuint64_t dims[4] = {static_cast<cuuint64_t>(d), static_cast<cuuint64_t>(N),
                          static_cast<cuuint64_t>(H), static_cast<cuuint64_t>(B)};
    cuuint64_t strides[3] = {static_cast<cuuint64_t>(sn) * elem_bytes,
                             static_cast<cuuint64_t>(sh) * elem_bytes,
                             static_cast<cuuint64_t>(sb) * elem_bytes};
    cuuint32_t box[4] = {static_cast<cuuint32_t>(box_cols), static_cast<cuuint32_t>(box_rows), 1, 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUresult r = enc(tm, dt, 4, const_cast<void*>(base), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                           CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS)
        return set_error(CHORUS_ERR_CUDA, "cuTensorMapEncodeTiled(%s) failed with CUresult %d", name,
                         static_cast<int>(r));
    ++g_tmap_encodes;
    g_tmaps->key[slot] = k;
    g_tmaps->map[slot] = *tm;
    g_tmaps->used[slot] = true;
    return CHORUS_OK;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

}  // namespace

chorus_status set_error(chorus_status st, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return st;
}

chorus_status check_cuda(cudaError_t e, const char* what) {
    if (e == cudaSuccess) return CHORUS_OK;
    return set_error(CHORUS_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

void count_launch(int n) { g_launches += n; }

}  // namespace chorus

using namespace chorus;

extern "C" {

const char* chorus_last_error(void) { return g_err; }

const char* chorus_version(void) {
    return "libchorus 0.1 (sm_100a; blocks 128q x 64k, head_dim 128; built " __DATE__ ")";
}

int64_t chorus_launch_count(void) { return g_launches; }
int64_t chorus_tensor_map_encodes(void) { return g_tmap_encodes; }
void chorus_reset_launch_count(void) { g_launches = 0; }

static chorus_status mask_to_index_impl(const uint32_t* bitmask, int L, int H, int nq_blk, int nk_blk,
                                        int32_t* row_ptr, void* col_idx, bool idx16, int64_t col_cap,
                                        void* workspace, size_t* workspace_bytes, void* cuda_stream) {
    g_err[0] = 0;
    if (!workspace_bytes) return set_error(CHORUS_ERR_INVALID_ARG, "workspace_bytes is null");
    if (L <= 0 || H <= 0 || nq_blk <= 0 || nk_blk <= 0)
        return set_error(CHORUS_ERR_INVALID_ARG, "L, H, nq_blk, nk_blk must be positive (%d %d %d %d)",
                         L, H, nq_blk, nk_blk);
    if (idx16 && nk_blk > 65536)
        return set_error(CHORUS_ERR_UNSUPPORTED, "nk_blk = %d does not fit a 16-bit index", nk_blk);
    const int64_t rows = static_cast<int64_t>(L) * H * nq_blk;
    if (rows * nk_blk > INT32_MAX)
        return set_error(CHORUS_ERR_CAPACITY, "L*H*nq_blk*nk_blk = %lld exceeds INT32_MAX",
                         static_cast<long long>(rows * nk_blk));
    const size_t need = decode_workspace_bytes(rows, (nk_blk + 31) / 32);
    if (!workspace) {
        *workspace_bytes = need;
        return CHORUS_OK;
    }
    if (!bitmask || !row_ptr) return set_error(CHORUS_ERR_INVALID_ARG, "bitmask / row_ptr is null");
    if (col_cap < 0) return set_error(CHORUS_ERR_INVALID_ARG, "col_cap < 0");
    if ((reinterpret_cast<uintptr_t>(bitmask) | reinterpret_cast<uintptr_t>(row_ptr) |
         reinterpret_cast<uintptr_t>(workspace)) & 3u)
        return set_error(CHORUS_ERR_INVALID_ARG, "pointers must be 4-byte aligned");
    if (reinterpret_cast<uintptr_t>(col_idx) & (idx16 ? 1u : 3u))
        return set_error(CHORUS_ERR_INVALID_ARG, "col_idx must be aligned to its entry size");
    if (*workspace_bytes < need)
        return set_error(CHORUS_ERR_CAPACITY, "workspace too small: %zu < %zu", *workspace_bytes, need);
    const int words = (nk_blk + 31) / 32;
    return check_cuda(launch_mask_decode(bitmask, rows, nk_blk, words, row_ptr, col_idx, idx16, col_cap,
                                         workspace, static_cast<cudaStream_t>(cuda_stream)),
                      "mask decode launch");
}

chorus_status chorus_mask_to_index(const uint32_t* bitmask, int L, int H, int nq_blk, int nk_blk,
                                   int32_t* row_ptr, int32_t* col_idx, int64_t col_cap,
                                   void* workspace, size_t* workspace_bytes, void* cuda_stream) {
    return mask_to_index_impl(bitmask, L, H, nq_blk, nk_blk, row_ptr, col_idx, false, col_cap, workspace,
                              workspace_bytes, cuda_stream);
}

chorus_status chorus_mask_to_index_u16(const uint32_t* bitmask, int L, int H, int nq_blk, int nk_blk,
                                       int32_t* row_ptr, uint16_t* col_idx, int64_t col_cap,
                                       void* workspace, size_t* workspace_bytes, void* cuda_stream) {
    return mask_to_index_impl(bitmask, L, H, nq_blk, nk_blk, row_ptr, col_idx, true, col_cap, workspace,
                              workspace_bytes, cuda_stream);
}

chorus_status chorus_mask_to_index_static(const uint32_t* bitmask, int L, int H, int nq_blk, int nk_blk,
                                          int32_t* row_ptr, int32_t* col_idx, int64_t col_cap,
                                          void* cuda_stream) {
    static_assert(STATIC_DECODE_MAX_TILES == CHORUS_STATIC_DECODE_MAX_TILES, "header and kernel disagree");
    g_err[0] = 0;
    if (L <= 0 || H <= 0 || nq_blk <= 0 || nk_blk <= 0)
        return set_error(CHORUS_ERR_INVALID_ARG, "L, H, nq_blk, nk_blk must be positive (%d %d %d %d)",
                         L, H, nq_blk, nk_blk);
    const int64_t rows = static_cast<int64_t>(L) * H * nq_blk;
    if (rows * nk_blk > INT32_MAX)
        return set_error(CHORUS_ERR_CAPACITY, "L*H*nq_blk*nk_blk = %lld exceeds INT32_MAX",
                         static_cast<long long>(rows * nk_blk));
    const int words = (nk_blk + 31) / 32;
    if (rows * words > CHORUS_STATIC_DECODE_MAX_WORDS || decode_static_tiles(rows, words) > STATIC_DECODE_MAX_TILES)
        return set_error(CHORUS_ERR_CAPACITY,
                         "mask set of %lld words exceeds the %d words the static scratch of "
                         "chorus_mask_to_index_static covers (use chorus_mask_to_index with a workspace)",
                         static_cast<long long>(rows * words), CHORUS_STATIC_DECODE_MAX_WORDS);
    if (!bitmask || !row_ptr) return set_error(CHORUS_ERR_INVALID_ARG, "bitmask / row_ptr is null");
    if (col_cap < 0) return set_error(CHORUS_ERR_INVALID_ARG, "col_cap < 0");
    if ((reinterpret_cast<uintptr_t>(bitmask) | reinterpret_cast<uintptr_t>(row_ptr) |
         reinterpret_cast<uintptr_t>(col_idx)) & 3u)
        return set_error(CHORUS_ERR_INVALID_ARG, "pointers must be 4-byte aligned");
    return check_cuda(launch_mask_decode_static(bitmask, rows, nk_blk, words, row_ptr, col_idx, false, col_cap,
                                                static_cast<cudaStream_t>(cuda_stream)),
                      "mask decode (static scratch) launch");
}

static chorus_status mask_to_index_64x128_impl(const uint32_t* bitmask, int L, int H, int N,
                                               int32_t* row_ptr, void* col_idx, bool idx16, int64_t col_cap,
                                               void* workspace, size_t* workspace_bytes, void* cuda_stream) {
    g_err[0] = 0;
    if (!workspace_bytes) return set_error(CHORUS_ERR_INVALID_ARG, "workspace_bytes is null");
    if (L <= 0 || H <= 0 || N <= 0)
        return set_error(CHORUS_ERR_INVALID_ARG, "L, H, N must be positive (%d %d %d)", L, H, N);
    const int64_t heads = static_cast<int64_t>(L) * H;
    const int64_t nq128 = (static_cast<int64_t>(N) + 127) / 128, nk64 = (static_cast<int64_t>(N) + 63) / 64;
    if (idx16 && nk64 > 16384)
        return set_error(CHORUS_ERR_UNSUPPORTED, "%lld tiles do not fit a 14-bit index", static_cast<long long>(nk64));
    if (heads * nq128 * nk64 > INT32_MAX)
        return set_error(CHORUS_ERR_CAPACITY, "L*H*ceil(N/128)*ceil(N/64) = %lld exceeds INT32_MAX",
                         static_cast<long long>(heads * nq128 * nk64));
    const size_t need = decode_64x128_workspace_bytes(heads, N);
    if (!workspace) {
        *workspace_bytes = need;
        return CHORUS_OK;
    }
    if (!bitmask || !row_ptr) return set_error(CHORUS_ERR_INVALID_ARG, "bitmask / row_ptr is null");
    if (col_cap < 0) return set_error(CHORUS_ERR_INVALID_ARG, "col_cap < 0");
    if ((reinterpret_cast<uintptr_t>(bitmask) | reinterpret_cast<uintptr_t>(row_ptr)) & 3u)
        return set_error(CHORUS_ERR_INVALID_ARG, "pointers must be 4-byte aligned");
    if (reinterpret_cast<uintptr_t>(col_idx) & (idx16 ? 1u : 3u))
        return set_error(CHORUS_ERR_INVALID_ARG, "col_idx must be aligned to its entry size");
    if (reinterpret_cast<uintptr_t>(workspace) & 15u)
        return set_error(CHORUS_ERR_INVALID_ARG, "workspace must be 16-byte aligned");
    if (*workspace_bytes < need)
        return set_error(CHORUS_ERR_CAPACITY, "workspace too small: %zu < %zu", *workspace_bytes, need);
    return check_cuda(launch_mask_decode_64x128(bitmask, heads, N, row_ptr, col_idx, idx16, col_cap, workspace,
                                                static_cast<cudaStream_t>(cuda_stream)),
                      "64x128 mask decode launch");
}

chorus_status chorus_mask_to_index_64x128(const uint32_t* bitmask, int L, int H, int N,
                                          int32_t* row_ptr, int32_t* col_idx, int64_t col_cap,
                                          void* workspace, size_t* workspace_bytes, void* cuda_stream) {
    return mask_to_index_64x128_impl(bitmask, L, H, N, row_ptr, col_idx, false, col_cap, workspace, workspace_bytes,
                                     cuda_stream);
}

chorus_status chorus_mask_to_index_64x128_u16(const uint32_t* bitmask, int L, int H, int N,
                                              int32_t* row_ptr, uint16_t* col_idx, int64_t col_cap,
                                              void* workspace, size_t* workspace_bytes, void* cuda_stream) {
    return mask_to_index_64x128_impl(bitmask, L, H, N, row_ptr, col_idx, true, col_cap, workspace, workspace_bytes,
                                     cuda_stream);
}

chorus_status chorus_visit_refresh(uint32_t* bitmask, int L, int H, int nq_blk, int nk_blk,
                                   int group, void* cuda_stream) {
    g_err[0] = 0;
    if (!bitmask) return set_error(CHORUS_ERR_INVALID_ARG, "bitmask is null");
    if (L <= 0 || H <= 0 || nq_blk <= 0 || nk_blk <= 0 || group < 1)
        return set_error(CHORUS_ERR_INVALID_ARG, "L, H, nq_blk, nk_blk must be positive, group >= 1");
    const int words = (nk_blk + 31) / 32;
    return check_cuda(launch_visit_refresh(bitmask, L, static_cast<int64_t>(H) * nq_blk * words,
                                           words, nk_blk, group,
                                           static_cast<cudaStream_t>(cuda_stream)),
                      "visit refresh launch");
}

static chorus_status validate_shape(const chorus_attn_shape* s, int elem_mult, bool check_o) {
    if (!s) return set_error(CHORUS_ERR_INVALID_ARG, "shape is null");
    if (s->d != CHORUS_HEAD_DIM)
        return set_error(CHORUS_ERR_UNSUPPORTED, "head_dim %d is not supported (only 128)", s->d);
    if (s->B <= 0 || s->H <= 0 || s->N <= 0)
        return set_error(CHORUS_ERR_INVALID_ARG, "B, H, N must be positive (%d %d %d)", s->B, s->H, s->N);
    const int64_t st[9] = {s->q_stride_b, s->q_stride_n, s->q_stride_h, s->k_stride_b, s->k_stride_n,
                           s->k_stride_h, s->v_stride_b, s->v_stride_n, s->v_stride_h};
    const int dimsz[3] = {s->B, s->N, s->H};
    for (int i = 0; i < 9; ++i) {
        if (dimsz[i % 3] == 1) continue;
        if (st[i] <= 0 || st[i] % elem_mult)
            return set_error(CHORUS_ERR_INVALID_ARG,
                             "Q/K/V stride #%d = %lld must be a positive multiple of %d elements", i,
                             static_cast<long long>(st[i]), elem_mult);
    }
    if (check_o) {
        const int64_t so[3] = {s->o_stride_b, s->o_stride_n, s->o_stride_h};
        for (int i = 0; i < 3; ++i) {
            if (dimsz[i] == 1) continue;
            if (so[i] <= 0 || so[i] % 8)
                return set_error(CHORUS_ERR_INVALID_ARG,
                                 "O stride #%d = %lld must be a positive multiple of 8 elements", i,
                                 static_cast<long long>(so[i]));
        }
    }
    return CHORUS_OK;
}

chorus_status chorus_block_sparse_attn_fwd(const void* Q, const void* K, const void* V,
                                           const int32_t* row_ptr, const int32_t* col_idx,
                                           float scale, chorus_dtype dtype, void* O,
                                           const chorus_attn_shape* shape,
                                           const chorus_fp8_scales* fp8, void* cuda_stream) {
    return chorus_block_sparse_attn_fwd_lse(Q, K, V, row_ptr, col_idx, scale, dtype, O, shape, fp8,
                                            nullptr, cuda_stream);
}

chorus_status chorus_block_sparse_attn_fwd_lse(const void* Q, const void* K, const void* V,
                                               const int32_t* row_ptr, const int32_t* col_idx,
                                               float scale, chorus_dtype dtype, void* O,
                                               const chorus_attn_shape* shape,
                                               const chorus_fp8_scales* fp8, float* lse,
                                               void* cuda_stream) {
    return chorus_block_sparse_attn_fwd_first_frame(Q, K, V, row_ptr, col_idx, scale, dtype, O, shape, fp8,
                                                    lse, 0, 1.0f, cuda_stream);
}

static chorus_status attn_impl(const void* Q, const void* K, const void* V, const int32_t* row_ptr,
                               const void* col_idx, bool idx16, float scale, chorus_dtype dtype, void* O,
                               const chorus_attn_shape* shape, const chorus_fp8_scales* fp8, float* lse,
                               int n_first, float beta, bool half_flags, void* cuda_stream);

chorus_status chorus_block_sparse_attn_fwd_first_frame(const void* Q, const void* K, const void* V,
                                                       const int32_t* row_ptr, const int32_t* col_idx,
                                                       float scale, chorus_dtype dtype, void* O,
                                                       const chorus_attn_shape* shape,
                                                       const chorus_fp8_scales* fp8, float* lse,
                                                       int n_first, float beta, void* cuda_stream) {
    return attn_impl(Q, K, V, row_ptr, col_idx, false, scale, dtype, O, shape, fp8, lse, n_first, beta, false, cuda_stream);
}

chorus_status chorus_block_sparse_attn_fwd_64x128(const void* Q, const void* K, const void* V,
                                                  const int32_t* row_ptr, const int32_t* col_idx,
                                                  float scale, chorus_dtype dtype, void* O,
                                                  const chorus_attn_shape* shape,
                                                  const chorus_fp8_scales* fp8, float* lse,
                                                  int n_first, float beta, void* cuda_stream) {
    return attn_impl(Q, K, V, row_ptr, col_idx, false, scale, dtype, O, shape, fp8, lse, n_first, beta, true, cuda_stream);
}

chorus_status chorus_block_sparse_attn_fwd_idx16(const void* Q, const void* K, const void* V,
                                                 const int32_t* row_ptr, const uint16_t* col_idx,
                                                 float scale, chorus_dtype dtype, void* O,
                                                 const chorus_attn_shape* shape,
                                                 const chorus_fp8_scales* fp8, float* lse,
                                                 int n_first, float beta, int geometry_64x128,
                                                 void* cuda_stream) {
    return attn_impl(Q, K, V, row_ptr, col_idx, true, scale, dtype, O, shape, fp8, lse, n_first, beta,
                     geometry_64x128 != 0, cuda_stream);
}

static chorus_status attn_impl(const void* Q, const void* K, const void* V, const int32_t* row_ptr,
                               const void* col_idx, bool idx16, float scale, chorus_dtype dtype, void* O,
                               const chorus_attn_shape* shape, const chorus_fp8_scales* fp8, float* lse,
                               int n_first, float beta, bool half_flags, void* cuda_stream) {
    g_err[0] = 0;
    if (!(scale > 0.f) || !(scale <= 3.0e38f))
        return set_error(CHORUS_ERR_INVALID_ARG, "scale = %g must be positive and finite", static_cast<double>(scale));
    if (n_first < 0) return set_error(CHORUS_ERR_INVALID_ARG, "n_first = %d is negative", n_first);
    if (!(beta > 0.f) || !(beta <= 3.0e38f))
        return set_error(CHORUS_ERR_INVALID_ARG, "beta = %g must be positive and finite", static_cast<double>(beta));
    if (dtype != CHORUS_BF16 && dtype != CHORUS_FP8_E4M3 && dtype != CHORUS_FP16)
        return set_error(CHORUS_ERR_UNSUPPORTED, "unknown dtype %d", static_cast<int>(dtype));
    if (!Q || !K || !V || !O || !row_ptr || !col_idx)
        return set_error(CHORUS_ERR_INVALID_ARG, "Q, K, V, O, row_ptr, col_idx must be non-null");
    if (!aligned16(Q) || !aligned16(K) || !aligned16(V) || !aligned16(O))
        return set_error(CHORUS_ERR_INVALID_ARG, "Q, K, V, O must be 16-byte aligned");
    if ((dtype == CHORUS_FP8_E4M3) != (fp8 != nullptr))
        return set_error(CHORUS_ERR_INVALID_ARG, "fp8 scales must be given iff dtype is FP8_E4M3");
    if (fp8 && (!fp8->q_scale || !fp8->k_scale || !fp8->v_scale))
        return set_error(CHORUS_ERR_INVALID_ARG, "fp8 scale pointers must be non-null");
    const int eb = dtype == CHORUS_FP8_E4M3 ? 1 : 2;
    chorus_status st = validate_shape(shape, 16 / eb, true);
    if (st != CHORUS_OK) return st;
    const chorus_attn_shape& s = *shape;

    CUtensorMap tmQ, tmK, tmV, tmO;
    const int cols = 128 / eb;  // 128-byte inner box: 64 bf16 or 128 fp8 channels
    if ((st = make_tmap(&tmQ, Q, eb, s.B, s.H, s.N, s.d, s.q_stride_b, s.q_stride_n, s.q_stride_h,
                        cols, CHORUS_BLOCK_Q, "Q")) != CHORUS_OK) return st;
    if ((st = make_tmap(&tmK, K, eb, s.B, s.H, s.N, s.d, s.k_stride_b, s.k_stride_n, s.k_stride_h,
                        cols, CHORUS_BLOCK_K, "K")) != CHORUS_OK) return st;
    if ((st = make_tmap(&tmV, V, eb, s.B, s.H, s.N, s.d, s.v_stride_b, s.v_stride_n, s.v_stride_h,
                        cols, CHORUS_BLOCK_K, "V")) != CHORUS_OK) return st;
    if ((st = make_tmap(&tmO, O, 2, s.B, s.H, s.N, s.d, s.o_stride_b, s.o_stride_n, s.o_stride_h,
                        64, CHORUS_BLOCK_Q, "O")) != CHORUS_OK) return st;

    AttnParams p;
    p.row_ptr = row_ptr;
    p.col_idx = col_idx;
    p.idx16 = idx16;
    p.O = O;
    p.o_sb = s.o_stride_b; p.o_sn = s.o_stride_n; p.o_sh = s.o_stride_h;
    p.B = s.B; p.H = s.H; p.N = s.N;
    p.nq = (s.N + CHORUS_BLOCK_Q - 1) / CHORUS_BLOCK_Q;
    p.nk = (s.N + CHORUS_BLOCK_K - 1) / CHORUS_BLOCK_K;
    if (idx16 && p.nk > (half_flags ? 16384 : 65536))
        return set_error(CHORUS_ERR_UNSUPPORTED, "%d key blocks do not fit the 16-bit index", p.nk);
    p.scale_log2 = scale * 1.4426950408889634f;
    p.q_scale = fp8 ? fp8->q_scale : nullptr;
    p.k_scale = fp8 ? fp8->k_scale : nullptr;
    p.v_scale = fp8 ? fp8->v_scale : nullptr;
    p.lse = lse;
    p.n_first = n_first < s.N ? n_first : s.N;
    p.beta = beta;
    p.half_flags = half_flags;
    cudaError_t e = launch_attn_fwd(tmQ, tmK, tmV, tmO, p, dtype, static_cast<cudaStream_t>(cuda_stream));
    if (e == cudaErrorNotSupported)
        return set_error(CHORUS_ERR_UNSUPPORTED, "dtype %d not implemented by this build", (int)dtype);
    return check_cuda(e, "attention launch");
}

static chorus_status block_mass_impl(const void* Q, const void* K, float scale, const chorus_attn_shape* shape,
                                     const float* lse, float* mass, bool geo64, void* cuda_stream);

chorus_status chorus_block_mass(const void* Q, const void* K, float scale,
                                const chorus_attn_shape* shape, const float* lse, float* mass,
                                void* cuda_stream) {
    return block_mass_impl(Q, K, scale, shape, lse, mass, false, cuda_stream);
}

chorus_status chorus_block_mass_64x128(const void* Q, const void* K, float scale,
                                       const chorus_attn_shape* shape, const float* lse, float* mass,
                                       void* cuda_stream) {
    return block_mass_impl(Q, K, scale, shape, lse, mass, true, cuda_stream);
}

static chorus_status block_mass_impl(const void* Q, const void* K, float scale, const chorus_attn_shape* shape,
                                     const float* lse, float* mass, bool geo64, void* cuda_stream) {
    g_err[0] = 0;
    if (!(scale > 0.f) || !(scale <= 3.0e38f))
        return set_error(CHORUS_ERR_INVALID_ARG, "scale = %g must be positive and finite", static_cast<double>(scale));
    if (!Q || !K || !mass) return set_error(CHORUS_ERR_INVALID_ARG, "Q, K, mass must be non-null");
    if (!aligned16(Q) || !aligned16(K)) return set_error(CHORUS_ERR_INVALID_ARG, "Q, K must be 16-byte aligned");
    if (!shape) return set_error(CHORUS_ERR_INVALID_ARG, "shape is null");
    // only the q_ / k_ strides are used: validate a copy whose v_ strides repeat k_
    chorus_attn_shape s = *shape;
    s.v_stride_b = s.k_stride_b; s.v_stride_n = s.k_stride_n; s.v_stride_h = s.k_stride_h;
    chorus_status st = validate_shape(&s, 8, false);
    if (st != CHORUS_OK) return st;
    CUtensorMap tmQ, tmK;
    if ((st = make_tmap(&tmQ, Q, 2, s.B, s.H, s.N, s.d, s.q_stride_b, s.q_stride_n, s.q_stride_h,
                        64, 128, "Q")) != CHORUS_OK) return st;
    if ((st = make_tmap(&tmK, K, 2, s.B, s.H, s.N, s.d, s.k_stride_b, s.k_stride_n, s.k_stride_h,
                        64, 128, "K")) != CHORUS_OK) return st;
    return check_cuda(launch_block_mass(tmQ, tmK, lse, mass, s.B, s.H, s.N, scale * 1.4426950408889634f, geo64,
                                        static_cast<cudaStream_t>(cuda_stream)), "block mass launch");
}

chorus_status chorus_mask_from_mass(const float* mass, int64_t rows, int nk_blk, double top_p,
                                    double min_top_k, uint32_t* bitmask, int32_t* kept,
                                    void* cuda_stream) {
    g_err[0] = 0;
    if (!mass || !bitmask) return set_error(CHORUS_ERR_INVALID_ARG, "mass / bitmask is null");
    if (rows <= 0 || nk_blk <= 0) return set_error(CHORUS_ERR_INVALID_ARG, "rows, nk_blk must be positive");
    if (rows > INT32_MAX) return set_error(CHORUS_ERR_CAPACITY, "rows = %lld exceeds INT32_MAX", (long long)rows);
    if (nk_blk > 2048) return set_error(CHORUS_ERR_UNSUPPORTED, "nk_blk = %d > 2048", nk_blk);
    if (!(top_p >= 0.0 && top_p <= 1.0) || !(min_top_k >= 0.0 && min_top_k <= 1.0))
        return set_error(CHORUS_ERR_INVALID_ARG, "top_p and min_top_k must lie in [0, 1]");
    return check_cuda(launch_mask_from_mass(mass, rows, nk_blk, top_p, min_top_k, bitmask, kept,
                                            static_cast<cudaStream_t>(cuda_stream)), "mask_from_mass launch");
}

chorus_status chorus_mask_coverage(const float* mass, const uint32_t* bitmask, int heads, int nq_blk,
                                   int nk_blk, float* coverage, void* cuda_stream) {
    g_err[0] = 0;
    if (!mass || !bitmask || !coverage) return set_error(CHORUS_ERR_INVALID_ARG, "mass / bitmask / coverage is null");
    if (heads <= 0 || nq_blk <= 0 || nk_blk <= 0)
        return set_error(CHORUS_ERR_INVALID_ARG, "heads, nq_blk, nk_blk must be positive");
    return check_cuda(launch_mask_coverage(mass, bitmask, heads, nq_blk, nk_blk, coverage,
                                           static_cast<cudaStream_t>(cuda_stream)), "mask_coverage launch");
}

chorus_status chorus_head_costs(const int32_t* row_ptr, int H, int nq_blk, int64_t* cost,
                                void* cuda_stream) {
    g_err[0] = 0;
    if (!row_ptr || !cost) return set_error(CHORUS_ERR_INVALID_ARG, "row_ptr / cost is null");
    if (H <= 0 || nq_blk <= 0) return set_error(CHORUS_ERR_INVALID_ARG, "H, nq_blk must be positive");
    return check_cuda(launch_head_costs(row_ptr, H, nq_blk, cost, static_cast<cudaStream_t>(cuda_stream)),
                      "head_costs launch");
}

chorus_status chorus_schedule_heads(const int64_t* cost, int H, int n_ranks, int32_t* order,
                                    int64_t* load) {
    g_err[0] = 0;
    if (!cost || !order) return set_error(CHORUS_ERR_INVALID_ARG, "cost / order is null");
    if (H <= 0 || n_ranks <= 0) return set_error(CHORUS_ERR_INVALID_ARG, "H, n_ranks must be positive");
    for (int h = 0; h < H; ++h)
        if (cost[h] < 0) return set_error(CHORUS_ERR_INVALID_ARG, "cost[%d] is negative", h);
    schedule_heads_host(cost, H, n_ranks, order, load);
    return CHORUS_OK;
}

static chorus_status move_heads(bool scatter, const void* src, void* dst, const int32_t* order, int n_tokens,
                                int H, int n_ranks, int d, int elem_bytes, int64_t stride_n, int64_t stride_h,
                                void* cuda_stream) {
    g_err[0] = 0;
    if (!src || !dst || !order) return set_error(CHORUS_ERR_INVALID_ARG, "X, packed, order must be non-null");
    if (n_tokens < 0 || H <= 0 || n_ranks <= 0 || d <= 0)
        return set_error(CHORUS_ERR_INVALID_ARG, "n_tokens >= 0 and H, n_ranks, d > 0 required");
    if (H % n_ranks) return set_error(CHORUS_ERR_INVALID_ARG, "H = %d is not a multiple of n_ranks = %d", H, n_ranks);
    if (H > CHORUS_MAX_EXCHANGE_HEADS) return set_error(CHORUS_ERR_UNSUPPORTED, "H = %d > %d", H, CHORUS_MAX_EXCHANGE_HEADS);
    if (static_cast<int64_t>(n_tokens) * H > INT32_MAX)
        return set_error(CHORUS_ERR_CAPACITY, "n_tokens * H = %lld exceeds INT32_MAX", static_cast<long long>(n_tokens) * H);
    if (elem_bytes != 1 && elem_bytes != 2 && elem_bytes != 4)
        return set_error(CHORUS_ERR_INVALID_ARG, "elem_bytes must be 1, 2 or 4");
    const int64_t row_bytes = static_cast<int64_t>(d) * elem_bytes;
    if (row_bytes % 16 || (stride_n * elem_bytes) % 16 || (stride_h * elem_bytes) % 16)
        return set_error(CHORUS_ERR_INVALID_ARG, "rows and strides must be multiples of 16 bytes");
    if (stride_h < d || stride_n < d) return set_error(CHORUS_ERR_INVALID_ARG, "strides smaller than a row");
    if (!aligned16(src) || !aligned16(dst)) return set_error(CHORUS_ERR_INVALID_ARG, "X, packed must be 16-byte aligned");
    bool seen[CHORUS_MAX_EXCHANGE_HEADS] = {false};
    for (int k = 0; k < H; ++k) {
        if (order[k] < 0 || order[k] >= H || seen[order[k]])
            return set_error(CHORUS_ERR_INVALID_ARG, "order is not a permutation of 0..H-1 (entry %d = %d)", k, order[k]);
        seen[order[k]] = true;
    }
    return check_cuda(launch_move_heads(scatter, src, dst, order, n_tokens, H, n_ranks, static_cast<int>(row_bytes),
                                        stride_n * elem_bytes, stride_h * elem_bytes,
                                        static_cast<cudaStream_t>(cuda_stream)), "head exchange copy launch");
}

chorus_status chorus_gather_heads(const void* X, int n_tokens, int H, int d, int elem_bytes, int64_t stride_n,
                                  int64_t stride_h, const int32_t* order, int n_ranks, void* packed,
                                  void* cuda_stream) {
    return move_heads(false, X, packed, order, n_tokens, H, n_ranks, d, elem_bytes, stride_n, stride_h, cuda_stream);
}

chorus_status chorus_scatter_heads(const void* packed, int n_tokens, int H, int d, int elem_bytes,
                                   int64_t stride_n, int64_t stride_h, const int32_t* order, int n_ranks,
                                   void* X, void* cuda_stream) {
    return move_heads(true, packed, X, order, n_tokens, H, n_ranks, d, elem_bytes, stride_n, stride_h, cuda_stream);
}

chorus_status chorus_quantize_fp8(const void* Q, const void* K, const void* V,
                                  const chorus_attn_shape* shape, void* q8, void* k8, void* v8,
                                  float* q_scale, float* k_scale, float* v_scale,
                                  void* cuda_stream) {
    g_err[0] = 0;
    if (!Q || !K || !V || !q8 || !k8 || !v8 || !q_scale || !k_scale || !v_scale)
        return set_error(CHORUS_ERR_INVALID_ARG, "all pointers must be non-null");
    if (!aligned16(Q) || !aligned16(K) || !aligned16(V) || !aligned16(q8) || !aligned16(k8) ||
        !aligned16(v8))
        return set_error(CHORUS_ERR_INVALID_ARG, "tensors must be 16-byte aligned");
    chorus_status st = validate_shape(shape, 8, false);
    if (st != CHORUS_OK) return st;
    return check_cuda(launch_quantize_fp8(Q, K, V, *shape, q8, k8, v8, q_scale, k_scale, v_scale,
                                          static_cast<cudaStream_t>(cuda_stream)),
                      "fp8 quantise launch");
}

chorus_status chorus_retrieve_top1(const float* bank, int n, int dim, const float* query, float tau,
                                   int32_t* best_idx, float* best_sim, int32_t* hit,
                                   void* workspace, size_t* workspace_bytes, void* cuda_stream) {
    g_err[0] = 0;
    if (!workspace_bytes) return set_error(CHORUS_ERR_INVALID_ARG, "workspace_bytes is null");
    if (n <= 0 || dim <= 0 || (dim & 3))
        return set_error(CHORUS_ERR_INVALID_ARG, "n > 0, dim > 0 and dim %% 4 == 0 required (%d, %d)", n, dim);
    const size_t need = retrieve_workspace_bytes(n);
    if (!workspace) {
        *workspace_bytes = need;
        return CHORUS_OK;
    }
    if (!bank || !query || !best_idx || !best_sim || !hit)
        return set_error(CHORUS_ERR_INVALID_ARG, "bank, query, best_idx, best_sim, hit must be non-null");
    if (!aligned16(bank) || !aligned16(query))
        return set_error(CHORUS_ERR_INVALID_ARG, "bank and query must be 16-byte aligned");
    if (*workspace_bytes < need)
        return set_error(CHORUS_ERR_CAPACITY, "workspace too small: %zu < %zu", *workspace_bytes, need);
    if (static_cast<size_t>(dim) * sizeof(float) > 200 * 1024)
        return set_error(CHORUS_ERR_CAPACITY, "dim %d does not fit the shared-memory query buffer", dim);
    return check_cuda(launch_retrieve_top1(bank, n, dim, query, tau, best_idx, best_sim, hit,
                                           workspace, static_cast<cudaStream_t>(cuda_stream)),
                      "retrieve launch");
}

}  // extern "C"
