// chorus_internal.h — declarations shared by the translation units of libchorus.so (host side).
#pragma once
#include <cstdint>
#include <cuda.h>
#include <cuda_runtime.h>

#include "../../include/chorus.h"

namespace chorus {

// thread-local error string + launch counter (chorus_api.cu)
chorus_status set_error(chorus_status st, const char* fmt, ...);
chorus_status check_cuda(cudaError_t e, const char* what);
void count_launch(int n = 1);

// ---- mask_decode.cu ----------------------------------------------------------------------------
size_t decode_workspace_bytes(int64_t rows, int words);
// col_idx: int32 entries, or uint16 entries when idx16
cudaError_t launch_mask_decode(const uint32_t* bitmask, int64_t rows, int nk, int words,
                               int32_t* row_ptr, void* col_idx, bool idx16, int64_t col_cap, void* workspace,
                               cudaStream_t stream);
size_t decode_64x128_workspace_bytes(int64_t heads, int N);
// decode with the status words in a file-scope device array of mask_decode.cu (no allocation, no workspace)
constexpr int64_t STATIC_DECODE_MAX_TILES = 16384;
int64_t decode_static_tiles(int64_t rows, int words);
cudaError_t launch_mask_decode_static(const uint32_t* bitmask, int64_t rows, int nk, int words, int32_t* row_ptr,
                                      void* col_idx, bool idx16, int64_t col_cap, cudaStream_t stream);
cudaError_t launch_mask_decode_64x128(const uint32_t* bm64, int64_t heads, int N, int32_t* row_ptr,
                                      void* col_idx, bool idx16, int64_t col_cap, void* workspace, cudaStream_t stream);
cudaError_t launch_visit_refresh(uint32_t* bitmask, int L, int64_t words_per_layer, int words,
                                 int nk, int group, cudaStream_t stream);

// ---- retrieve.cu -------------------------------------------------------------------------------
size_t retrieve_workspace_bytes(int n);
cudaError_t launch_retrieve_top1(const float* bank, int n, int dim, const float* query, float tau,
                                 int32_t* best_idx, float* best_sim, int32_t* hit, void* workspace,
                                 cudaStream_t stream);

// ---- quantize_fp8.cu ---------------------------------------------------------------------------
cudaError_t launch_quantize_fp8(const void* Q, const void* K, const void* V,
                                const chorus_attn_shape& s, void* q8, void* k8, void* v8,
                                float* q_scale, float* k_scale, float* v_scale,
                                cudaStream_t stream);

// ---- attn_fwd.cu -------------------------------------------------------------------------------
struct AttnParams {
    const int32_t* row_ptr;
    const void* col_idx;   // int32 entries, or uint16 entries when idx16 (flags of the 64 x 128 form at bits 14 / 15)
    bool idx16;
    void* O;
    int64_t o_sb, o_sn, o_sh;
    int B, H, N, nq, nk;
    float scale_log2;  // scale * log2(e)
    const float* q_scale;
    const float* k_scale;
    const float* v_scale;
    float* lse;  // optional [B][H][N] row log-sum-exp (natural log), or null
    int n_first;  // first-frame key enhancement (eq. 1): scores of keys < n_first are multiplied by beta
    float beta;   // > 0; n_first = 0 or beta = 1 selects the plain kernel
    bool half_flags;  // col_idx entries carry bits 30 / 31 (chorus_mask_to_index_64x128)
    int ticket_slot;  // which self-resetting work counter this launch draws its items from (set by the launcher)
};
cudaError_t launch_attn_fwd(const CUtensorMap& tmQ, const CUtensorMap& tmK, const CUtensorMap& tmV,
                            const CUtensorMap& tmO, const AttnParams& p, chorus_dtype dtype,
                            cudaStream_t stream);

// attn_fwd_fp8.cu: the e4m3 kernel (launch_attn_fwd dispatches to it)
cudaError_t launch_attn_fwd_fp8(const CUtensorMap& tmQ, const CUtensorMap& tmK, const CUtensorMap& tmV,
                                const CUtensorMap& tmO, const AttnParams& p, cudaStream_t stream);

// ---- mask_build.cu -----------------------------------------------------------------------------
cudaError_t launch_block_mass(const CUtensorMap& tmQ, const CUtensorMap& tmK, const float* lse, float* mass,
                              int B, int H, int N, float scale_log2, bool geo64, cudaStream_t stream);
cudaError_t launch_mask_from_mass(const float* mass, int64_t rows, int nk, double top_p, double min_top_k,
                                  uint32_t* bitmask, int32_t* kept, cudaStream_t stream);
cudaError_t launch_mask_coverage(const float* mass, const uint32_t* bitmask, int heads, int nq, int nk,
                                 float* coverage, cudaStream_t stream);

// ---- head_schedule.cu --------------------------------------------------------------------------
cudaError_t launch_head_costs(const int32_t* row_ptr, int H, int nq, int64_t* cost, cudaStream_t stream);
constexpr int CHORUS_MAX_EXCHANGE_HEADS = 256;
// order: HOST array of H head indices (a permutation, validated by the caller)
cudaError_t launch_move_heads(bool scatter, const void* src, void* dst, const int32_t* order, int n_tokens,
                              int H, int n_ranks, int row_bytes, int64_t stride_n_bytes,
                              int64_t stride_h_bytes, cudaStream_t stream);
void schedule_heads_host(const int64_t* cost, int H, int n_ranks, int32_t* order, int64_t* load);

}  // namespace chorus
