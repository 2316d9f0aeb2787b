// mask_decode.cu — chorus_mask_to_index and chorus_visit_refresh kernels (HBM-bound integer work).
//
// Decode (PAPER.md:L81/L87/L93; include/chorus.h): packed block bitmask [rows][words] ->
// CSR (row_ptr, col_idx), ascending inside each row.  Three launches:
//   1. count_rows:   one warp per row: popcount of the valid bits -> row_ptr[r+1] holds the row's
//                    count; each block also writes the sum of its ROWS_PER_BLOCK rows.
//   2. scan_blocks:  one block turns the per-block sums into exclusive offsets.
//   3. scatter_rows: each block scans its rows' counts (block offset + local exclusive scan),
//                    writes the final row_ptr, and each warp expands its rows' set bits through a
//                    shared-memory staging buffer so that col_idx is written in contiguous,
//                    coalesced runs.
// Algorithmic traffic: 4*(rows*words) read + 4*(rows+1) + 4*nnz written (the bitmask is read a
// second time by launch 3; for every workload here it is still L2-resident).
#include <algorithm>

#include "chorus_internal.h"

namespace chorus {
namespace {

constexpr int DEC_THREADS = 256;
constexpr int DEC_WARPS = DEC_THREADS / 32;
constexpr int ROWS_PER_WARP = 16;
constexpr int ROWS_PER_BLOCK = DEC_WARPS * ROWS_PER_WARP;  // 128

__device__ __forceinline__ uint32_t valid_word(const uint32_t* __restrict__ row, int w, int nk) {
    // word w of a row with the pad bits (>= nk) cleared; 0 beyond the row
    const int lo = w * 32;
    if (lo >= nk) return 0u;
    uint32_t v = __ldg(row + w);
    const int rem = nk - lo;
    if (rem < 32) v &= (1u << rem) - 1u;
    return v;
}

__global__ void __launch_bounds__(DEC_THREADS)
count_rows_kernel(const uint32_t* __restrict__ bitmask, int64_t rows, int nk, int words,
                  int32_t* __restrict__ row_ptr, int32_t* __restrict__ block_sums) {
    __shared__ int warp_sums[DEC_WARPS];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t row0 = static_cast<int64_t>(blockIdx.x) * ROWS_PER_BLOCK + warp * ROWS_PER_WARP;
    int wsum = 0;
    for (int i = 0; i < ROWS_PER_WARP; ++i) {
        const int64_t r = row0 + i;
        if (r >= rows) break;
        const uint32_t* row = bitmask + r * words;
        int c = 0;
        for (int w = lane; w < words; w += 32) c += __popc(valid_word(row, w, nk));
        c = __reduce_add_sync(0xffffffffu, c);
        if (lane == 0) row_ptr[r + 1] = c;
        wsum += c;
    }
    if (lane == 0) warp_sums[warp] = wsum;
    __syncthreads();
    if (threadIdx.x == 0) {
        int s = 0;
        for (int w = 0; w < DEC_WARPS; ++w) s += warp_sums[w];
        block_sums[blockIdx.x] = s;
    }
}

// exclusive scan of block_sums (n entries) in place; one block of 1024 threads
__global__ void __launch_bounds__(1024)
scan_blocks_kernel(int32_t* __restrict__ block_sums, int n) {
    __shared__ int warp_tot[32];
    __shared__ int carry_s;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < n; base += 1024) {
        const int i = base + threadIdx.x;
        const int v = (i < n) ? block_sums[i] : 0;
        int inc = v;
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) warp_tot[warp] = inc;
        __syncthreads();
        if (warp == 0) {
            int t = warp_tot[lane];
            int ti = t;
            for (int o = 1; o < 32; o <<= 1) {
                const int u = __shfl_up_sync(0xffffffffu, ti, o);
                if (lane >= o) ti += u;
            }
            warp_tot[lane] = ti - t;  // exclusive prefix of the warp totals
        }
        __syncthreads();
        const int carry = carry_s;
        if (i < n) block_sums[i] = carry + warp_tot[warp] + inc - v;
        __syncthreads();
        if (threadIdx.x == 1023) carry_s = carry + warp_tot[warp] + inc;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(DEC_THREADS)
scatter_rows_kernel(const uint32_t* __restrict__ bitmask, int64_t rows, int nk, int words,
                    int32_t* __restrict__ row_ptr, const int32_t* __restrict__ block_offsets,
                    int32_t* __restrict__ col_idx, int64_t col_cap) {
    __shared__ int s_cnt[ROWS_PER_BLOCK];
    __shared__ int s_off[ROWS_PER_BLOCK + 1];
    __shared__ int32_t s_stage[DEC_WARPS][1024];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t blk_row0 = static_cast<int64_t>(blockIdx.x) * ROWS_PER_BLOCK;

    // counts of this block's rows (written by launch 1 into row_ptr[r+1])
    if (threadIdx.x < ROWS_PER_BLOCK) {
        const int64_t r = blk_row0 + threadIdx.x;
        s_cnt[threadIdx.x] = (r < rows) ? row_ptr[r + 1] : 0;
    }
    __syncthreads();
    // exclusive scan of 128 counts by warp 0 (4 per lane)
    if (warp == 0) {
        int v[4], tot = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) { v[k] = s_cnt[lane * 4 + k]; tot += v[k]; }
        int inc = tot;
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        int run = block_offsets[blockIdx.x] + inc - tot;
#pragma unroll
        for (int k = 0; k < 4; ++k) { s_off[lane * 4 + k] = run; run += v[k]; }
        if (lane == 31) s_off[ROWS_PER_BLOCK] = run;
    }
    __syncthreads();
    // final row_ptr: row_ptr[r+1] = offset of row r+1 = off[r] + cnt[r]
    if (threadIdx.x < ROWS_PER_BLOCK) {
        const int64_t r = blk_row0 + threadIdx.x;
        if (r < rows) row_ptr[r + 1] = s_off[threadIdx.x + 1];
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) row_ptr[0] = 0;
    if (col_idx == nullptr) return;

    int32_t* stage = s_stage[warp];
    for (int i = 0; i < ROWS_PER_WARP; ++i) {
        const int lr = warp * ROWS_PER_WARP + i;
        const int64_t r = blk_row0 + lr;
        if (r >= rows) break;
        const uint32_t* row = bitmask + r * words;
        int64_t out = s_off[lr];
        // 32 words (1024 key blocks) per pass
        for (int w0 = 0; w0 < words; w0 += 32) {
            uint32_t v = valid_word(row, w0 + lane, (w0 + lane < words) ? nk : 0);
            const int c = __popc(v);
            int inc = c;
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += t;
            }
            const int total = __shfl_sync(0xffffffffu, inc, 31);
            int e = inc - c;
            const int kb0 = (w0 + lane) * 32;
            while (v) {
                const int b = __ffs(v) - 1;
                stage[e++] = kb0 + b;
                v &= v - 1;
            }
            __syncwarp();
            for (int t = lane; t < total; t += 32)
                if (out + t < col_cap) col_idx[out + t] = stage[t];
            __syncwarp();
            out += total;
        }
    }
}

// Visit refresh (PAPER.md:L93 (1)): one thread per (group, word of a layer).
__global__ void __launch_bounds__(256)
visit_refresh_kernel(uint32_t* __restrict__ bitmask, int n_groups, int64_t words_per_layer,
                     int words, int nk, int group) {
    const int64_t total = static_cast<int64_t>(n_groups) * words_per_layer;
    for (int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x; i < total;
         i += static_cast<int64_t>(gridDim.x) * blockDim.x) {
        const int64_t g = i / words_per_layer, x = i - g * words_per_layer;
        uint32_t* base = bitmask + (g * group) * words_per_layer + x;
        uint32_t seen = 0u;
        for (int l = 0; l < group - 1; ++l) seen |= base[l * words_per_layer];
        const int w = static_cast<int>(x % words);
        const int rem = nk - w * 32;
        const uint32_t valid = rem >= 32 ? 0xffffffffu : (rem <= 0 ? 0u : ((1u << rem) - 1u));
        base[(group - 1) * words_per_layer] |= (~seen) & valid;
    }
}

inline int64_t n_blocks_for(int64_t rows) { return (rows + ROWS_PER_BLOCK - 1) / ROWS_PER_BLOCK; }

}  // namespace

size_t decode_workspace_bytes(int64_t rows) {
    return static_cast<size_t>(n_blocks_for(rows)) * sizeof(int32_t);
}

cudaError_t launch_mask_decode(const uint32_t* bitmask, int64_t rows, int nk, int words,
                               int32_t* row_ptr, int32_t* col_idx, int64_t col_cap, void* workspace,
                               cudaStream_t stream) {
    const int nb = static_cast<int>(n_blocks_for(rows));
    int32_t* block_sums = static_cast<int32_t*>(workspace);
    count_rows_kernel<<<nb, DEC_THREADS, 0, stream>>>(bitmask, rows, nk, words, row_ptr, block_sums);
    scan_blocks_kernel<<<1, 1024, 0, stream>>>(block_sums, nb);
    scatter_rows_kernel<<<nb, DEC_THREADS, 0, stream>>>(bitmask, rows, nk, words, row_ptr,
                                                        block_sums, col_idx, col_cap);
    count_launch(3);
    return cudaGetLastError();
}

cudaError_t launch_visit_refresh(uint32_t* bitmask, int L, int64_t words_per_layer, int words,
                                 int nk, int group, cudaStream_t stream) {
    const int n_groups = L / group;
    if (n_groups == 0) return cudaSuccess;
    const int64_t total = static_cast<int64_t>(n_groups) * words_per_layer;
    const int blocks = static_cast<int>(std::min<int64_t>((total + 255) / 256, 148 * 16));
    visit_refresh_kernel<<<blocks, 256, 0, stream>>>(bitmask, n_groups, words_per_layer, words, nk,
                                                     group);
    count_launch(1);
    return cudaGetLastError();
}

}  // namespace chorus
