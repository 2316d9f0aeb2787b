// head_exchange.cu — the two local copies around the Ulysses all-to-all (appendix A
// L264-275: "re-partitions (reorders) heads across ranks before the all-to-all communication").
// A rank holds its n_tokens tokens of every head, [n_tokens][H][d].  Before the exchange the heads are
// gathered in schedule order into one contiguous chunk per destination rank:
//     out[p][i][s][:] = X[i][order[p * slots + s]][:]          p < n_ranks, s < slots = H / n_ranks
// (chorus_gather_heads); after the exchange of the attention output the inverse copy
//     X[i][order[p * slots + s]][:] = in[p][i][s][:]
// puts the heads back (chorus_scatter_heads).  Pure data movement, HBM-bound: 16 bytes per thread and
// step, a row of d elements (256 B in bf16) is read and written by consecutive threads.
#include "chorus_internal.h"

namespace chorus {
namespace {

struct HeadOrder {          // the schedule, passed by value (kernel parameter space)
    int32_t h[CHORUS_MAX_EXCHANGE_HEADS];
};

template <bool kScatter>
__global__ void __launch_bounds__(256)
move_heads_kernel(const uint4* __restrict__ src, uint4* __restrict__ dst, const HeadOrder order,
                  uint32_t n_tokens, uint32_t rows /* n_tokens * H */, uint32_t slots,
                  int vec_per_row /* d * elem_bytes / 16 */, int64_t stride_n,
                  int64_t stride_h /* of X, in 16-byte units */) {
    // threadIdx.x walks the 16-byte pieces of a row, threadIdx.y the rows of the packed side [p][i][s]
    for (uint32_t r = blockIdx.x * blockDim.y + threadIdx.y; r < rows; r += gridDim.x * blockDim.y) {
        const uint32_t t = r / slots, s = r - t * slots;
        const uint32_t p = t / n_tokens, i = t - p * n_tokens;
        const int h = order.h[p * slots + s];
        const uint4* a = src + (kScatter ? static_cast<int64_t>(r) * vec_per_row : i * stride_n + h * stride_h);
        uint4* b = dst + (kScatter ? i * stride_n + h * stride_h : static_cast<int64_t>(r) * vec_per_row);
        for (int v = threadIdx.x; v < vec_per_row; v += blockDim.x) b[v] = a[v];
    }
}

}  // namespace

cudaError_t launch_move_heads(bool scatter, const void* src, void* dst, const int32_t* order, int n_tokens,
                              int H, int n_ranks, int row_bytes, int64_t stride_n_bytes,
                              int64_t stride_h_bytes, cudaStream_t stream) {
    const int vec = row_bytes / 16, slots = H / n_ranks;
    const int64_t rows = static_cast<int64_t>(n_tokens) * H;
    if (rows == 0) return cudaSuccess;
    HeadOrder ho;
    for (int k = 0; k < H; ++k) ho.h[k] = order[k];
    int bx = 1;
    while (bx < vec && bx < 32) bx <<= 1;              // threads along a row
    const dim3 block(bx, 256 / bx);
    const int64_t want = (rows + block.y - 1) / block.y;
    const unsigned blocks = static_cast<unsigned>(want < 148 * 16 ? want : 148 * 16);
    if (scatter)
        move_heads_kernel<true><<<blocks, block, 0, stream>>>(static_cast<const uint4*>(src), static_cast<uint4*>(dst), ho,
                                                              n_tokens, static_cast<uint32_t>(rows), slots, vec,
                                                              stride_n_bytes / 16, stride_h_bytes / 16);
    else
        move_heads_kernel<false><<<blocks, block, 0, stream>>>(static_cast<const uint4*>(src), static_cast<uint4*>(dst), ho,
                                                               n_tokens, static_cast<uint32_t>(rows), slots, vec,
                                                               stride_n_bytes / 16, stride_h_bytes / 16);
    count_launch(1);
    return cudaGetLastError();
}

}  // namespace chorus
