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
                  int n_tokens, int H, int slots, int vec_per_row /* d * elem_bytes / 16 */,
                  int64_t stride_n, int64_t stride_h /* of X, in 16-byte units */) {
    const int64_t total = static_cast<int64_t>(n_tokens) * H * vec_per_row;
    for (int64_t idx = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x; idx < total;
         idx += static_cast<int64_t>(gridDim.x) * blockDim.x) {
        // idx walks the packed side [p][i][s][v]
        const int v = static_cast<int>(idx % vec_per_row);
        int64_t r = idx / vec_per_row;
        const int s = static_cast<int>(r % slots);
        r /= slots;
        const int i = static_cast<int>(r % n_tokens);
        const int p = static_cast<int>(r / n_tokens);
        const int h = order.h[p * slots + s];
        const int64_t x = i * stride_n + h * stride_h + v;
        if (kScatter) dst[x] = src[idx];
        else dst[idx] = src[x];
    }
}

}  // namespace

cudaError_t launch_move_heads(bool scatter, const void* src, void* dst, const int32_t* order, int n_tokens,
                              int H, int n_ranks, int row_bytes, int64_t stride_n_bytes,
                              int64_t stride_h_bytes, cudaStream_t stream) {
    const int vec = row_bytes / 16, slots = H / n_ranks;
    const int64_t total = static_cast<int64_t>(n_tokens) * H * vec;
    if (total == 0) return cudaSuccess;
    HeadOrder ho;
    for (int k = 0; k < H; ++k) ho.h[k] = order[k];
    const int64_t want = (total + 255) / 256;
    const int blocks = static_cast<int>(want < 148 * 32 ? want : 148 * 32);
    if (scatter)
        move_heads_kernel<true><<<blocks, 256, 0, stream>>>(static_cast<const uint4*>(src), static_cast<uint4*>(dst),
                                                            ho, n_tokens, H, slots, vec, stride_n_bytes / 16,
                                                            stride_h_bytes / 16);
    else
        move_heads_kernel<false><<<blocks, 256, 0, stream>>>(static_cast<const uint4*>(src), static_cast<uint4*>(dst),
                                                             ho, n_tokens, H, slots, vec, stride_n_bytes / 16,
                                                             stride_h_bytes / 16);
    count_launch(1);
    return cudaGetLastError();
}

}  // namespace chorus
