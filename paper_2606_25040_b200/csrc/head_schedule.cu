// head_schedule.cu — head-level scheduling for load balance (appendix A):
// "the sparsity mask is known ahead of the attention computation, so each head's cost can be
// estimated in advance ... a greedy algorithm that re-partitions (reorders) heads across ranks
// before the all-to-all communication", "assigning heads with lower sparsity (i.e., heavier
// workload) to the GPUs with the lightest current load".
//   chorus_head_costs      device: kept tiles per head from the CSR row_ptr (one thread per head)
//   chorus_schedule_heads  host:   the greedy assignment (H is 40: nothing to gain on the device)
#include <algorithm>
#include <numeric>
#include <vector>

#include "chorus_internal.h"

namespace chorus {
namespace {

__global__ void head_costs_kernel(const int32_t* __restrict__ row_ptr, int H, int nq,
                                  int64_t* __restrict__ cost) {
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h < H) cost[h] = static_cast<int64_t>(row_ptr[(h + 1) * nq]) - static_cast<int64_t>(row_ptr[h * nq]);
}

}  // namespace

cudaError_t launch_head_costs(const int32_t* row_ptr, int H, int nq, int64_t* cost, cudaStream_t stream) {
    head_costs_kernel<<<(H + 127) / 128, 128, 0, stream>>>(row_ptr, H, nq, cost);
    count_launch(1);
    return cudaGetLastError();
}

// Heads in order of decreasing cost (ties: lower head first) go to the rank with the lightest load
// among those that still have room (ties: lower rank); a rank takes at most ceil(H / n_ranks) heads,
// because the all-to-all that follows hands every rank the same number of head slots (R24).
// order[r * cap + i] = i-th head of rank r, ascending inside a rank, -1 in unused slots.
void schedule_heads_host(const int64_t* cost, int H, int n_ranks, int32_t* order, int64_t* load) {
    const int cap = (H + n_ranks - 1) / n_ranks;
    std::vector<int> idx(H);
    std::iota(idx.begin(), idx.end(), 0);
    std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) { return cost[a] > cost[b]; });
    std::vector<std::vector<int>> mine(n_ranks);
    std::vector<int64_t> ld(n_ranks, 0);
    for (int h : idx) {
        int best = -1;
        for (int r = 0; r < n_ranks; ++r)
            if (static_cast<int>(mine[r].size()) < cap && (best < 0 || ld[r] < ld[best])) best = r;
        mine[best].push_back(h);
        ld[best] += cost[h];
    }
    for (int r = 0; r < n_ranks; ++r) {
        std::sort(mine[r].begin(), mine[r].end());
        for (int i = 0; i < cap; ++i)
            order[r * cap + i] = i < static_cast<int>(mine[r].size()) ? mine[r][i] : -1;
        if (load) load[r] = ld[r];
    }
}

}  // namespace chorus
