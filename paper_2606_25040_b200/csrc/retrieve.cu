// retrieve.cu — chorus_retrieve_top1: cosine top-1 over unit-norm request embeddings with a
// threshold (tau = 0.4 at L149).  HBM-bound GEMV + argmax:
//   1. dot_rows:  one warp per bank row, float4 loads, query staged in shared memory;
//   2. argmax:    one block reduces (sim, idx) with ties -> lowest index and applies tau.
// Algorithmic traffic: 4*n*dim bytes read.
#include <algorithm>

#include "chorus_internal.h"

namespace chorus {
namespace {

constexpr int RT_THREADS = 256;
constexpr int RT_WARPS = RT_THREADS / 32;

__global__ void __launch_bounds__(RT_THREADS)
dot_rows_kernel(const float* __restrict__ bank, int n, int dim, const float* __restrict__ query,
                float* __restrict__ sims) {
    extern __shared__ float4 s_q[];
    const int dim4 = dim >> 2;
    const float4* q4 = reinterpret_cast<const float4*>(query);
    for (int i = threadIdx.x; i < dim4; i += RT_THREADS) s_q[i] = __ldg(q4 + i);
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int r = blockIdx.x * RT_WARPS + warp; r < n; r += gridDim.x * RT_WARPS) {
        const float4* row = reinterpret_cast<const float4*>(bank + static_cast<int64_t>(r) * dim);
        float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
#pragma unroll 4
        for (int i = lane; i < dim4; i += 32) {
            const float4 x = __ldg(row + i);
            const float4 y = s_q[i];
            a0 = fmaf(x.x, y.x, a0);
            a1 = fmaf(x.y, y.y, a1);
            a2 = fmaf(x.z, y.z, a2);
            a3 = fmaf(x.w, y.w, a3);
        }
        float a = (a0 + a1) + (a2 + a3);
        for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
        if (lane == 0) sims[r] = a;
    }
}

__device__ __forceinline__ void better(float& s, int& i, float s2, int i2) {
    if (s2 > s || (s2 == s && i2 < i)) { s = s2; i = i2; }
}

__global__ void __launch_bounds__(1024)
argmax_kernel(const float* __restrict__ sims, int n, float tau, int32_t* __restrict__ best_idx,
              float* __restrict__ best_sim, int32_t* __restrict__ hit) {
    __shared__ float ws[32];
    __shared__ int wi[32];
    float s = -INFINITY;
    int idx = 0x7fffffff;
    for (int i = threadIdx.x; i < n; i += 1024) better(s, idx, sims[i], i);
    for (int o = 16; o > 0; o >>= 1) {
        const float s2 = __shfl_xor_sync(0xffffffffu, s, o);
        const int i2 = __shfl_xor_sync(0xffffffffu, idx, o);
        better(s, idx, s2, i2);
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { ws[warp] = s; wi[warp] = idx; }
    __syncthreads();
    if (warp == 0) {
        s = ws[lane];
        idx = wi[lane];
        for (int o = 16; o > 0; o >>= 1) {
            const float s2 = __shfl_xor_sync(0xffffffffu, s, o);
            const int i2 = __shfl_xor_sync(0xffffffffu, idx, o);
            better(s, idx, s2, i2);
        }
        if (lane == 0) {
            *best_idx = idx;
            *best_sim = s;
            *hit = (s >= tau) ? 1 : 0;
        }
    }
}

}  // namespace

size_t retrieve_workspace_bytes(int n) { return static_cast<size_t>(n) * sizeof(float); }

cudaError_t launch_retrieve_top1(const float* bank, int n, int dim, const float* query, float tau,
                                 int32_t* best_idx, float* best_sim, int32_t* hit, void* workspace,
                                 cudaStream_t stream) {
    float* sims = static_cast<float*>(workspace);
    const int blocks = std::min((n + RT_WARPS - 1) / RT_WARPS, 148 * 8);
    const size_t smem = static_cast<size_t>(dim) * sizeof(float);
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(dot_rows_kernel,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             static_cast<int>(smem));
        if (e != cudaSuccess) return e;
    }
    dot_rows_kernel<<<blocks, RT_THREADS, smem, stream>>>(bank, n, dim, query, sims);
    argmax_kernel<<<1, 1024, 0, stream>>>(sims, n, tau, best_idx, best_sim, hit);
    count_launch(2);
    return cudaGetLastError();
}

}  // namespace chorus
