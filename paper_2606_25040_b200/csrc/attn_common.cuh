// attn_common.cuh — small device helpers shared by the attention kernels (attn_fwd.cu: bf16 / fp16,
// attn_fwd_fp8.cu: e4m3): the work item of the persistent kernels and a few register-level utilities.
#pragma once
#include "chorus_internal.h"
#include "sm100_ptx.cuh"

namespace chorus {
namespace attn {

using namespace ptx;

constexpr int BQ = 128, BK = 64;
constexpr int NUM_THREADS = 384;
constexpr int PRODUCER_WARP = 8, MMA_WARP = 9;

__device__ __forceinline__ void setmaxnreg_inc_216() { asm volatile("setmaxnreg.inc.sync.aligned.u32 216;"); }
__device__ __forceinline__ void setmaxnreg_dec_56() { asm volatile("setmaxnreg.dec.sync.aligned.u32 56;"); }

template <bool V>
struct BoolTag {
    static constexpr bool value = V;
};

// entry i of the index in its 32-bit form, whichever width it is stored in: a 16-bit entry is zero-extended, and
// its two per-half flags (bits 14 / 15, 64 x 128 geometry) go to bits 30 / 31
__device__ __forceinline__ int ld_col(const AttnParams& p, int64_t i) {
    if (!p.idx16) return __ldg(static_cast<const int32_t*>(p.col_idx) + i);
    const uint32_t e = __ldg(static_cast<const uint16_t*>(p.col_idx) + i);
    return p.half_flags ? static_cast<int>((e & 0x3fffu) | ((e >> 14) << 30)) : static_cast<int>(e);
}

struct Item {
    int b, h, qb, r0, nt, np;
};
__device__ __forceinline__ Item get_item(const AttnParams& p, int idx) {
    Item it;
    it.qb = idx % p.nq;
    const int bh = idx / p.nq;
    it.h = bh % p.H;
    it.b = bh / p.H;
    const int row = it.h * p.nq + it.qb;
    it.r0 = __ldg(p.row_ptr + row);
    it.nt = __ldg(p.row_ptr + row + 1) - it.r0;
    it.np = (it.nt + 1) >> 1;
    return it;
}

// the same, with every field broadcast from lane 0: the compiler then knows the values are
// warp-uniform (needed by the converged producer / MMA warps)
__device__ __forceinline__ Item get_item_uniform(const AttnParams& p, int idx) {
    Item it = get_item(p, idx);
    it.r0 = __shfl_sync(0xffffffffu, it.r0, 0);
    it.nt = __shfl_sync(0xffffffffu, it.nt, 0);
    it.np = (it.nt + 1) >> 1;
    return it;
}

__device__ __forceinline__ float max3(float a, float b, float c) { return fmaxf(fmaxf(a, b), c); }

// max of 64 fp32 bit patterns
__device__ __forceinline__ float max64(const uint32_t* sv) {
    float a0 = -INFINITY, a1 = -INFINITY, a2 = -INFINITY, a3 = -INFINITY;
#pragma unroll
    for (int k = 0; k < 64; k += 8) {
        a0 = max3(a0, __uint_as_float(sv[k]), __uint_as_float(sv[k + 1]));
        a1 = max3(a1, __uint_as_float(sv[k + 2]), __uint_as_float(sv[k + 3]));
        a2 = max3(a2, __uint_as_float(sv[k + 4]), __uint_as_float(sv[k + 5]));
        a3 = max3(a3, __uint_as_float(sv[k + 6]), __uint_as_float(sv[k + 7]));
    }
    return fmaxf(fmaxf(a0, a1), fmaxf(a2, a3));
}

}  // namespace attn
}  // namespace chorus
