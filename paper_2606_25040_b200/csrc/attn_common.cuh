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

// ---- dynamic item order ------------------------------------------------------------------------------------------
// The CTAs of a launch draw their work items from one counter instead of taking every gridDim-th item: rows of
// reused masks differ in length ("assigns a different sparsity level to each attention head"), and
// with a fixed share per CTA the longest share sets the kernel time.  Items are still handed out in head-major
// order, so the CTAs in flight keep working on one or two heads and their K / V stay in L2.
// The counter is one of a few device words that reset themselves: the last CTA of a launch to finish zeroes its
// slot, so no memset precedes the kernel.  The producer warp draws an index and passes it to the other roles of the
// CTA through a small ring in shared memory.
constexpr int ITEM_RING = 4, TICKET_SLOTS = 64;
static __device__ unsigned int g_item_ticket[TICKET_SLOTS], g_item_done[TICKET_SLOTS];

struct ItemRing {
    uint32_t full, empty;      // shared-memory addresses of ITEM_RING mbarriers each
    volatile int* slots;       // ITEM_RING indices
};
// producer warp, converged: the k-th item of this CTA (-1: none left), announced to the consumers
__device__ __forceinline__ int item_draw(const ItemRing& r, uint32_t k, int n_items, int ticket_slot) {
    const uint32_t s = k % ITEM_RING;
    mbar_wait(r.empty + 8 * s, ((k / ITEM_RING) & 1) ^ 1);
    int idx = 0;
    if ((threadIdx.x & 31) == 0)
        idx = k == 0 ? static_cast<int>(blockIdx.x)
                     : static_cast<int>(gridDim.x + atomicAdd(&g_item_ticket[ticket_slot], 1u));
    idx = __shfl_sync(0xffffffffu, idx, 0);
    if (idx >= n_items) idx = -1;
    if ((threadIdx.x & 31) == 0) {
        r.slots[s] = idx;
        mbar_arrive(r.full + 8 * s);
    }
    return idx;
}
// any other warp (all lanes): the k-th item of this CTA as the producer announced it
__device__ __forceinline__ int item_take(const ItemRing& r, uint32_t k) {
    const uint32_t s = k % ITEM_RING;
    mbar_wait(r.full + 8 * s, (k / ITEM_RING) & 1);
    const int idx = r.slots[s];
    __syncwarp();
    if ((threadIdx.x & 31) == 0) mbar_arrive(r.empty + 8 * s);
    return idx;
}
// one thread per CTA, after everything else: the last CTA of the launch resets the slot
__device__ __forceinline__ void item_ticket_release(int ticket_slot) {
    if (atomicAdd(&g_item_done[ticket_slot], 1u) == gridDim.x - 1) {
        g_item_ticket[ticket_slot] = 0u;
        g_item_done[ticket_slot] = 0u;
        __threadfence();
    }
}
inline int next_ticket_slot() {
    static unsigned int n = 0;      // launches are enqueued by one thread at a time per process in practice; a
    return static_cast<int>(n++ % TICKET_SLOTS);   // collision needs 64 launches of one kernel in flight at once
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
