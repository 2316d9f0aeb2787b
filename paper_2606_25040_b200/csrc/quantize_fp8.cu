// quantize_fp8.cu — chorus_quantize_fp8: bf16 Q/K/V -> e4m3 codes + fp32 scales for the FP8
// attention path (format per BASELINE.json configs[2], R10/R11):
//     s = max(amax, 1e-12) / 448 ;  x8 = e4m3_rne_saturate(x / s)          (fp32, IEEE division)
// Q, K: one scale per (b, h, 128-token block); V: one scale per (b, h, channel) over all tokens.
// HBM-bound.  Launches: memset(v_scale) -> v_amax (atomicMax on float bits) -> qk_quantize
// (one CTA per (b, h, block): amax in registers, then cast) -> v_quantize (reads v amax, casts)
// -> v_finalize (amax -> scale in place).
#include <cuda_bf16.h>
#include <cuda_fp8.h>

#include "chorus_internal.h"

namespace chorus {
namespace {

constexpr int QT = 256;  // threads per CTA; one CTA handles 128 tokens x 128 channels

__device__ __forceinline__ float bf16_bits_to_float(uint32_t b16) {
    return __uint_as_float(b16 << 16);
}
__device__ __forceinline__ uint32_t cvt4_e4m3(float a, float b, float c, float d) {
    const uint32_t lo = __nv_cvt_float2_to_fp8x2(make_float2(a, b), __NV_SATFINITE, __NV_E4M3);
    const uint32_t hi = __nv_cvt_float2_to_fp8x2(make_float2(c, d), __NV_SATFINITE, __NV_E4M3);
    return lo | (hi << 16);
}
__device__ __forceinline__ float scale_from_amax(float amax) {
    return __fdiv_rn(fmaxf(amax, 1e-12f), 448.0f);
}
// RN(x / s) for many x and one s: r = RN(1 / s) is computed once; per element a product and two
// FMA corrections (the second is exact-rounding by Markstein's theorem once the first has brought
// the quotient within an ulp).  |x / s| <= 448 and s >= 2.2e-15, so nothing over- or underflows on
// the way (quotients below 2^-10 round to the code 0 whatever their last bit is).  The generic
// __fdiv_rn costs about three times as many instructions, which made the cast compute-bound.
struct Divisor {
    float s, r;
};
__device__ __forceinline__ Divisor make_divisor(float s) { return Divisor{s, __frcp_rn(s)}; }
__device__ __forceinline__ float div_rn(float x, const Divisor& d) {
    float q = x * d.r;
    q = __fmaf_rn(__fmaf_rn(-d.s, q, x), d.r, q);
    q = __fmaf_rn(__fmaf_rn(-d.s, q, x), d.r, q);
    return q;
}

// thread layout inside a CTA: 16 threads per token row (16 B = 8 channels each), 16 rows per pass
struct Tile {
    uint4 v[8];  // 8 passes x 8 bf16
};

__device__ __forceinline__ float amax8(const uint4& u) {
    const uint32_t w[4] = {u.x, u.y, u.z, u.w};
    float m = 0.f;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        m = fmaxf(m, fabsf(bf16_bits_to_float(w[i] & 0xffffu)));
        m = fmaxf(m, fabsf(bf16_bits_to_float(w[i] >> 16)));
    }
    return m;
}

__device__ __forceinline__ uint2 quant8(const uint4& u, const Divisor& s) {
    const uint32_t w[4] = {u.x, u.y, u.z, u.w};
    float f[8];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        f[2 * i] = div_rn(bf16_bits_to_float(w[i] & 0xffffu), s);
        f[2 * i + 1] = div_rn(bf16_bits_to_float(w[i] >> 16), s);
    }
    return make_uint2(cvt4_e4m3(f[0], f[1], f[2], f[3]), cvt4_e4m3(f[4], f[5], f[6], f[7]));
}

// grid: (H, nsb, 2*B), heads fastest so that the CTAs in flight together cover whole 128-token
// slabs of the [N][H][d] tensor (contiguous DRAM pages); blockIdx.z = 2*b + which (0: Q, 1: K).
// The tile is read twice (amax, then cast; the second read comes from L1/L2) instead of being held
// in registers: 32 registers per thread, eight CTAs per SM instead of four.
__global__ void __launch_bounds__(QT, 8)
qk_quantize_kernel(const uint16_t* __restrict__ Q, const uint16_t* __restrict__ K,
                   chorus_attn_shape s, uint8_t* __restrict__ q8, uint8_t* __restrict__ k8,
                   float* __restrict__ q_scale, float* __restrict__ k_scale, int nsb) {
    __shared__ float s_red[QT / 32];
    __shared__ float s_scale;
    const int blk = blockIdx.y, h = blockIdx.x, b = blockIdx.z >> 1, which = blockIdx.z & 1;
    const uint16_t* X = which ? K : Q;
    const int64_t sb = which ? s.k_stride_b : s.q_stride_b;
    const int64_t sn = which ? s.k_stride_n : s.q_stride_n;
    const int64_t sh = which ? s.k_stride_h : s.q_stride_h;
    uint8_t* X8 = which ? k8 : q8;
    float* S = which ? k_scale : q_scale;

    const int sub = threadIdx.x & 15, rowp = threadIdx.x >> 4;
    const uint4* src = reinterpret_cast<const uint4*>(X + b * sb + (static_cast<int64_t>(blk) * 128 + rowp) * sn + h * sh) + sub;
    const int64_t step = 16 * sn / 8;                 // 16 token rows further, in uint4 units
    const int rows_left = s.N - blk * 128 - rowp;     // this thread's rows: rowp, rowp + 16, ... while < rows_left
    float m = 0.f;
#pragma unroll
    for (int p = 0; p < 8; ++p)
        if (p * 16 < rows_left) m = fmaxf(m, amax8(__ldg(src + p * step)));
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        float a = 0.f;
        for (int w = 0; w < QT / 32; ++w) a = fmaxf(a, s_red[w]);
        const float sc = scale_from_amax(a);
        s_scale = sc;
        S[(static_cast<int64_t>(b) * s.H + h) * nsb + blk] = sc;
    }
    __syncthreads();
    const Divisor sc = make_divisor(s_scale);
    uint2* dst = reinterpret_cast<uint2*>(X8 + ((static_cast<int64_t>(b) * s.N + blk * 128 + rowp) * s.H + h) * 128) + sub;
    const int64_t dstep = 16 * static_cast<int64_t>(s.H) * 128 / 8;
#pragma unroll
    for (int p = 0; p < 8; ++p)
        if (p * 16 < rows_left) dst[p * dstep] = quant8(__ldg(src + p * step), sc);
}

// V column amax: grid (H, chunks, B); each CTA covers V_ROWS tokens; atomicMax on float bits
constexpr int V_ROWS = 512;
__global__ void __launch_bounds__(QT)
v_amax_kernel(const uint16_t* __restrict__ V, chorus_attn_shape s, float* __restrict__ v_amax) {
    __shared__ float s_m[16][128];
    const int h = blockIdx.x, b = blockIdx.z;
    const int sub = threadIdx.x & 15, rowp = threadIdx.x >> 4;
    float m[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    const int n0 = blockIdx.y * V_ROWS;
    for (int n = n0 + rowp; n < n0 + V_ROWS && n < s.N; n += 16) {
        const uint4 u = __ldg(reinterpret_cast<const uint4*>(V + b * s.v_stride_b + n * s.v_stride_n +
                                                             h * s.v_stride_h) + sub);
        const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            m[2 * i] = fmaxf(m[2 * i], fabsf(bf16_bits_to_float(w[i] & 0xffffu)));
            m[2 * i + 1] = fmaxf(m[2 * i + 1], fabsf(bf16_bits_to_float(w[i] >> 16)));
        }
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) s_m[rowp][sub * 8 + i] = m[i];
    __syncthreads();
    if (threadIdx.x < 128) {
        float a = 0.f;
#pragma unroll
        for (int r = 0; r < 16; ++r) a = fmaxf(a, s_m[r][threadIdx.x]);
        // non-negative floats order like their bit patterns
        atomicMax(reinterpret_cast<int*>(v_amax + (static_cast<int64_t>(b) * s.H + h) * 128 +
                                         threadIdx.x),
                  __float_as_int(a));
    }
}

__global__ void __launch_bounds__(QT)
v_quantize_kernel(const uint16_t* __restrict__ V, chorus_attn_shape s,
                  const float* __restrict__ v_amax, uint8_t* __restrict__ v8) {
    const int h = blockIdx.x, b = blockIdx.z;
    const int sub = threadIdx.x & 15, rowp = threadIdx.x >> 4;
    Divisor sc[8];
#pragma unroll
    for (int i = 0; i < 8; ++i)
        sc[i] = make_divisor(scale_from_amax(v_amax[(static_cast<int64_t>(b) * s.H + h) * 128 + sub * 8 + i]));
    const int n0 = blockIdx.y * V_ROWS;
    for (int n = n0 + rowp; n < n0 + V_ROWS && n < s.N; n += 16) {
        const uint4 u = __ldg(reinterpret_cast<const uint4*>(V + b * s.v_stride_b + n * s.v_stride_n +
                                                             h * s.v_stride_h) + sub);
        const uint32_t w[4] = {u.x, u.y, u.z, u.w};
        float f[8];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            f[2 * i] = div_rn(bf16_bits_to_float(w[i] & 0xffffu), sc[2 * i]);
            f[2 * i + 1] = div_rn(bf16_bits_to_float(w[i] >> 16), sc[2 * i + 1]);
        }
        uint8_t* dst = v8 + ((static_cast<int64_t>(b) * s.N + n) * s.H + h) * 128;
        reinterpret_cast<uint2*>(dst)[sub] =
            make_uint2(cvt4_e4m3(f[0], f[1], f[2], f[3]), cvt4_e4m3(f[4], f[5], f[6], f[7]));
    }
}

__global__ void v_finalize_kernel(float* __restrict__ v_scale, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) v_scale[i] = scale_from_amax(v_scale[i]);
}

}  // namespace

cudaError_t launch_quantize_fp8(const void* Q, const void* K, const void* V,
                                const chorus_attn_shape& s, void* q8, void* k8, void* v8,
                                float* q_scale, float* k_scale, float* v_scale,
                                cudaStream_t stream) {
    const int nsb = (s.N + 127) / 128;
    const int nv = s.B * s.H * 128;
    cudaError_t e = cudaMemsetAsync(v_scale, 0, sizeof(float) * nv, stream);
    if (e != cudaSuccess) return e;
    const dim3 gv(s.H, (s.N + V_ROWS - 1) / V_ROWS, s.B);
    v_amax_kernel<<<gv, QT, 0, stream>>>(static_cast<const uint16_t*>(V), s, v_scale);
    qk_quantize_kernel<<<dim3(s.H, nsb, 2 * s.B), QT, 0, stream>>>(
        static_cast<const uint16_t*>(Q), static_cast<const uint16_t*>(K), s,
        static_cast<uint8_t*>(q8), static_cast<uint8_t*>(k8), q_scale, k_scale, nsb);
    v_quantize_kernel<<<gv, QT, 0, stream>>>(static_cast<const uint16_t*>(V), s, v_scale,
                                             static_cast<uint8_t*>(v8));
    v_finalize_kernel<<<(nv + 255) / 256, 256, 0, stream>>>(v_scale, nv);
    count_launch(4);
    return cudaGetLastError();
}

}  // namespace chorus
