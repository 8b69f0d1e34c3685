// aux_kernels.cuh -- HBM-bound helpers around the attention backward (all elementwise / row-wise):
//   bwd_preprocess : delta[h,t] = <dO[t,h], O[t,h]>,  lse2 = LSE * log2(e),
//                    both padded to a multiple of 128 rows (+inf / 0) for the tile loads
//   acc_to_bf16    : fp32 staging [L,H,D] (contiguous) * scale -> bf16 strided output
// Each thread moves 16 bytes of bf16 (8 elements); rows are coalesced along d.
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>

namespace pf {

__device__ __forceinline__ float2 bf2_to_f2(uint32_t u) {
    return make_float2(__uint_as_float(u << 16), __uint_as_float(u & 0xffff0000u));
}

// grid: (ceil(Lpad * D/8 / 256), Hq); one row (t,h) is handled by D/8 consecutive threads
template <int D>
__global__ void __launch_bounds__(256)
bwd_preprocess_kernel(const __nv_bfloat16* __restrict__ O, int64_t o_st, int64_t o_sh,
                      const __nv_bfloat16* __restrict__ dO, int64_t do_st, int64_t do_sh,
                      const float* __restrict__ LSE, int64_t lse_stride, float* __restrict__ lse2,
                      float* __restrict__ delta, int64_t stat_stride, int Lq, int Lpad) {
    constexpr int TPR = D / 8;  // threads per row
    const int h = blockIdx.y;
    const int64_t gid = int64_t(blockIdx.x) * 256 + threadIdx.x;
    const int t = int(gid / TPR), c = int(gid % TPR);
    float acc = 0.f;
    if (t < Lq) {
        const uint4 a = *reinterpret_cast<const uint4*>(O + int64_t(t) * o_st + int64_t(h) * o_sh + c * 8);
        const uint4 b = *reinterpret_cast<const uint4*>(dO + int64_t(t) * do_st + int64_t(h) * do_sh + c * 8);
        const uint32_t aw[4] = {a.x, a.y, a.z, a.w}, bw[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float2 x = bf2_to_f2(aw[i]), y = bf2_to_f2(bw[i]);
            acc = fmaf(x.x, y.x, acc);
            acc = fmaf(x.y, y.y, acc);
        }
    }
#pragma unroll
    for (int o = TPR / 2; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (c == 0 && t < Lpad) {
        const bool ok = t < Lq;
        delta[int64_t(h) * stat_stride + t] = ok ? acc : 0.f;
        lse2[int64_t(h) * stat_stride + t] =
            ok ? LSE[int64_t(h) * lse_stride + t] * 1.4426950408889634f : __int_as_float(0x7f800000);
    }
}

// src fp32 [L, H, D] contiguous -> dst bf16 [L, H, D] strided, dst = bf16_rne(src * scale)
template <int D>
__global__ void __launch_bounds__(256)
acc_to_bf16_kernel(const float* __restrict__ src, __nv_bfloat16* __restrict__ dst, int64_t d_st,
                   int64_t d_sh, int64_t L, int H, float scale) {
    constexpr int TPR = D / 8;
    const int64_t gid = int64_t(blockIdx.x) * 256 + threadIdx.x;
    const int64_t row = gid / TPR;  // t * H + h
    const int c = int(gid % TPR);
    if (row >= L * H) return;
    const int64_t t = row / H;
    const int h = int(row % H);
    const float4 a = *reinterpret_cast<const float4*>(src + row * D + c * 8);
    const float4 b = *reinterpret_cast<const float4*>(src + row * D + c * 8 + 4);
    __nv_bfloat162 p0 = __floats2bfloat162_rn(a.x * scale, a.y * scale);
    __nv_bfloat162 p1 = __floats2bfloat162_rn(a.z * scale, a.w * scale);
    __nv_bfloat162 p2 = __floats2bfloat162_rn(b.x * scale, b.y * scale);
    __nv_bfloat162 p3 = __floats2bfloat162_rn(b.z * scale, b.w * scale);
    uint4 v;
    v.x = *reinterpret_cast<uint32_t*>(&p0);
    v.y = *reinterpret_cast<uint32_t*>(&p1);
    v.z = *reinterpret_cast<uint32_t*>(&p2);
    v.w = *reinterpret_cast<uint32_t*>(&p3);
    *reinterpret_cast<uint4*>(dst + t * d_st + int64_t(h) * d_sh + c * 8) = v;
}

}  // namespace pf
