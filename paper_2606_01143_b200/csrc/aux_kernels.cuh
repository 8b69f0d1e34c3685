// aux_kernels.cuh -- HBM-bound helpers around the attention backward (all elementwise / row-wise):
//   bwd_preprocess : delta[h,t] = <dO[t,h], O[t,h]>,  lse2 = LSE * log2(e),
//                    every sequence padded to a multiple of 64 rows (+inf / 0) for the tile loads;
//                    also zero-fills the fp32 dQ^T workspace the backward reduce-adds into and,
//                    when asked, the launch's fp32 dK2/dV2 staging
//   dq_finish      : fp32 dQ^T tile workspace of the backward -> bf16 dQ rows
//   acc2_to_bf16   : two fp32 accumulators [L,H,D] (contiguous: dK and dV) -> bf16 strided outputs
// Each thread moves 16 bytes of bf16 (8 elements); rows are coalesced along d.
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include "seq_table.cuh"

namespace pf {

__device__ __forceinline__ float2 bf2_to_f2(uint32_t u) {
    return make_float2(__uint_as_float(u << 16), __uint_as_float(u & 0xffff0000u));
}

// grid: (ceil(nQS*64 * D/8 / 256), Hq); one padded position is handled by D/8 consecutive threads.
// Padded positions: sequence s of the launch owns positions [64*pqs[s], 64*pqs[s+1]).
template <int D>
__global__ void __launch_bounds__(256)
bwd_preprocess_kernel(const __nv_bfloat16* __restrict__ O, int64_t o_st, int64_t o_sh,
                      const __nv_bfloat16* __restrict__ dO, int64_t do_st, int64_t do_sh,
                      const float* __restrict__ LSE, int64_t lse_stride, float* __restrict__ lse2,
                      float* __restrict__ delta, int64_t stat_stride, float4* __restrict__ dq_zero,
                      float4* __restrict__ zero_k, float4* __restrict__ zero_v, int64_t zero_n4,
                      const __grid_constant__ SeqTable seq) {
    constexpr int TPR = D / 8;  // threads per row
    const int h = blockIdx.y;
    const int64_t gid = int64_t(blockIdx.x) * 256 + threadIdx.x;
    const int pp = int(gid / TPR), c = int(gid % TPR);
    const int npad = seq.pqs[seq.n] * 64;
    {   // zero this head's share of the dQ^T workspace (npad * D floats = 2 float4 per thread)
        const int64_t n4 = int64_t(npad) * TPR * 2;
        float4* z = dq_zero + int64_t(h) * n4;
        const int64_t i0 = int64_t(blockIdx.x) * 512 + threadIdx.x;
        if (i0 < n4) z[i0] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (i0 + 256 < n4) z[i0 + 256] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    if (zero_k) {   // the launch's dK2/dV2 staging (zero_n4 float4 each), spread over the whole grid
        const int64_t nthr = int64_t(gridDim.x) * gridDim.y * 256;
        for (int64_t i = (int64_t(h) * gridDim.x + blockIdx.x) * 256 + threadIdx.x; i < zero_n4; i += nthr) {
            zero_k[i] = make_float4(0.f, 0.f, 0.f, 0.f);
            zero_v[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
    }
    int s = 0;
    while (s + 1 < seq.n && seq.pqs[s + 1] * 64 <= pp) ++s;
    const int tl = pp - seq.pqs[s] * 64;                       // row within its sequence
    const bool ok = pp < npad && tl < seq.cu[s + 1] - seq.cu[s];
    const int64_t t = seq.cu[s] + tl;                          // packed token row
    float acc = 0.f;
    if (ok) {
        const uint4 a = *reinterpret_cast<const uint4*>(O + t * o_st + int64_t(h) * o_sh + c * 8);
        const uint4 b = *reinterpret_cast<const uint4*>(dO + t * do_st + int64_t(h) * do_sh + c * 8);
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
    if (c == 0 && pp < npad) {
        delta[int64_t(h) * stat_stride + pp] = ok ? acc : 0.f;
        lse2[int64_t(h) * stat_stride + pp] =
            ok ? LSE[int64_t(h) * lse_stride + t] * 1.4426950408889634f : __int_as_float(0x7f800000);
    }
}

// dQ^T tiles of the backward (fp32, [Hq][nQS][2][D][32], 16-byte chunks of each 128-byte row
// xor-swizzled by d & 7) -> dQ bf16 [t, h, :] = bf16_rne(sigma * dQ).  grid (nQS, Hq), 256 threads.
// Transposed in registers: a thread owns 4 query rows (one logical 16-byte chunk lc of the 32-row
// half) x 8 consecutive d; for d = 8 dg + j that chunk sits at physical chunk lc ^ j, so the 8 loads
// of a thread are independent 16-byte reads (8 lanes cover one 128-byte line) and every store is one
// 16-byte piece of an output row.  No shared memory, no barrier.
template <int D>
__global__ void __launch_bounds__(256)
dq_finish_kernel(const float* __restrict__ acc, __nv_bfloat16* __restrict__ dst, int64_t d_st,
                 int64_t d_sh, float scale, const __grid_constant__ SeqTable seq) {
    const int qsg = blockIdx.x, h = blockIdx.y;
    const int nQS = seq.pqs[seq.n];
    int s = 0;
    while (s + 1 < seq.n && seq.pqs[s + 1] <= qsg) ++s;
    const int t0 = (qsg - seq.pqs[s]) * 64;                    // first row of the tile in its sequence
    const int Ls = seq.cu[s + 1] - seq.cu[s];
    const float4* src = reinterpret_cast<const float4*>(acc + (int64_t(h) * nQS + qsg) * (2 * D * 32));
    __nv_bfloat16* out = dst + (int64_t(seq.cu[s]) + t0) * d_st + int64_t(h) * d_sh;
    for (int u = threadIdx.x; u < 2 * (D / 8) * 8; u += 256) {
        const int lc = u & 7, dg = (u >> 3) % (D / 8), half = (u >> 3) / (D / 8);
        const int q0 = half * 32 + lc * 4;
        if (t0 + q0 >= Ls) continue;
        float4 v[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) v[j] = __ldcs(src + (half * D + dg * 8 + j) * 8 + (lc ^ j));
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            float r[8];
#pragma unroll
            for (int j = 0; j < 8; ++j)
                r[j] = (k == 0 ? v[j].x : k == 1 ? v[j].y : k == 2 ? v[j].z : v[j].w) * scale;
            if (t0 + q0 + k >= Ls) break;
            __nv_bfloat162 p0 = __floats2bfloat162_rn(r[0], r[1]);
            __nv_bfloat162 p1 = __floats2bfloat162_rn(r[2], r[3]);
            __nv_bfloat162 p2 = __floats2bfloat162_rn(r[4], r[5]);
            __nv_bfloat162 p3 = __floats2bfloat162_rn(r[6], r[7]);
            uint4 w;
            w.x = *reinterpret_cast<uint32_t*>(&p0);
            w.y = *reinterpret_cast<uint32_t*>(&p1);
            w.z = *reinterpret_cast<uint32_t*>(&p2);
            w.w = *reinterpret_cast<uint32_t*>(&p3);
            *reinterpret_cast<uint4*>(out + int64_t(q0 + k) * d_st + dg * 8) = w;
        }
    }
}

// Two fp32 accumulators [L, H, D] contiguous (dK and dV) -> two bf16 strided outputs in one launch:
// blockIdx.y selects the pair; dst = bf16_rne(src)
template <int D>
__global__ void __launch_bounds__(256)
acc2_to_bf16_kernel(const float* __restrict__ src0, __nv_bfloat16* __restrict__ dst0, int64_t st0,
                    int64_t sh0, const float* __restrict__ src1, __nv_bfloat16* __restrict__ dst1,
                    int64_t st1, int64_t sh1, int64_t L, int H) {
    constexpr int TPR = D / 8;
    const bool second = blockIdx.y != 0;
    const float* src = second ? src1 : src0;
    __nv_bfloat16* dst = second ? dst1 : dst0;
    const int64_t d_st = second ? st1 : st0, d_sh = second ? sh1 : sh0;
    const int64_t gid = int64_t(blockIdx.x) * 256 + threadIdx.x;
    const int64_t row = gid / TPR;  // t * H + h
    const int c = int(gid % TPR);
    if (row >= L * H) return;
    const int64_t t = row / H;
    const int h = int(row % H);
    const float4 a = *reinterpret_cast<const float4*>(src + row * D + c * 8);
    const float4 b = *reinterpret_cast<const float4*>(src + row * D + c * 8 + 4);
    __nv_bfloat162 p0 = __floats2bfloat162_rn(a.x, a.y);
    __nv_bfloat162 p1 = __floats2bfloat162_rn(a.z, a.w);
    __nv_bfloat162 p2 = __floats2bfloat162_rn(b.x, b.y);
    __nv_bfloat162 p3 = __floats2bfloat162_rn(b.z, b.w);
    uint4 v;
    v.x = *reinterpret_cast<uint32_t*>(&p0);
    v.y = *reinterpret_cast<uint32_t*>(&p1);
    v.z = *reinterpret_cast<uint32_t*>(&p2);
    v.w = *reinterpret_cast<uint32_t*>(&p3);
    *reinterpret_cast<uint4*>(dst + t * d_st + int64_t(h) * d_sh + c * 8) = v;
}

}  // namespace pf
