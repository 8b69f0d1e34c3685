// companions.cuh -- the two companions of the attention path:
//   rope_kernel          rotary position embedding of a packed bf16 tensor, in place, with positions
//                        that continue after the prefix; HBM-bound, one block per token
//   kv_proj_grad_kernel  dW += X^T dY, the K/V-projection weight gradient term of one phase
//                        (PAPER.md:212); tcgen05 MMAs with both operands MN-major straight from
//                        TMA-staged [tokens][64] tiles, fp32 accumulator in TMEM, vector reduce-add
//                        into dW (so that the token range can be split over CTAs)
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include "sm100_ptx.cuh"
#include "seq_table.cuh"

namespace pf {

constexpr int kRopeMaxHalf = 128;   // head_dim <= 256

struct RopeFreq {
    double inv[kRopeMaxHalf];       // theta_base^(-2j/d), formed on the host in fp64
};

// grid: one block per packed token row, 128 threads.  Shared memory: cos / sin of the row's d/2 angles.
__global__ void __launch_bounds__(128)
rope_kernel(__nv_bfloat16* __restrict__ X, int64_t st, int64_t sh, int H, int d, int64_t pos0, int inverse,
            const __grid_constant__ SeqTable seq, const __grid_constant__ RopeFreq fr) {
    __shared__ float cs[kRopeMaxHalf], sn[kRopeMaxHalf];
    const int r = blockIdx.x, half = d >> 1;
    int s = 0;
    while (s + 1 < seq.n && seq.cu[s + 1] <= r) ++s;
    const double pos = double(pos0 + (r - seq.cu[s]));
    for (int j = threadIdx.x; j < half; j += 128) {
        double a = pos * fr.inv[j];
        a -= 6.283185307179586 * rint(a * 0.15915494309189535);   // |a| <= pi, exact enough in fp64
        float sv, cv;
        sincosf(float(a), &sv, &cv);
        cs[j] = cv;
        sn[j] = inverse ? -sv : sv;
    }
    __syncthreads();
    const int cpr = half >> 3;                                  // 16-byte chunks per half row
    for (int i = threadIdx.x; i < H * cpr; i += 128) {
        const int h = i / cpr, j0 = (i % cpr) << 3;
        __nv_bfloat16* lo = X + int64_t(r) * st + int64_t(h) * sh + j0;
        __nv_bfloat16* hi = lo + half;
        uint4 a = *reinterpret_cast<const uint4*>(lo), b = *reinterpret_cast<const uint4*>(hi);
        uint32_t aw[4] = {a.x, a.y, a.z, a.w}, bw[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const float x0 = __uint_as_float(aw[k] << 16), x1 = __uint_as_float(aw[k] & 0xffff0000u);
            const float y0 = __uint_as_float(bw[k] << 16), y1 = __uint_as_float(bw[k] & 0xffff0000u);
            const float c0 = cs[j0 + 2 * k], s0 = sn[j0 + 2 * k], c1 = cs[j0 + 2 * k + 1], s1 = sn[j0 + 2 * k + 1];
            aw[k] = pack_bf16(x0 * c0 - y0 * s0, x1 * c1 - y1 * s1);
            bw[k] = pack_bf16(y0 * c0 + x0 * s0, y1 * c1 + x1 * s1);
        }
        *reinterpret_cast<uint4*>(lo) = make_uint4(aw[0], aw[1], aw[2], aw[3]);
        *reinterpret_cast<uint4*>(hi) = make_uint4(bw[0], bw[1], bw[2], bw[3]);
    }
}

// ---------------------------------------------------------------------------------------------
// dW[M, N] (fp32, row-major) += X[L, M]^T dY[L, N]      (M = d_model, N = Hkv * d, K = tokens)
// Both operands are read as they lie in memory -- token rows, feature columns contiguous -- i.e.
// MN-major for the tensor core: A = X^T and B = dY come from TMA boxes of [64 tokens][64 features]
// (swizzle-128B), no transpose pass.  CTA = one (128 MH) x BN tile of dW over a range of 64-token
// chunks (grid.z splits the token range); fp32 accumulators = MH x BN TMEM columns.  Tile size is what
// bounds the main loop: a chunk of 64 tokens costs (128 MH + BN) x 128 bytes of L2 -> shared-memory
// traffic for MH x BN / 2 clocks of MMA, i.e. 128 B/clk at 128 x 128, 64 B/clk at 256 x 256 against
// the ~73 B/clk/SM the L2 delivers (profiles/r2_kernel_experiments.md).
// Epilogue: each thread copies its accumulator row (BN fp32) from TMEM into the idle operand ring and
// adds it into dW with ONE bulk reduce-add of BN x 4 contiguous bytes, so splits and successive calls
// (prefix term, suffix terms) sum.
//   warp 0 TMA producer | warp 1 TMEM alloc + tcgen05.mma issuer | warps 2-5 epilogue
// ---------------------------------------------------------------------------------------------
template <int MH, int BN>
struct GemmCfg {
    static constexpr int SUB = 64 * 128;               // [64 tokens][64 bf16] box
    static constexpr int ABOX = 2 * MH, BBOX = BN / 64;
    static constexpr int STAGE = (ABOX + BBOX) * SUB;
    static constexpr int ST = (200 * 1024) / STAGE > 4 ? 4 : (200 * 1024) / STAGE;   // ring depth
    static constexpr int OFF_BAR = ST * STAGE;
    static constexpr int SMEM = OFF_BAR + 256;
    static constexpr int THREADS = 192;
    static constexpr int TMEM_COLS = MH * BN;
    static constexpr int EPI_ROW = BN * 4 + 16;        // staged accumulator row, padded against bank conflicts
    static_assert(TMEM_COLS == 128 || TMEM_COLS == 256 || TMEM_COLS == 512, "TMEM allocation is a power of two");
    static_assert(ST >= 3, "ring too shallow");
    static_assert(128 * EPI_ROW <= OFF_BAR, "epilogue staging must fit the operand ring");
};

__device__ __forceinline__ void tma_load_2d(void* dst, const void* tmap, uint64_t* bar, int c0, int c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes"
        " [%0], [%1, {%3, %4}], [%2];"
        ::"r"(smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(tmap)), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
        : "memory");
}
// shared -> global, element-wise fp32 add of `bytes` contiguous bytes (bulk async-group of the thread)
__device__ __forceinline__ void bulk_red_add_row(float* dst, const void* src, uint32_t bytes) {
    asm volatile(
        "cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f32 [%0], [%1], %2;"
        ::"l"(reinterpret_cast<uint64_t>(dst)), "r"(smem_u32(src)), "r"(bytes)
        : "memory");
}

template <int MH, int BN>
__global__ void __launch_bounds__(192, 1)
kv_proj_grad_kernel(const __grid_constant__ CUtensorMap tmX, const __grid_constant__ CUtensorMap tmY,
                    float* __restrict__ dW, int n_cols, int n_chunks, int chunks_per_split) {
    using C = GemmCfg<MH, BN>;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
    uint64_t* bar_full = bars;              // [ST]
    uint64_t* bar_empty = bars + C::ST;     // [ST]
    uint64_t* bar_done = bars + 2 * C::ST;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * C::ST + 1);
    const int tid = threadIdx.x, warp = tid >> 5;
    if ((smem_u32(smem) & 1023u) != 0) __trap();
    const int m0 = blockIdx.x * (128 * MH), n0 = blockIdx.y * BN;
    const int c_lo = blockIdx.z * chunks_per_split;
    const int n_it = min(n_chunks, c_lo + chunks_per_split) - c_lo;   // >= 1 by construction of the grid

    if (tid == 0) {
        for (int s = 0; s < C::ST; ++s) { mbar_init(&bar_full[s], 1); mbar_init(&bar_empty[s], 1); }
        mbar_init(bar_done, 1);
        fence_mbar_init();
    }
    if (warp == 1) tmem_alloc(tmem_slot, C::TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp == 0) {
        if (elect_one()) {
            tma_prefetch_desc(&tmX); tma_prefetch_desc(&tmY);
            for (int it = 0; it < n_it; ++it) {
                const int st = it % C::ST, k0 = (c_lo + it) * 64;
                uint8_t* base = smem + st * C::STAGE;
                mbar_wait(&bar_empty[st], ((it / C::ST) & 1) ^ 1);
                mbar_arrive_expect_tx(&bar_full[st], C::STAGE);
#pragma unroll
                for (int i = 0; i < C::ABOX; ++i) tma_load_2d(base + i * C::SUB, &tmX, &bar_full[st], m0 + 64 * i, k0);
#pragma unroll
                for (int i = 0; i < C::BBOX; ++i)
                    tma_load_2d(base + (C::ABOX + i) * C::SUB, &tmY, &bar_full[st], n0 + 64 * i, k0);
            }
        }
    } else if (warp == 1) {
        if (elect_one()) {
            constexpr uint32_t idesc = make_idesc_bf16(128, BN, true, true);
            for (int it = 0; it < n_it; ++it) {
                const int st = it % C::ST;
                const uint32_t sa = smem_u32(smem + st * C::STAGE);
                const uint64_t ad = make_smem_desc_sw128(sa, C::SUB, 1024);                      // X^T, MN-major
                const uint64_t bd = make_smem_desc_sw128(sa + C::ABOX * C::SUB, C::SUB, 1024);   // dY, MN-major
                mbar_wait(&bar_full[st], (it / C::ST) & 1);
                tc_fence_after();
#pragma unroll
                for (int kk = 0; kk < 4; ++kk)          // 16 tokens per instruction
#pragma unroll
                    for (int mh = 0; mh < MH; ++mh)     // 128 features of X per instruction, dY shared
                        mma_ss(tmem + mh * BN, ad + ((mh * 2 * C::SUB + kk * 2048) >> 4), bd + ((kk * 2048) >> 4),
                               idesc, (it > 0 || kk > 0) ? 1u : 0u);
                mma_commit(&bar_empty[st]);
            }
            mma_commit(bar_done);
        }
    } else {
        // epilogue: thread <-> TMEM lane <-> row of a 128-row half.  bar_done = every MMA complete, hence
        // every operand stage read: the ring is free and stages the rows.  A thread touches only its
        // own staged row, so the only ordering needed is its own bulk group.
        const int q = warp & 3, r = q * 32 + (tid & 31);
        const uint32_t lane_off = uint32_t(q * 32) << 16;
        uint8_t* stage = smem + r * C::EPI_ROW;
        mbar_wait(bar_done, 0);
        tc_fence_after();
#pragma unroll 1
        for (int mh = 0; mh < MH; ++mh) {
            if (mh > 0) bulk_wait_read<0>();            // the previous half's row has been read out
#pragma unroll 1
            for (int c = 0; c < BN / 32; ++c) {
                uint32_t v[32];
                tmem_ld32(tmem + mh * BN + c * 32 + lane_off, v);
                tmem_wait_ld();
#pragma unroll
                for (int k = 0; k < 8; ++k)
                    *reinterpret_cast<uint4*>(stage + c * 128 + k * 16) =
                        make_uint4(v[4 * k], v[4 * k + 1], v[4 * k + 2], v[4 * k + 3]);
            }
            fence_proxy_async_smem();
            bulk_red_add_row(dW + int64_t(m0 + mh * 128 + r) * n_cols + n0, stage, BN * 4);
            bulk_commit();
        }
        bulk_wait<0>();
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem, C::TMEM_COLS);
}


}  // namespace pf
