// attn_bwd.cuh -- sm_100a attention backward, KV-stationary, two KV sources.
//
// For one KV tile of 128 keys (of KV head g) and a range of query heads of that group, loop over
// the query tiles that see it and issue the five contractions of flash backward
// (PAPER.md:194-198):
//     S^T  = K Q^T                 dP^T = V dO^T
//     P^T  = exp(sigma S^T - LSE)  dS^T = P^T o (dP^T - delta)
//     dV  += P^T dO                dK  += dS^T Q            dQ_tile = dS K
// dV and dK stay in TMEM for the whole loop (summing the G query heads of the KV head and all
// query tiles) and are added once into an fp32 accumulator [L, Hkv, d]: for prefix-source keys
// that accumulator IS the persistent gK1 / gV1 of the training-time KV cache -
// Phase B adds the coupling term, Phase C adds the own-prefix term on top of it.  dQ tiles are
// added into an fp32 workspace [Lq, Hq, d] (several KV tiles contribute to one query tile).
//
//   warps 0-3  compute (thread j <-> key row j <-> TMEM lane j; for dQ: lane = query row)
//   warp  4    TMA producer (K, V once; Q, dO, LSE, delta tiles through a 2-stage ring)
//   warp  5    tcgen05.mma issuer (one thread)
// TMEM (512 columns): S^T/P^T [0,128) | dP^T / dQ [128,256) | dV [256,256+D) | dK [256+D,256+2D)
#pragma once
#include <cuda.h>
#include "sm100_ptx.cuh"

namespace pf {

struct BwdParams {
    float* dQacc;                  // [Lq, Hq, D] fp32, contiguous
    float* accK1; float* accV1;    // prefix-source accumulators [Lp, Hkv, D] fp32 (gK1 / gV1)
    float* accK2; float* accV2;    // causal-source accumulators [Lq, Hkv, D] fp32
    const float* lse2;             // [Hq, Lpad] LSE * log2(e); +inf beyond Lq
    const float* delta;            // [Hq, Lpad] rowsum(dO o O); 0 beyond Lq
    int64_t stat_stride;           // Lpad (multiple of 128)
    int Lq, Lp;
    int Hq, Hkv, G;
    int nQT;                       // ceil(Lq / 128)
    int nPT;                       // ceil(Lp / 128)
    int parts, hpp;                // head parts per KV head, heads per part
    float scale_log2;              // sigma * log2(e)
    float sigma;
};

template <int D>
struct BwdCfg {
    static constexpr int QS = 2;                       // Q/dO ring depth
    static constexpr int TILE = 128 * D * 2;
    static constexpr int SUB = 128 * 64 * 2;
    static constexpr int NSUB = D / 64;
    static constexpr int OFF_K = 0;
    static constexpr int OFF_V = TILE;
    static constexpr int OFF_Q = 2 * TILE;             // QS tiles
    static constexpr int OFF_DO = OFF_Q + QS * TILE;   // QS tiles
    static constexpr int OFF_DS = OFF_DO + QS * TILE;  // 128 x 128 bf16 = 32 KB
    static constexpr int OFF_STAT = OFF_DS + 32768;    // QS x (lse2[128], delta[128]) fp32
    static constexpr int OFF_BAR = OFF_STAT + QS * 1024;
    static constexpr int SMEM = OFF_BAR + 128;
    static constexpr int THREADS = 192;
};

__device__ __forceinline__ void bulk_load_1d(void* dst, const void* src, uint32_t bytes,
                                             uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        ::"r"(smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(src)), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

template <int D>
__global__ void __launch_bounds__(192, 1)
attn_bwd_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmdO,
                const __grid_constant__ CUtensorMap tmK1, const __grid_constant__ CUtensorMap tmV1,
                const __grid_constant__ CUtensorMap tmK2, const __grid_constant__ CUtensorMap tmV2,
                const BwdParams p) {
    using C = BwdCfg<D>;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
    uint64_t* bar_KV = bars;            // K and V landed
    uint64_t* bar_Qf = bars + 1;        // [QS] Q, dO, lse2, delta tile landed
    uint64_t* bar_Qe = bars + 3;        // [QS] tile consumed
    uint64_t* bar_S = bars + 5;         // S^T and dP^T ready
    uint64_t* bar_P = bars + 6;         // P^T (TMEM) and dS^T (smem) ready
    uint64_t* bar_dQ = bars + 7;        // dQ tile (and dV, dK so far) ready
    uint64_t* bar_dQfree = bars + 8;    // dQ tile read out of TMEM
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 10);

    const int tid = threadIdx.x, warp = tid >> 5;
    if ((smem_u32(smem) & 1023u) != 0) __trap();

    // ---- item decode: prefix-source items first (heaviest), then causal tiles 0, 1, ... ----
    const int per_tile = p.Hkv * p.parts;
    int item = blockIdx.x;
    const bool pre = item < p.nPT * per_tile;
    if (!pre) item -= p.nPT * per_tile;
    const int kt = item / per_tile;                         // KV tile within its source
    const int g = (item % per_tile) / p.parts;
    const int part = item % p.parts;
    const int h_lo = g * p.G + part * p.hpp;
    const int h_hi = min(g * p.G + p.G, h_lo + p.hpp);
    const int qt_lo = pre ? 0 : kt;                         // first query tile that sees this tile
    const int n_qt = p.nQT - qt_lo;
    const int n_iter = max(0, (h_hi - h_lo)) * n_qt;
    const int Lkv = pre ? p.Lp : p.Lq;
    const int kv0 = kt * 128;

    if (tid == 0) {
        mbar_init(bar_KV, 1);
        for (int s = 0; s < C::QS; ++s) { mbar_init(&bar_Qf[s], 1); mbar_init(&bar_Qe[s], 1); }
        mbar_init(bar_S, 1); mbar_init(bar_P, 128); mbar_init(bar_dQ, 1); mbar_init(bar_dQfree, 128);
        fence_mbar_init();
    }
    if (warp == 4) {
        tmem_alloc(tmem_slot, 512);
        if (elect_one()) {
            tma_prefetch_desc(&tmQ); tma_prefetch_desc(&tmdO);
            tma_prefetch_desc(pre ? &tmK1 : &tmK2); tma_prefetch_desc(pre ? &tmV1 : &tmV2);
        }
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    constexpr uint32_t T_ST = 0, T_DP = 128, T_DV = 256, T_DK = 256 + D;

    if (warp == 4) {
        // =============================== TMA producer ===============================
        if (elect_one() && n_iter > 0) {
            mbar_arrive_expect_tx(bar_KV, 2 * C::TILE);
            for (int k = 0; k < C::NSUB; ++k) {
                tma_load_3d(smem + C::OFF_K + k * C::SUB, pre ? &tmK1 : &tmK2, bar_KV, 64 * k, g, kv0);
                tma_load_3d(smem + C::OFF_V + k * C::SUB, pre ? &tmV1 : &tmV2, bar_KV, 64 * k, g, kv0);
            }
            int it = 0;
            for (int h = h_lo; h < h_hi; ++h) {
                for (int qt = qt_lo; qt < p.nQT; ++qt, ++it) {
                    const int st = it % C::QS;
                    const uint32_t ph = (it / C::QS) & 1;
                    mbar_wait(&bar_Qe[st], ph ^ 1);
                    mbar_arrive_expect_tx(&bar_Qf[st], 2 * C::TILE + 1024);
                    for (int k = 0; k < C::NSUB; ++k) {
                        tma_load_3d(smem + C::OFF_Q + st * C::TILE + k * C::SUB, &tmQ, &bar_Qf[st],
                                    64 * k, h, qt * 128);
                        tma_load_3d(smem + C::OFF_DO + st * C::TILE + k * C::SUB, &tmdO, &bar_Qf[st],
                                    64 * k, h, qt * 128);
                    }
                    float* stat = reinterpret_cast<float*>(smem + C::OFF_STAT + st * 1024);
                    bulk_load_1d(stat, p.lse2 + int64_t(h) * p.stat_stride + qt * 128, 512, &bar_Qf[st]);
                    bulk_load_1d(stat + 128, p.delta + int64_t(h) * p.stat_stride + qt * 128, 512,
                                 &bar_Qf[st]);
                }
            }
        }
    } else if (warp == 5) {
        // =============================== MMA issuer ===============================
        if (elect_one() && n_iter > 0) {
            constexpr uint32_t id_kk = make_idesc_bf16(128, 128, false, false);  // S^T, dP^T
            constexpr uint32_t id_kmn = make_idesc_bf16(128, D, false, true);    // dV, dK
            constexpr uint32_t id_mnmn = make_idesc_bf16(128, D, true, true);    // dQ
            const uint32_t sK = smem_u32(smem + C::OFF_K), sV = smem_u32(smem + C::OFF_V),
                           sdS = smem_u32(smem + C::OFF_DS);
            mbar_wait(bar_KV, 0);
            for (int it = 0; it < n_iter; ++it) {
                const int st = it % C::QS;
                const uint32_t ph = (it / C::QS) & 1;
                const uint32_t sQ = smem_u32(smem + C::OFF_Q + st * C::TILE);
                const uint32_t sdO = smem_u32(smem + C::OFF_DO + st * C::TILE);
                mbar_wait(&bar_Qf[st], ph);
                if (it > 0) mbar_wait(bar_dQfree, (it - 1) & 1);  // dP^T region still holds dQ
                tc_fence_after();
#pragma unroll
                for (int kk = 0; kk < D / 16; ++kk) {  // S^T = K Q^T
                    const uint32_t off = (kk >> 2) * C::SUB + (kk & 3) * 32;
                    mma_ss(tmem + T_ST, make_smem_desc_sw128(sK + off, 16, 1024),
                           make_smem_desc_sw128(sQ + off, 16, 1024), id_kk, kk > 0);
                }
#pragma unroll
                for (int kk = 0; kk < D / 16; ++kk) {  // dP^T = V dO^T
                    const uint32_t off = (kk >> 2) * C::SUB + (kk & 3) * 32;
                    mma_ss(tmem + T_DP, make_smem_desc_sw128(sV + off, 16, 1024),
                           make_smem_desc_sw128(sdO + off, 16, 1024), id_kk, kk > 0);
                }
                mma_commit(bar_S);
                mbar_wait(bar_P, it & 1);
                tc_fence_after();
#pragma unroll
                for (int kk = 0; kk < 8; ++kk)  // dV += P^T dO   (A from TMEM, B = dO MN-major)
                    mma_ts(tmem + T_DV, tmem + T_ST + kk * 8,
                           make_smem_desc_sw128(sdO + kk * 2048, C::SUB, 1024), id_kmn,
                           (it > 0 || kk > 0) ? 1u : 0u);
#pragma unroll
                for (int kk = 0; kk < 8; ++kk) {  // dK += dS^T Q  (A = dS^T K-major, B = Q MN-major)
                    const uint32_t off = (kk >> 2) * C::SUB + (kk & 3) * 32;
                    mma_ss(tmem + T_DK, make_smem_desc_sw128(sdS + off, 16, 1024),
                           make_smem_desc_sw128(sQ + kk * 2048, C::SUB, 1024), id_kmn,
                           (it > 0 || kk > 0) ? 1u : 0u);
                }
#pragma unroll
                for (int kk = 0; kk < 8; ++kk)  // dQ = dS K  (A = dS^T read MN-major, B = K MN-major)
                    mma_ss(tmem + T_DP, make_smem_desc_sw128(sdS + kk * 2048, C::SUB, 1024),
                           make_smem_desc_sw128(sK + kk * 2048, C::SUB, 1024), id_mnmn, kk > 0);
                mma_commit(&bar_Qe[st]);
                mma_commit(bar_dQ);
            }
        }
    } else if (n_iter > 0) {
        // =============================== compute warps ===============================
        const int j = tid;                                   // key row in tile / query row for dQ
        const uint32_t lane_off = uint32_t(warp * 32) << 16;
        const int kj = kv0 + j;                              // key index within its source
        uint8_t* sdS = smem + C::OFF_DS;
        int it = 0;
        for (int h = h_lo; h < h_hi; ++h) {
            for (int qt = qt_lo; qt < p.nQT; ++qt, ++it) {
                const int st = it % C::QS;
                const float* s_lse = reinterpret_cast<const float*>(smem + C::OFF_STAT + st * 1024);
                const float* s_dl = s_lse + 128;
                mbar_wait(&bar_Qf[st], (it / C::QS) & 1);    // lse2 / delta tile visible
                mbar_wait(bar_S, it & 1);
                tc_fence_after();
                // visible query columns t' of this tile for key kj: causal => t >= kj
                const int t0 = qt * 128;
                int first = 0;                               // first visible column
                if (!pre) first = kj - t0;                   // may be <= 0 (all visible) or > 127
                const bool key_ok = kj < Lkv;
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    uint32_t s[32], dp[32];
                    tmem_ld32(tmem + T_ST + c * 32 + lane_off, s);
                    tmem_ld32(tmem + T_DP + c * 32 + lane_off, dp);
                    tmem_wait_ld();
                    uint32_t pk[16], dsk[16];
#pragma unroll
                    for (int q = 0; q < 32; q += 2) {
                        const int col = c * 32 + q;
                        float p0 = fast_exp2(fmaf(__uint_as_float(s[q]), p.scale_log2, -s_lse[col]));
                        float p1 = fast_exp2(fmaf(__uint_as_float(s[q + 1]), p.scale_log2, -s_lse[col + 1]));
                        if (!key_ok || col < first) p0 = 0.f;
                        if (!key_ok || col + 1 < first) p1 = 0.f;
                        const float d0 = p0 * (__uint_as_float(dp[q]) - s_dl[col]);
                        const float d1 = p1 * (__uint_as_float(dp[q + 1]) - s_dl[col + 1]);
                        pk[q >> 1] = pack_bf16(p0, p1);
                        dsk[q >> 1] = pack_bf16(d0, d1);
                    }
                    // P^T -> TMEM (bf16 pairs): columns [16c, 16c+16) of the S^T region
                    tmem_st16(tmem + T_ST + c * 16 + lane_off, pk);
                    // dS^T -> smem, K-major swizzle-128B tiles [128 keys][64 queries]
                    uint8_t* row = sdS + (c >> 1) * C::SUB + j * 128;
#pragma unroll
                    for (int ch = 0; ch < 4; ++ch) {
                        const int chunk = (c & 1) * 4 + ch;
                        *reinterpret_cast<uint4*>(row + ((chunk ^ (j & 7)) << 4)) =
                            make_uint4(dsk[ch * 4], dsk[ch * 4 + 1], dsk[ch * 4 + 2], dsk[ch * 4 + 3]);
                    }
                }
                tmem_wait_st();
                fence_proxy_async_smem();
                tc_fence_before();
                mbar_arrive(bar_P);
                // ---- dQ tile: lane = query row ----
                mbar_wait(bar_dQ, it & 1);
                tc_fence_after();
                const int t = t0 + j;
                float* dq = p.dQacc + (int64_t(t) * p.Hq + h) * D;
#pragma unroll
                for (int c = 0; c < D / 32; ++c) {
                    uint32_t v[32];
                    tmem_ld32(tmem + T_DP + c * 32 + lane_off, v);
                    tmem_wait_ld();
                    if (t < p.Lq) {
#pragma unroll
                        for (int q = 0; q < 32; q += 4)
                            red_add_v4(dq + c * 32 + q, __uint_as_float(v[q]), __uint_as_float(v[q + 1]),
                                       __uint_as_float(v[q + 2]), __uint_as_float(v[q + 3]));
                    }
                }
                tc_fence_before();
                mbar_arrive(bar_dQfree);
            }
        }
        // ---- epilogue: dV, dK rows of this KV tile -> fp32 accumulators ----
        // (the last bar_dQ commit covers every MMA issued before it)
        {
            const bool ok = kj < Lkv;  // ragged last tile: loads stay warp-uniform, stores are predicated
            float* av = (pre ? p.accV1 : p.accV2) + (int64_t(kj) * p.Hkv + g) * D;
            float* ak = (pre ? p.accK1 : p.accK2) + (int64_t(kj) * p.Hkv + g) * D;
#pragma unroll 1
            for (int c = 0; c < D / 32; ++c) {
                uint32_t v[32];
                tmem_ld32(tmem + T_DV + c * 32 + lane_off, v);
                tmem_wait_ld();
                if (ok) {
#pragma unroll
                    for (int q = 0; q < 32; q += 4)
                        red_add_v4(av + c * 32 + q, __uint_as_float(v[q]), __uint_as_float(v[q + 1]),
                                   __uint_as_float(v[q + 2]), __uint_as_float(v[q + 3]));
                }
                tmem_ld32(tmem + T_DK + c * 32 + lane_off, v);
                tmem_wait_ld();
                if (ok) {
#pragma unroll
                    for (int q = 0; q < 32; q += 4)
                        red_add_v4(ak + c * 32 + q, __uint_as_float(v[q]) * p.sigma,
                                   __uint_as_float(v[q + 1]) * p.sigma, __uint_as_float(v[q + 2]) * p.sigma,
                                   __uint_as_float(v[q + 3]) * p.sigma);
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 4) tmem_dealloc(tmem, 512);
}

}  // namespace pf
