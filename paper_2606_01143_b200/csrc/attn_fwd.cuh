// attn_fwd.cuh -- sm_100a attention forward with two KV sources, packed sequences.
//
//   O[t,h] = softmax_j( sigma <q[h,t], k[g,j]> ) v[g,j],   LSE[h,t] = log sum_j exp(sigma <q,k>)
//
// KV source 1 ("prefix", length Lp): every key is visible to every query (cached K1/V1, read in
// place -- no concat copy).  KV source 2 ("causal"): the keys of the query's own sequence, key j
// visible to query t iff j <= t.  Phase A / replay: Lp = 0, one sequence.  Phase B: source 1 = the
// cached prefix, the sequences are the suffixes of the wave packed along the token axis.
//
// One CTA = two query tiles of 128 rows ("slots": consecutive (row block, q head) items of one KV
// head and one sequence, so both read the same K/V stream) ping-ponged on the tensor core:
//   warps 0-7   softmax of slot 0: warps 0-3 key columns [0,64), warps 4-7 key columns [64,128)
//   warps 8-15  softmax of slot 1   (thread r of a warpgroup <-> query row r <-> TMEM lane r)
//   warp  16    TMA producer (Q once, K/V tiles through a 2-stage ring)
//   warp  17    tcgen05.mma issuer (one thread)
// TMEM (512 columns): S0 | S1 | O0 | O1, 128 fp32 columns each; each column half of P (bf16, 32
// columns) overwrites the start of its own half of S and is consumed from TMEM as the A operand of
// P.V; the two halves are handed over separately.  The two warpgroups of a slot exchange their
// partial row maxima through shared memory once per KV tile.
// A quarter of the exponentials is evaluated by a degree-3 polynomial on the FMA pipe, the rest by
// MUFU.EX2 (16 / clk / SM, which alone would tie with the tensor pipe).
#pragma once
#include <cuda.h>
#include "sm100_ptx.cuh"
#include "seq_table.cuh"

// exp2 evaluations (per 16 pairs) done by the polynomial on the FMA pipe instead of MUFU.EX2
#ifndef PF_FWD_POLY16
#define PF_FWD_POLY16 5
#endif

namespace pf {

struct FwdParams {
    __nv_bfloat16* O;
    int64_t o_stride_tok, o_stride_head;  // elements
    float* LSE;                           // [Hq, lse_stride], column = packed token row
    int64_t lse_stride;
    int Lp;        // prefix-source keys (0: none)
    int Hq, Hkv, G;
    float scale_log2;  // sigma * log2(e)
    SeqTable seq;
};

template <int D>
struct FwdCfg {
    static constexpr int KS = 2;                       // K/V ring depth
    static constexpr int TILE = 128 * D * 2;           // bytes of one 128 x D bf16 tile
    static constexpr int SUB = 128 * 64 * 2;           // one 128 x 64 swizzle-128B sub-tile
    static constexpr int NSUB = D / 64;
    static constexpr int OFF_Q = 0;                    // 2 tiles
    static constexpr int OFF_K = 2 * TILE;             // KS tiles
    static constexpr int OFF_V = OFF_K + KS * TILE;    // KS tiles
    static constexpr int OFF_BAR = OFF_V + KS * TILE;
    static constexpr int OFF_X = OFF_BAR + 256;        // row-max / row-sum exchange between column halves
    static constexpr int SMEM = OFF_X + 2 * 2 * 2 * 128 * 4;
    static constexpr int THREADS = 576;
};

// 2^x for a pair of x <= ~8 on the FMA / ALU pipes (packed f32x2 math): round-to-nearest split
// x = j + f, |f| <= 1/2, degree-3 minimax polynomial for 2^f (max relative error 7.5e-5, far below
// the bf16 rounding of P), and the exponent added with an integer shift-add.  x is clamped at -126
// (result ~ 1e-38, i.e. 0 for P).  Finite inputs only.
__device__ __forceinline__ float2 exp2_poly2(float2 x) {
    x.x = fmaxf(x.x, -126.f);
    x.y = fmaxf(x.y, -126.f);
    const float2 magic = make_float2(12582912.f, 12582912.f);   // 1.5 * 2^23: integer in the low mantissa bits
    const float2 t = __fadd2_rn(x, magic);
    const float2 f = __fadd2_rn(x, __fadd2_rn(make_float2(12582912.f, 12582912.f), make_float2(-t.x, -t.y)));
    float2 r = __ffma2_rn(f, make_float2(0.05517164617776871f, 0.05517164617776871f),
                          make_float2(0.2426111251115799f, 0.2426111251115799f));
    r = __ffma2_rn(r, f, make_float2(0.6932609677314758f, 0.6932609677314758f));
    r = __ffma2_rn(r, f, make_float2(0.9999280571937561f, 0.9999280571937561f));
    return make_float2(__int_as_float(__float_as_int(r.x) + (__float_as_int(t.x) << 23)),
                       __int_as_float(__float_as_int(r.y) + (__float_as_int(t.y) << 23)));
}

template <int D>
__global__ void __launch_bounds__(576, 1)
attn_fwd_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK1,
                const __grid_constant__ CUtensorMap tmV1, const __grid_constant__ CUtensorMap tmK2,
                const __grid_constant__ CUtensorMap tmV2, const __grid_constant__ FwdParams p) {
    using C = FwdCfg<D>;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
    uint64_t* bar_Q = bars;                 // [2]
    uint64_t* bar_Kf = bars + 2;            // [KS]
    uint64_t* bar_Ke = bars + 4;
    uint64_t* bar_Vf = bars + 6;
    uint64_t* bar_Ve = bars + 8;
    uint64_t* bar_S = bars + 10;            // [2] S_s ready (MMA -> softmax)
    uint64_t* bar_P = bars + 12;            // [2 slots][2 halves] P_s half ready (softmax -> MMA)
    uint64_t* bar_done = bars + 16;         // all MMAs complete
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 17);

    const int tid = threadIdx.x, warp = tid >> 5;
    if ((smem_u32(smem) & 1023u) != 0) __trap();

    // ---- work decode: sequence, then its items (rb, h') of KV head g with index rb*G + h',
    // heaviest (largest rb) first; the two slots of a CTA are consecutive items of one sequence
    const int g = blockIdx.y;
    int sq = 0, base = 0, nRB = 0;
    for (;; ++sq) {
        nRB = p.seq.ckt[sq + 1] - p.seq.ckt[sq];
        const int ncta = (nRB * p.G + 1) >> 1;
        if (int(blockIdx.x) < base + ncta || sq + 1 >= p.seq.n) break;
        base += ncta;
    }
    const int tok0 = p.seq.cu[sq], Ls = p.seq.cu[sq + 1] - tok0;
    const int nItems = nRB * p.G;
    const int idx0 = nItems - 1 - 2 * (int(blockIdx.x) - base);
    const int idx1 = idx0 - 1;                       // < 0: slot 1 idle
    const int rb0 = idx0 / p.G, h0 = g * p.G + idx0 % p.G;
    const int rb1 = idx1 >= 0 ? idx1 / p.G : -1, h1 = idx1 >= 0 ? g * p.G + idx1 % p.G : 0;
    const int nP = (p.Lp + 127) >> 7;
    const int n_iter0 = nP + rb0 + 1;                // slot 0 is the longer one
    const int n_iter1 = idx1 >= 0 ? nP + rb1 + 1 : 0;

    if (tid == 0) {
        mbar_init(&bar_Q[0], 1); mbar_init(&bar_Q[1], 1);
        for (int s = 0; s < C::KS; ++s) {
            mbar_init(&bar_Kf[s], 1); mbar_init(&bar_Ke[s], 1);
            mbar_init(&bar_Vf[s], 1); mbar_init(&bar_Ve[s], 1);
        }
        mbar_init(&bar_S[0], 1); mbar_init(&bar_S[1], 1);
        for (int i = 0; i < 4; ++i) mbar_init(&bar_P[i], 128);
        mbar_init(bar_done, 1);
        fence_mbar_init();
    }
    if (warp == 16) {
        tmem_alloc(tmem_slot, 512);
        if (elect_one()) {
            tma_prefetch_desc(&tmQ); tma_prefetch_desc(&tmK1); tma_prefetch_desc(&tmV1);
            tma_prefetch_desc(&tmK2); tma_prefetch_desc(&tmV2);
        }
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp == 16) {
        // =============================== TMA producer ===============================
        if (elect_one()) {
            mbar_arrive_expect_tx(&bar_Q[0], C::TILE);
            for (int k = 0; k < C::NSUB; ++k)
                tma_load_3d(smem + C::OFF_Q + k * C::SUB, &tmQ, &bar_Q[0], 64 * k, h0, tok0 + rb0 * 128);
            if (idx1 >= 0) {
                mbar_arrive_expect_tx(&bar_Q[1], C::TILE);
                for (int k = 0; k < C::NSUB; ++k)
                    tma_load_3d(smem + C::OFF_Q + C::TILE + k * C::SUB, &tmQ, &bar_Q[1], 64 * k, h1,
                                tok0 + rb1 * 128);
            }
            for (int it = 0; it < n_iter0; ++it) {
                const int st = it % C::KS;
                const uint32_t ph = (it / C::KS) & 1;
                const bool pre = it < nP;
                const int row0 = pre ? it * 128 : tok0 + (it - nP) * 128;
                mbar_wait(&bar_Ke[st], ph ^ 1);
                mbar_arrive_expect_tx(&bar_Kf[st], C::TILE);
                for (int k = 0; k < C::NSUB; ++k)
                    tma_load_3d(smem + C::OFF_K + st * C::TILE + k * C::SUB, pre ? &tmK1 : &tmK2,
                                &bar_Kf[st], 64 * k, g, row0);
                mbar_wait(&bar_Ve[st], ph ^ 1);
                mbar_arrive_expect_tx(&bar_Vf[st], C::TILE);
                for (int k = 0; k < C::NSUB; ++k)
                    tma_load_3d(smem + C::OFF_V + st * C::TILE + k * C::SUB, pre ? &tmV1 : &tmV2,
                                &bar_Vf[st], 64 * k, g, row0);
            }
        }
    } else if (warp == 17) {
        // =============================== MMA issuer ===============================
        if (elect_one()) {
            constexpr uint32_t idesc_qk = make_idesc_bf16(128, 128, false, false);
            constexpr uint32_t idesc_pv = make_idesc_bf16(128, D, false, true);
            const uint32_t sQ = smem_u32(smem + C::OFF_Q), sK = smem_u32(smem + C::OFF_K),
                           sV = smem_u32(smem + C::OFF_V);
            auto issue_S = [&](int s, int st) {  // S_s = Q_s . K^T
                const uint64_t q = make_smem_desc_sw128(sQ + s * C::TILE, 16, 1024);
                const uint64_t k = make_smem_desc_sw128(sK + st * C::TILE, 16, 1024);
#pragma unroll
                for (int kk = 0; kk < D / 16; ++kk) {
                    const uint32_t off = ((kk >> 2) * C::SUB + (kk & 3) * 32) >> 4;
                    mma_ss(tmem + s * 128, q + off, k + off, idesc_qk, kk > 0);
                }
            };
            auto issue_PV = [&](int s, int st, int half, bool acc) {  // O_s += P_s[:, half] . V[half]
                const uint64_t v = make_smem_desc_sw128(sV + st * C::TILE, C::SUB, 1024);
#pragma unroll
                for (int kk = half * 4; kk < half * 4 + 4; ++kk)
                    mma_ts(tmem + 256 + s * D, tmem + s * 128 + half * 64 + (kk & 3) * 8, v + ((kk * 2048) >> 4), idesc_pv,
                           (acc || kk > 0) ? 1u : 0u);
            };
            mbar_wait(&bar_Q[0], 0);
            mbar_wait(&bar_Kf[0], 0);
            tc_fence_after();
            issue_S(0, 0);
            mma_commit(&bar_S[0]);
            if (n_iter1 > 0) {
                mbar_wait(&bar_Q[1], 0);
                tc_fence_after();
                issue_S(1, 0);
                mma_commit(&bar_S[1]);
            }
            mma_commit(&bar_Ke[0]);
            for (int it = 0; it < n_iter0; ++it) {
                const int st = it % C::KS;
                const uint32_t ph = (it / C::KS) & 1;
                const bool next = it + 1 < n_iter0;
                const int st1 = (it + 1) % C::KS;
                const uint32_t ph1 = ((it + 1) / C::KS) & 1;
                mbar_wait(&bar_Vf[st], ph);
                mbar_wait(&bar_P[0], it & 1);
                tc_fence_after();
                issue_PV(0, st, 0, it > 0);
                mbar_wait(&bar_P[1], it & 1);
                tc_fence_after();
                issue_PV(0, st, 1, true);
                if (next) {
                    mbar_wait(&bar_Kf[st1], ph1);
                    tc_fence_after();
                    issue_S(0, st1);
                    mma_commit(&bar_S[0]);
                }
                if (it < n_iter1) {
                    mbar_wait(&bar_P[2], it & 1);
                    tc_fence_after();
                    issue_PV(1, st, 0, it > 0);
                    mbar_wait(&bar_P[3], it & 1);
                    tc_fence_after();
                    issue_PV(1, st, 1, true);
                }
                mma_commit(&bar_Ve[st]);
                if (next) {
                    if (it + 1 < n_iter1) {
                        issue_S(1, st1);
                        mma_commit(&bar_S[1]);
                    }
                    mma_commit(&bar_Ke[st1]);
                }
            }
            mma_commit(bar_done);
        }
    } else {
        // =============================== softmax warpgroups ===============================
        const int s = warp >> 3;                 // slot
        const int hh = (warp >> 2) & 1;          // key-column half of the S tile
        const int r = tid & 127;                 // row in tile == TMEM lane
        const int n_iter = s == 0 ? n_iter0 : n_iter1;
        const int rb = s == 0 ? rb0 : rb1;
        const int h = s == 0 ? h0 : h1;
        const int t = rb * 128 + r;              // query row within its sequence
        const uint32_t lane_off = uint32_t((warp & 3) * 32) << 16;
        const uint32_t tS = tmem + s * 128 + hh * 64 + lane_off;       // this half of S; P at its start
        const uint32_t tO = tmem + 256 + s * D + hh * (D / 2) + lane_off;  // this half of the O columns
        float* xch = reinterpret_cast<float*>(smem + C::OFF_X) + s * 256;  // [parity][slot][half][128]
        const float c = p.scale_log2;
        float m_used = -INFINITY, l = 0.f;
        for (int it = 0; it < n_iter; ++it) {
            mbar_wait(&bar_S[s], it & 1);
            tc_fence_after();
            // visible keys of this tile for this row, relative to this half's first column
            const int limit = (it < nP ? p.Lp - it * 128 : t - (it - nP) * 128 + 1) - hh * 64;
            const bool masked = limit < 64;      // ragged prefix tail or causal diagonal
            // ---- pass 1: row maximum (S is read from TMEM twice to keep the live registers low)
            float mx0 = -INFINITY, mx1 = -INFINITY;
            {
                uint32_t x[2][32];
                tmem_ld32(tS + 0, x[0]);
                tmem_ld32(tS + 32, x[1]);
                tmem_wait_ld();
                if (masked) {
#pragma unroll
                    for (int q = 0; q < 2; ++q)
#pragma unroll
                        for (int j = 0; j < 32; ++j)
                            if (q * 32 + j >= limit) x[q][j] = 0xf149f2cau;  // -1e30: exp2 -> 0, stays finite
                }
#pragma unroll
                for (int q = 0; q < 2; ++q)
#pragma unroll
                    for (int j = 0; j < 32; j += 2) {
                        mx0 = fmaxf(mx0, __uint_as_float(x[q][j]));
                        mx1 = fmaxf(mx1, __uint_as_float(x[q][j + 1]));
                    }
            }
            float* xm = xch + (it & 1) * 512;
            const float mine = fmaxf(mx0, mx1);
            xm[hh * 128 + r] = mine;
            named_bar_sync(1 + s, 256);          // the two warpgroups of the slot
            const float m_new = fmaxf(mine, xm[(hh ^ 1) * 128 + r]) * c;
            // lazy rescale: keep a stale max while the new one is within 2^8 of it
            const bool need = (it == 0) || (m_new > m_used + 8.f);
            if (__any_sync(0xffffffffu, need && it > 0)) {
                const float alpha = need ? fast_exp2(m_used - m_new) : 1.f;
                l *= alpha;
#pragma unroll
                for (int q = 0; q < D / 64; ++q) {
                    uint32_t o[32];
                    tmem_ld32(tO + q * 32, o);
                    tmem_wait_ld();
#pragma unroll
                    for (int j = 0; j < 32; ++j) o[j] = __float_as_uint(__uint_as_float(o[j]) * alpha);
                    tmem_st32(tO + q * 32, o);
                }
            }
            if (need) m_used = m_new;
            // ---- pass 2: P = exp2(c S - m), packed to bf16 over the first 32 columns of this half
            // of S.  Chunk q (columns [32q, 32q+32)) writes P columns [16q, 16q+16): behind the reads.
            const float2 c2 = make_float2(c, c), nm2 = make_float2(-m_used, -m_used);
            float2 sum2 = make_float2(0.f, 0.f);
            uint32_t xb[2][32];                  // chunk 1 is in flight while chunk 0 is exponentiated
            tmem_ld32(tS, xb[0]);
            tmem_wait_ld();
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                uint32_t (&x)[32] = xb[q];
                if (q == 0) tmem_ld32(tS + 32, xb[1]);
                if (masked) {
#pragma unroll
                    for (int j = 0; j < 32; ++j)
                        if (q * 32 + j >= limit) x[j] = 0xf149f2cau;
                }
                uint32_t pk[16];
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const float2 a = __ffma2_rn(make_float2(__uint_as_float(x[2 * j]),
                                                            __uint_as_float(x[2 * j + 1])), c2, nm2);
                    float2 e;
                    if ((j * PF_FWD_POLY16) % 16 < PF_FWD_POLY16) {   // PF_FWD_POLY16 pairs in 16 on the FMA pipe
                        e = exp2_poly2(a);
                    } else {
                        e.x = fast_exp2(a.x);
                        e.y = fast_exp2(a.y);
                    }
                    sum2 = __fadd2_rn(sum2, e);
                    pk[j] = pack_bf16(e.x, e.y);
                }
                tmem_wait_ld();
                tmem_st16(tS + q * 16, pk);
            }
            tmem_wait_st();
            tc_fence_before();
            mbar_arrive(&bar_P[2 * s + hh]);     // this half (64 keys) of P is ready for the MMA warp
            l += sum2.x + sum2.y;
        }
        if (n_iter > 0) {
            // combine the two halves' row sums, then each half normalises its half of the O columns
            float* xl = xch + (n_iter & 1) * 512;
            xl[hh * 128 + r] = l;
            named_bar_sync(1 + s, 256);
            l += xl[(hh ^ 1) * 128 + r];
            mbar_wait(bar_done, 0);
            tc_fence_after();
            const float inv = 1.f / l;
            const bool valid = t < Ls;
            __nv_bfloat16* orow = p.O + int64_t(tok0 + t) * p.o_stride_tok + int64_t(h) * p.o_stride_head +
                                  hh * (D / 2);
#pragma unroll
            for (int q = 0; q < D / 64; ++q) {
                uint32_t o[32];
                tmem_ld32(tO + q * 32, o);
                tmem_wait_ld();
                if (valid) {
#pragma unroll
                    for (int j = 0; j < 32; j += 8) {
                        uint4 v;
                        v.x = pack_bf16(__uint_as_float(o[j + 0]) * inv, __uint_as_float(o[j + 1]) * inv);
                        v.y = pack_bf16(__uint_as_float(o[j + 2]) * inv, __uint_as_float(o[j + 3]) * inv);
                        v.z = pack_bf16(__uint_as_float(o[j + 4]) * inv, __uint_as_float(o[j + 5]) * inv);
                        v.w = pack_bf16(__uint_as_float(o[j + 6]) * inv, __uint_as_float(o[j + 7]) * inv);
                        *reinterpret_cast<uint4*>(orow + q * 32 + j) = v;
                    }
                }
            }
            if (valid && hh == 0)
                p.LSE[int64_t(h) * p.lse_stride + tok0 + t] = (m_used + log2f(l)) * 0.6931471805599453f;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 16) tmem_dealloc(tmem, 512);
}

}  // namespace pf
