// attn_fwd.cuh -- sm_100a attention forward with two KV sources, packed sequences.
//
//   O[t,h] = softmax_j( sigma <q[h,t], k[g,j]> ) v[g,j],   LSE[h,t] = log sum_j exp(sigma <q,k>)
//
// KV source 1 ("prefix", length Lp): every key is visible to every query (cached K1/V1, read in
// place -- no concat copy).  KV source 2 ("causal"): the keys of the query's own sequence, key j
// visible to query t iff j <= t.  Phase A / replay: Lp = 0, one sequence.  Phase B: source 1 = the
// cached prefix, the sequences are the suffixes of the wave packed along the token axis.
//
// One CTA = 256 consecutive query rows of one head = TWO query tiles of 128 rows that share one
// K/V stream of 64-key sub-tiles:
//   warps 0-3   softmax of tile 0: thread r <-> query row r <-> TMEM lane r, ALL 64 keys of a sub-tile
//   warps 4-7   softmax of tile 1
//   warp  8     TMA producer (K/V sub-tiles through a KS-stage ring, prefix source then causal source)
//   warp  9     tcgen05.mma issuer (one thread)
// TMEM (512 columns): S0 | S1 (64 each) | Q0 | Q1 (D/2 each) | O0 | O1 (D each, at 256).
// Q (bf16) is written to TMEM once by the softmax threads and is the A operand of S = Q K^T, so the
// tensor core reads only K and V from shared memory (TS MMAs); P (bf16) overwrites the first 32
// columns of its S and is the TMEM A operand of O += P V.
//
// Why two tiles: a tile's chain  S -> softmax -> P -> O += P V -> next S  is serial (P aliases S), so
// the tensor pipe runs the other tile's MMAs while this tile's softmax computes:
//     tensor pipe : S0 S1 | PV0 S0' | PV1 S1' | PV0' S0'' | ...
//     softmax 0   :   [softmax S0 ]   [softmax S0' ] ...
//     softmax 1   :          [softmax S1 ]   [softmax S1' ] ...
// Why a row per thread: the running maximum, the row sum and the rescale decision are private to one
// thread -- no shared-memory exchange, no block barrier inside the KV loop.  O is rescaled lazily
// (only when the sub-tile's maximum exceeds the reference by more than 2^8), by the row's own thread,
// after the tile's previous P.V has landed and before its next one can be issued.
#pragma once
#include <cuda.h>
#include "sm100_ptx.cuh"
#include "seq_table.cuh"

namespace pf {

// Debug counter: (query row, KV sub-tile) events in which the running-max reference was re-based
// after the row's first sub-tile (the lazy-rescale path below).  Read through
// pf_counter("fwd_rescale_rows"); the tests use it to prove that the adversarial-logit inputs
// really drive that path.
__device__ unsigned long long g_fwd_rescale_rows;

struct FwdParams {
    const __nv_bfloat16* Q;
    int64_t q_stride_tok, q_stride_head;  // elements
    __nv_bfloat16* O;
    int64_t o_stride_tok, o_stride_head;  // elements
    float* LSE;                           // [Hq, lse_stride], column = packed token row
    int64_t lse_stride;
    PrefixRanges pre;  // visible ranges of the prefix source (n = 0: none)
    int Hq, Hkv, G;
    float scale_log2;  // sigma * log2(e)
    SeqTable seq;
};

template <int D>
struct FwdCfg {
    static constexpr int KS = 6;                       // K/V ring depth (64-key sub-tiles)
    static constexpr int SUB = 64 * 64 * 2;            // one [64 keys][64 elements] swizzle-128B box
    static constexpr int NSUB = D / 64;
    static constexpr int TILE = NSUB * SUB;            // one 64 x D bf16 sub-tile (K or V)
    static constexpr int STAGE = 2 * TILE;             // K then V
    static constexpr int OFF_BAR = KS * STAGE;
    static constexpr int SMEM = OFF_BAR + 512;
    static constexpr int THREADS = 320;
    static constexpr int POLY16 = 5;                   // of 16 exp2 pairs, done by the polynomial on the FMA pipe
    static constexpr uint32_t T_S = 0, T_Q = 128, T_O = 256;   // S_t at 64 t, Q_t at 128 + t D/2, O_t at 256 + t D
    static_assert(SMEM <= 232448, "shared memory budget");
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

__device__ __forceinline__ float fmax3(float a, float b, float c) {
    float r;
    asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
    return r;
}

template <int D>
__global__ void __launch_bounds__(320, 1)
attn_fwd_kernel(const __grid_constant__ CUtensorMap tmK1, const __grid_constant__ CUtensorMap tmV1,
                const __grid_constant__ CUtensorMap tmK2, const __grid_constant__ CUtensorMap tmV2,
                const __grid_constant__ FwdParams p) {
    using C = FwdCfg<D>;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
    uint64_t* bar_Kf = bars;                // [KS] K sub-tile landed
    uint64_t* bar_Ke = bars + C::KS;        // [KS] K sub-tile consumed by the S MMAs of both tiles
    uint64_t* bar_Vf = bars + 2 * C::KS;
    uint64_t* bar_Ve = bars + 3 * C::KS;
    uint64_t* bar_Q = bars + 4 * C::KS;     // [2] Q_t written to TMEM by its softmax threads
    uint64_t* bar_S = bar_Q + 2;            // [2] S_t ready (MMA -> softmax)
    uint64_t* bar_P = bar_S + 2;            // [2] P_t written (softmax -> MMA)
    uint64_t* bar_PV = bar_P + 2;           // [2] P.V of tile t complete (before O is rescaled / read out)
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bar_PV + 2);

    const int tid = threadIdx.x, warp = tid >> 5;
    if ((smem_u32(smem) & 1023u) != 0) __trap();

    // ---- work decode: items = (row-block pair, sequence, head of the KV head's group), deepest pair
    // (longest causal part) first over the whole grid so that the launch tail is made of short items
    const int g = blockIdx.y;
    int sq = 0, pr = 0, hh = 0;
    {
        int x = blockIdx.x, maxp = 0;
        for (int s = 0; s < p.seq.n; ++s) maxp = max(maxp, (p.seq.ckt[s + 1] - p.seq.ckt[s] + 1) >> 1);
        for (pr = maxp - 1; pr > 0; --pr) {
            int cnt = 0;
            for (int s = 0; s < p.seq.n; ++s) cnt += ((p.seq.ckt[s + 1] - p.seq.ckt[s] + 1) >> 1) > pr;
            if (x < cnt * p.G) break;
            x -= cnt * p.G;
        }
        int k = x / p.G;
        hh = x % p.G;
        for (sq = 0; sq < p.seq.n; ++sq)
            if (((p.seq.ckt[sq + 1] - p.seq.ckt[sq] + 1) >> 1) > pr && k-- == 0) break;
    }
    const int h = g * p.G + hh;
    const int tok0 = p.seq.cu[sq], Ls = p.seq.cu[sq + 1] - tok0;
    const int R0 = pr * 256;                                   // first query row of tile 0 in its sequence
    const bool act1 = R0 + 128 < Ls;                           // tile 1 has rows
    const int nP = p.pre.n > 0 ? p.pre.sub0[p.pre.n] : 0;      // prefix sub-tiles
    const int n0 = nP + (min(R0 + 128, Ls) + 63) / 64;         // sub-tiles of tile 0
    const int n1 = act1 ? nP + (min(R0 + 256, Ls) + 63) / 64 : 0;
    const int n_iter = act1 ? n1 : n0;                         // n0 <= n1 when tile 1 is active

    if (tid == 0) {
        for (int s = 0; s < C::KS; ++s) {
            mbar_init(&bar_Kf[s], 1); mbar_init(&bar_Ke[s], 1);
            mbar_init(&bar_Vf[s], 1); mbar_init(&bar_Ve[s], 1);
        }
        for (int t = 0; t < 2; ++t) {
            mbar_init(&bar_Q[t], 128); mbar_init(&bar_S[t], 1);
            mbar_init(&bar_P[t], 128); mbar_init(&bar_PV[t], 1);
        }
        fence_mbar_init();
    }
    if (warp == 8) {
        tmem_alloc(tmem_slot, 512);
        if (elect_one()) {
            tma_prefetch_desc(&tmK1); tma_prefetch_desc(&tmV1);
            tma_prefetch_desc(&tmK2); tma_prefetch_desc(&tmV2);
        }
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp == 8) {
        // =============================== TMA producer ===============================
        if (elect_one()) {
            for (int it = 0; it < n_iter; ++it) {
                const int st = it % C::KS;
                const uint32_t ph = (it / C::KS) & 1;
                const bool pre = it < nP;
                int row0 = tok0 + (it - nP) * 64, valid_rows;
                if (pre) p.pre.locate64(it, row0, valid_rows);
                uint8_t* stage = smem + st * C::STAGE;
                mbar_wait(&bar_Ke[st], ph ^ 1);
                mbar_arrive_expect_tx(&bar_Kf[st], C::TILE);
                for (int k = 0; k < C::NSUB; ++k)
                    tma_load_3d(stage + k * C::SUB, pre ? &tmK1 : &tmK2, &bar_Kf[st], 64 * k, g, row0);
                mbar_wait(&bar_Ve[st], ph ^ 1);
                mbar_arrive_expect_tx(&bar_Vf[st], C::TILE);
                for (int k = 0; k < C::NSUB; ++k)
                    tma_load_3d(stage + C::TILE + k * C::SUB, pre ? &tmV1 : &tmV2, &bar_Vf[st], 64 * k, g, row0);
            }
        }
    } else if (warp == 9) {
        // =============================== MMA issuer ===============================
        if (elect_one()) {
            constexpr uint32_t idesc_qk = make_idesc_bf16(128, 64, false, false);
            constexpr uint32_t idesc_pv = make_idesc_bf16(128, D, false, true);
            const uint32_t s0 = smem_u32(smem);
            const int nt[2] = {n0, n1};
            auto issue_S = [&](int t, int st) {  // S_t = Q_t . K^T   (A = Q_t from TMEM)
                const uint64_t k = make_smem_desc_sw128(s0 + st * C::STAGE, 16, 1024);
#pragma unroll
                for (int kk = 0; kk < D / 16; ++kk)
                    mma_ts(tmem + C::T_S + t * 64, tmem + C::T_Q + t * (D / 2) + kk * 8,
                           k + (((kk >> 2) * C::SUB + (kk & 3) * 32) >> 4), idesc_qk, kk > 0);
            };
            auto issue_PV = [&](int t, int st, bool acc) {  // O_t += P_t . V   (A = P_t from TMEM)
                const uint64_t v = make_smem_desc_sw128(s0 + st * C::STAGE + C::TILE, C::SUB, 1024);
#pragma unroll
                for (int kk = 0; kk < 4; ++kk)
                    mma_ts(tmem + C::T_O + t * D, tmem + C::T_S + t * 64 + kk * 8,
                           v + ((kk * 2048) >> 4), idesc_pv, (acc || kk > 0) ? 1u : 0u);
            };
            mbar_wait(&bar_Q[0], 0);
            if (act1) mbar_wait(&bar_Q[1], 0);
            mbar_wait(&bar_Kf[0], 0);
            tc_fence_after();
            issue_S(0, 0);
            mma_commit(&bar_S[0]);
            if (act1) {
                issue_S(1, 0);
                mma_commit(&bar_S[1]);
            }
            mma_commit(&bar_Ke[0]);
            for (int it = 0; it < n_iter; ++it) {
                const int st = it % C::KS, nx = it + 1, stn = nx % C::KS;
                mbar_wait(&bar_Vf[st], (it / C::KS) & 1);
                bool k_ready = false;
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    if (it >= nt[t]) continue;
                    mbar_wait(&bar_P[t], it & 1);
                    tc_fence_after();
                    issue_PV(t, st, it > 0);
                    mma_commit(&bar_PV[t]);
                    if (nx < nt[t]) {            // this tile's next S runs while the other tile's softmax works
                        if (!k_ready) {
                            mbar_wait(&bar_Kf[stn], (nx / C::KS) & 1);
                            tc_fence_after();
                            k_ready = true;
                        }
                        issue_S(t, stn);
                        mma_commit(&bar_S[t]);
                    }
                }
                if (k_ready) mma_commit(&bar_Ke[stn]);
                mma_commit(&bar_Ve[st]);
            }
        }
    } else {
        // =============================== softmax warpgroups ===============================
        const int t = warp >> 2;                 // query tile of this warpgroup
        const int r = tid & 127;                 // row in tile == TMEM lane
        const int tq = R0 + t * 128 + r;         // query row within its sequence
        const bool valid = tq < Ls;
        const int n_t = t == 0 ? n0 : n1;
        const uint32_t lane_off = uint32_t((warp & 3) * 32) << 16;
        const uint32_t tS = tmem + C::T_S + t * 64 + lane_off;           // S_t; P_t over its first 32 columns
        const uint32_t tO = tmem + C::T_O + t * D + lane_off;
        const float c = p.scale_log2;
        if (n_t > 0) {
            // ---- Q row -> TMEM (A operand layout: lane = row, column j = elements 2j, 2j+1)
            {
                const uint4* qrow = reinterpret_cast<const uint4*>(
                    p.Q + int64_t(tok0 + tq) * p.q_stride_tok + int64_t(h) * p.q_stride_head);
#pragma unroll
                for (int cnk = 0; cnk < D / 64; ++cnk) {
                    uint32_t qv[32];
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        const uint4 v = valid ? qrow[cnk * 8 + j] : make_uint4(0u, 0u, 0u, 0u);
                        qv[4 * j] = v.x; qv[4 * j + 1] = v.y; qv[4 * j + 2] = v.z; qv[4 * j + 3] = v.w;
                    }
                    tmem_st32(tmem + C::T_Q + t * (D / 2) + cnk * 32 + lane_off, qv);
                }
                tmem_wait_st();
                tc_fence_before();
                mbar_arrive(&bar_Q[t]);
            }
            float m_used = -INFINITY, l = 0.f;
            for (int it = 0; it < n_t; ++it) {
                mbar_wait(&bar_S[t], it & 1);
                tc_fence_after();
                uint32_t x[64];
                tmem_ld32(tS, *reinterpret_cast<uint32_t(*)[32]>(&x[0]));
                tmem_ld32(tS + 32, *reinterpret_cast<uint32_t(*)[32]>(&x[32]));
                tmem_wait_ld();
                // visible keys of this sub-tile for this row
                int limit = tq - (it - nP) * 64 + 1;
                if (it < nP) {
                    int row0;
                    p.pre.locate64(it, row0, limit);
                }
                if (limit < 64) {                    // ragged prefix tail or causal diagonal
#pragma unroll
                    for (int j = 0; j < 64; ++j)
                        if (j >= limit) x[j] = 0xf149f2cau;  // -1e30: exp2 -> 0, stays finite
                }
                float mx[4];
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    mx[q] = fmax3(__uint_as_float(x[q]), __uint_as_float(x[4 + q]), __uint_as_float(x[8 + q]));
#pragma unroll
                for (int j = 12; j < 60; j += 8)
#pragma unroll
                    for (int q = 0; q < 4; ++q)
                        mx[q] = fmax3(mx[q], __uint_as_float(x[j + q]), __uint_as_float(x[j + 4 + q]));
#pragma unroll
                for (int q = 0; q < 4; ++q) mx[q] = fmaxf(mx[q], __uint_as_float(x[60 + q]));
                const float m_new = fmaxf(fmaxf(mx[0], mx[1]), fmaxf(mx[2], mx[3])) * c;
                // lazy rescale: keep a stale reference while the new maximum is within 2^8 of it
                const bool need = (it == 0) || (m_new > m_used + 8.f);
                const unsigned rescale_mask = __ballot_sync(0xffffffffu, need && it > 0);
                if (rescale_mask != 0u) {
                    if ((tid & 31) == 0)
                        atomicAdd(&g_fwd_rescale_rows, (unsigned long long)__popc(rescale_mask));
                    mbar_wait(&bar_PV[t], (it - 1) & 1);   // P.V(it-1) of this tile has landed in O_t
                    tc_fence_after();
                    const float alpha = need ? fast_exp2(m_used - m_new) : 1.f;
                    l *= alpha;
#pragma unroll 1
                    for (int cnk = 0; cnk < D / 32; ++cnk) {
                        uint32_t o[32];
                        tmem_ld32(tO + cnk * 32, o);
                        tmem_wait_ld();
#pragma unroll
                        for (int j = 0; j < 32; ++j) o[j] = __float_as_uint(__uint_as_float(o[j]) * alpha);
                        tmem_st32(tO + cnk * 32, o);
                    }
                }
                if (need) m_used = m_new;
                // ---- P = exp2(c S - m), packed to bf16 over the first 32 columns of S_t
                const float2 c2 = make_float2(c, c), nm2 = make_float2(-m_used, -m_used);
                float2 sum2 = make_float2(0.f, 0.f);
                uint32_t pk[32];
#pragma unroll
                for (int j = 0; j < 32; ++j) {
                    const float2 a = __ffma2_rn(make_float2(__uint_as_float(x[2 * j]),
                                                            __uint_as_float(x[2 * j + 1])), c2, nm2);
                    float2 e;
                    if ((j * C::POLY16) % 16 < C::POLY16) {   // POLY16 pairs in 16 on the FMA pipe
                        e = exp2_poly2(a);
                    } else {
                        e.x = fast_exp2(a.x);
                        e.y = fast_exp2(a.y);
                    }
                    sum2 = __fadd2_rn(sum2, e);
                    pk[j] = pack_bf16(e.x, e.y);
                }
                tmem_st32(tS, pk);
                tmem_wait_st();
                tc_fence_before();
                mbar_arrive(&bar_P[t]);
                l += sum2.x + sum2.y;
            }
            // ---- epilogue: O_t / l -> bf16 rows, LSE
            mbar_wait(&bar_PV[t], (n_t - 1) & 1);
            tc_fence_after();
            const float inv = 1.f / l;
            __nv_bfloat16* orow = p.O + int64_t(tok0 + tq) * p.o_stride_tok + int64_t(h) * p.o_stride_head;
#pragma unroll 1
            for (int cnk = 0; cnk < D / 32; ++cnk) {
                uint32_t o[32];
                tmem_ld32(tO + cnk * 32, o);
                tmem_wait_ld();
                if (valid) {
#pragma unroll
                    for (int j = 0; j < 32; j += 8) {
                        uint4 v;
                        v.x = pack_bf16(__uint_as_float(o[j + 0]) * inv, __uint_as_float(o[j + 1]) * inv);
                        v.y = pack_bf16(__uint_as_float(o[j + 2]) * inv, __uint_as_float(o[j + 3]) * inv);
                        v.z = pack_bf16(__uint_as_float(o[j + 4]) * inv, __uint_as_float(o[j + 5]) * inv);
                        v.w = pack_bf16(__uint_as_float(o[j + 6]) * inv, __uint_as_float(o[j + 7]) * inv);
                        *reinterpret_cast<uint4*>(orow + cnk * 32 + j) = v;
                    }
                }
            }
            if (valid)
                p.LSE[int64_t(h) * p.lse_stride + tok0 + tq] = (m_used + log2f(l)) * 0.6931471805599453f;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 8) tmem_dealloc(tmem, 512);
}

}  // namespace pf
