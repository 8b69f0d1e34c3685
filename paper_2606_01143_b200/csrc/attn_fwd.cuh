// attn_fwd.cuh -- sm_100a attention forward with two KV sources, packed sequences.
//
//   O[t,h] = softmax_j( sigma <q[h,t], k[g,j]> ) v[g,j],   LSE[h,t] = log sum_j exp(sigma <q,k>)
//
// KV source 1 ("prefix", length Lp): every key is visible to every query (cached K1/V1, read in
// place -- no concat copy).  KV source 2 ("causal"): the keys of the query's own sequence, key j
// visible to query t iff j <= t.  Phase A / replay: Lp = 0, one sequence.  Phase B: source 1 = the
// cached prefix, the sequences are the suffixes of the wave packed along the token axis.
//
// One CTA = one query tile of 128 rows of one head.  Its keys are walked in 64-key sub-tiles by TWO
// independent chains: chain x in {0,1} owns the sub-tiles x, x+2, x+4, ... and keeps its own scores
// S_x, probabilities P_x, output accumulator O_x, running maximum and row sum (a split of the KV
// axis inside the CTA); the two partial softmaxes are merged once at the end,
//     O = (w0 O0 + w1 O1) / (w0 l0 + w1 l1),  w_x = 2^(m_x - max(m0, m1)).
//   warps 0-3   softmax of chain 0: thread r <-> query row r <-> TMEM lane r, ALL 64 keys of a sub-tile
//   warps 4-7   softmax of chain 1
//   warp  8     TMA producer (K/V sub-tiles through a KS-stage ring, prefix source then causal source)
//   warps 9,10  tcgen05.mma issuers, one thread per chain
// TMEM (512 columns): S0 | S1 (64 each) | P0 | P1 (32 each) | Q (D/2) | O0 | O1 (D each, at 256).
// Q (bf16) is written to TMEM once by the softmax threads and is the A operand of S = Q K^T, P (bf16)
// is the TMEM A operand of O += P V: the tensor core reads only K and V from shared memory (TS MMAs).
//
// Why two chains: within a chain, S(k+1) is issued the moment the softmax warpgroup holds S(k) in
// registers (P has its own columns), so a warpgroup never waits for the tensor pipe in steady state,
// and the two warpgroups -- two warps per scheduler -- overlap each other's MUFU, FMA and ALU work.
// Why a row per thread: the running maximum, the row sum and the rescale decision are private to one
// thread -- no shared-memory exchange, no block barrier inside the KV loop.  O_x is rescaled lazily
// (only when a sub-tile's maximum exceeds the reference by more than 2^8), by the row's own thread,
// after the chain's previous P.V has landed and before its next one can be issued.
#pragma once
#include <cuda.h>
#include "sm100_ptx.cuh"
#include "seq_table.cuh"

namespace pf {

// Debug counter: (query row, KV sub-tile) events in which the running-max reference was re-based
// after the row's first sub-tile of a chain (the lazy-rescale path below).  Read through
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
    static constexpr int OFF_X = KS * STAGE;           // merge exchange: m[2][128], l[2][128] fp32
    static constexpr int OFF_BAR = OFF_X + 2048;
    static constexpr int SMEM = OFF_BAR + 512;
    static constexpr int THREADS = 352;
    static constexpr int POLY16 = 5;                   // of 16 exp2 pairs, done by the polynomial on the FMA pipe
    // TMEM columns: S_x at 64 x, P_x at 128 + 32 x, Q at 192, O_x at 256 + x D
    static constexpr uint32_t T_S = 0, T_P = 128, T_Q = 192, T_O = 256;
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
__global__ void __launch_bounds__(352, 1)
attn_fwd_kernel(const __grid_constant__ CUtensorMap tmK1, const __grid_constant__ CUtensorMap tmV1,
                const __grid_constant__ CUtensorMap tmK2, const __grid_constant__ CUtensorMap tmV2,
                const __grid_constant__ FwdParams p) {
    using C = FwdCfg<D>;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
    uint64_t* bar_Kf = bars;                // [KS] K sub-tile landed
    uint64_t* bar_Ke = bars + C::KS;        // [KS] K sub-tile consumed by its chain's S MMAs
    uint64_t* bar_Vf = bars + 2 * C::KS;
    uint64_t* bar_Ve = bars + 3 * C::KS;
    uint64_t* bar_Q = bars + 4 * C::KS;     // Q written to TMEM by the softmax threads (both warpgroups)
    uint64_t* bar_S = bar_Q + 1;            // [2] S_x ready (MMA -> softmax)
    uint64_t* bar_C = bar_S + 2;            // [2] S_x is in registers: its columns may be overwritten
    uint64_t* bar_P = bar_C + 2;            // [2] P_x written (softmax -> MMA)
    uint64_t* bar_PV = bar_P + 2;           // [2] P.V of chain x complete (O_x may be rescaled / read, P_x rewritten)
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bar_PV + 2);

    const int tid = threadIdx.x, warp = tid >> 5;
    if ((smem_u32(smem) & 1023u) != 0) __trap();

    // ---- work decode: items = (128-row block, sequence, head of the KV head's group), deepest row
    // block (longest causal part) first over the whole grid so that the launch tail is made of short items
    const int g = blockIdx.y;
    int sq = 0, rb = 0, hh = 0;
    {
        int x = blockIdx.x, maxb = 0;
        for (int s = 0; s < p.seq.n; ++s) maxb = max(maxb, p.seq.ckt[s + 1] - p.seq.ckt[s]);
        for (rb = maxb - 1; rb > 0; --rb) {
            int cnt = 0;
            for (int s = 0; s < p.seq.n; ++s) cnt += (p.seq.ckt[s + 1] - p.seq.ckt[s]) > rb;
            if (x < cnt * p.G) break;
            x -= cnt * p.G;
        }
        int k = x / p.G;
        hh = x % p.G;
        for (sq = 0; sq < p.seq.n; ++sq)
            if ((p.seq.ckt[sq + 1] - p.seq.ckt[sq]) > rb && k-- == 0) break;
    }
    const int h = g * p.G + hh;
    const int tok0 = p.seq.cu[sq], Ls = p.seq.cu[sq + 1] - tok0;
    const int R0 = rb * 128;                                   // first query row of the tile in its sequence
    const int nP = p.pre.n > 0 ? p.pre.sub0[p.pre.n] : 0;      // prefix sub-tiles
    const int n_sub = nP + (min(R0 + 128, Ls) + 63) / 64;      // sub-tiles of the tile (>= 1)

    if (tid == 0) {
        for (int s = 0; s < C::KS; ++s) {
            mbar_init(&bar_Kf[s], 1); mbar_init(&bar_Ke[s], 1);
            mbar_init(&bar_Vf[s], 1); mbar_init(&bar_Ve[s], 1);
        }
        mbar_init(bar_Q, 256);
        for (int x = 0; x < 2; ++x) {
            mbar_init(&bar_S[x], 1); mbar_init(&bar_C[x], 128);
            mbar_init(&bar_P[x], 128); mbar_init(&bar_PV[x], 1);
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
            for (int it = 0; it < n_sub; ++it) {
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
    } else if (warp >= 9) {
        // =============================== MMA issuers (warp 9: chain 0, warp 10: chain 1) ===============================
        const int x = warp - 9;
        const int n_x = (n_sub - x + 1) / 2;         // sub-tiles x, x+2, ... < n_sub
        if (elect_one() && n_x > 0) {
            constexpr uint32_t idesc_qk = make_idesc_bf16(128, 64, false, false);
            constexpr uint32_t idesc_pv = make_idesc_bf16(128, D, false, true);
            const uint32_t s0 = smem_u32(smem);
            auto issue_S = [&](int j) {  // S_x = Q . K(j)^T   (A = Q from TMEM)
                const int st = j % C::KS;
                mbar_wait(&bar_Kf[st], (j / C::KS) & 1);
                tc_fence_after();
                const uint64_t k = make_smem_desc_sw128(s0 + st * C::STAGE, 16, 1024);
#pragma unroll
                for (int kk = 0; kk < D / 16; ++kk)
                    mma_ts(tmem + C::T_S + x * 64, tmem + C::T_Q + kk * 8,
                           k + (((kk >> 2) * C::SUB + (kk & 3) * 32) >> 4), idesc_qk, kk > 0);
                mma_commit(&bar_S[x]);
                mma_commit(&bar_Ke[st]);
            };
            auto issue_PV = [&](int j, bool acc) {  // O_x += P_x . V(j)   (A = P_x from TMEM)
                const int st = j % C::KS;
                mbar_wait(&bar_Vf[st], (j / C::KS) & 1);
                tc_fence_after();
                const uint64_t v = make_smem_desc_sw128(s0 + st * C::STAGE + C::TILE, C::SUB, 1024);
#pragma unroll
                for (int kk = 0; kk < 4; ++kk)
                    mma_ts(tmem + C::T_O + x * D, tmem + C::T_P + x * 32 + kk * 8,
                           v + ((kk * 2048) >> 4), idesc_pv, (acc || kk > 0) ? 1u : 0u);
                mma_commit(&bar_PV[x]);
                mma_commit(&bar_Ve[st]);
            };
            mbar_wait(bar_Q, 0);
            issue_S(x);
            for (int k = 0; k < n_x; ++k) {
                const int j = x + 2 * k;
                if (k + 1 < n_x) {   // the next scores as soon as the softmax threads hold the current ones
                    mbar_wait(&bar_C[x], k & 1);
                    issue_S(j + 2);
                }
                mbar_wait(&bar_P[x], k & 1);
                issue_PV(j, k > 0);
            }
        }
    } else {
        // =============================== softmax warpgroups ===============================
        const int x = warp >> 2;                 // chain of this warpgroup
        const int r = tid & 127;                 // row in tile == TMEM lane
        const int tq = R0 + r;                   // query row within its sequence
        const bool valid = tq < Ls;
        const int n_x = (n_sub - x + 1) / 2;
        const uint32_t lane_off = uint32_t((warp & 3) * 32) << 16;
        const uint32_t tS = tmem + C::T_S + x * 64 + lane_off;
        const uint32_t tP = tmem + C::T_P + x * 32 + lane_off;
        const uint32_t tO = tmem + C::T_O + x * D + lane_off;
        const float c = p.scale_log2;
        // ---- Q row -> TMEM (A operand layout: lane = row, column j = elements 2j, 2j+1); each
        // warpgroup writes its half of the row
        {
            const uint4* qrow = reinterpret_cast<const uint4*>(
                p.Q + int64_t(tok0 + tq) * p.q_stride_tok + int64_t(h) * p.q_stride_head + x * (D / 2));
            uint32_t qv[D / 4];
#pragma unroll
            for (int j = 0; j < D / 16; ++j) {
                const uint4 v = valid ? qrow[j] : make_uint4(0u, 0u, 0u, 0u);
                qv[4 * j] = v.x; qv[4 * j + 1] = v.y; qv[4 * j + 2] = v.z; qv[4 * j + 3] = v.w;
            }
            if constexpr (D == 128) tmem_st32(tmem + C::T_Q + x * 32 + lane_off, qv);
            else tmem_st16(tmem + C::T_Q + x * 16 + lane_off, qv);
            tmem_wait_st();
            tc_fence_before();
            mbar_arrive(bar_Q);
        }
        float m_used = -INFINITY, l = 0.f;
        for (int k = 0; k < n_x; ++k) {
            const int it = x + 2 * k;            // sub-tile of this step
            mbar_wait(&bar_S[x], k & 1);
            tc_fence_after();
            uint32_t s[64];
            tmem_ld32(tS, *reinterpret_cast<uint32_t(*)[32]>(&s[0]));
            tmem_ld32(tS + 32, *reinterpret_cast<uint32_t(*)[32]>(&s[32]));
            tmem_wait_ld();
            tc_fence_before();
            mbar_arrive(&bar_C[x]);              // S_x may be overwritten by the chain's next scores
            // visible keys of this sub-tile for this row
            int limit = tq - (it - nP) * 64 + 1;
            if (it < nP) {
                int row0;
                p.pre.locate64(it, row0, limit);
            }
            if (limit < 64) {                    // ragged prefix tail or causal diagonal
#pragma unroll
                for (int j = 0; j < 64; ++j)
                    if (j >= limit) s[j] = 0xf149f2cau;  // -1e30: exp2 -> 0, stays finite
            }
            float mx[4];
#pragma unroll
            for (int q = 0; q < 4; ++q)
                mx[q] = fmax3(__uint_as_float(s[q]), __uint_as_float(s[4 + q]), __uint_as_float(s[8 + q]));
#pragma unroll
            for (int j = 12; j < 60; j += 8)
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    mx[q] = fmax3(mx[q], __uint_as_float(s[j + q]), __uint_as_float(s[j + 4 + q]));
#pragma unroll
            for (int q = 0; q < 4; ++q) mx[q] = fmaxf(mx[q], __uint_as_float(s[60 + q]));
            // a sub-tile with no visible key for this row (chain 1 on the first causal block) must not
            // set the reference: its maximum counts as -inf
            const float m_raw = fmaxf(fmaxf(mx[0], mx[1]), fmaxf(mx[2], mx[3]));
            const float m_new = m_raw < -1e29f ? -INFINITY : m_raw * c;
            // lazy rescale: keep a stale reference while the new maximum is within 2^8 of it; the
            // first visible key of the chain sets it (m_used = -inf until then)
            const bool need = m_new > m_used + 8.f;
            const unsigned rescale_mask = __ballot_sync(0xffffffffu, need && k > 0);
            if (rescale_mask != 0u) {
                if ((tid & 31) == 0)
                    atomicAdd(&g_fwd_rescale_rows, (unsigned long long)__popc(rescale_mask));
                mbar_wait(&bar_PV[x], (k - 1) & 1);   // P.V(k-1) of this chain has landed in O_x
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
            // ---- P = exp2(c S - m), packed to bf16 into P_x
            const float ref = m_used == -INFINITY ? 0.f : m_used;   // nothing visible yet: every P is 0
            const float2 c2 = make_float2(c, c), nm2 = make_float2(-ref, -ref);
            float2 sum2[2] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
            if (k > 0) {                         // P.V(k-1) has finished reading P_x (long ago, normally)
                mbar_wait(&bar_PV[x], (k - 1) & 1);
                tc_fence_after();
            }
            // four chunks of 8 key pairs, each stored as soon as it is packed: the stores pin the
            // exponentials of a chunk in front of the next chunk's arithmetic, so that MUFU work stays
            // spread between the FMA-pipe work instead of piling up at the end of the step
#pragma unroll
            for (int ch = 0; ch < 4; ++ch) {
                uint32_t pk[8];
#pragma unroll
                for (int jj = 0; jj < 8; ++jj) {
                    const int j = ch * 8 + jj;
                    const float2 a = __ffma2_rn(make_float2(__uint_as_float(s[2 * j]),
                                                            __uint_as_float(s[2 * j + 1])), c2, nm2);
                    float2 e;
                    if ((j * C::POLY16) % 16 < C::POLY16) {   // POLY16 pairs in 16 on the FMA pipe
                        e = exp2_poly2(a);
                    } else {
                        e.x = fast_exp2(a.x);
                        e.y = fast_exp2(a.y);
                    }
                    sum2[j & 1] = __fadd2_rn(sum2[j & 1], e);
                    pk[jj] = pack_bf16(e.x, e.y);
                }
                tmem_st8(tP + ch * 8, pk);
            }
            tmem_wait_st();
            tc_fence_before();
            mbar_arrive(&bar_P[x]);
            l += (sum2[0].x + sum2[1].x) + (sum2[0].y + sum2[1].y);
        }
        // ---- merge the two chains: exchange (m, l), wait for both chains' last P.V
        float* xm = reinterpret_cast<float*>(smem + C::OFF_X);      // [2][128]
        float* xl = xm + 256;
        xm[x * 128 + r] = m_used;
        xl[x * 128 + r] = l;
        if (n_x > 0) {
            mbar_wait(&bar_PV[x], (n_x - 1) & 1);
            tc_fence_after();
        }
        tc_fence_before();
        named_bar_sync(1, 256);                  // the two softmax warpgroups
        tc_fence_after();
        const float m_o = xm[(x ^ 1) * 128 + r], l_o = xl[(x ^ 1) * 128 + r];
        const float M = fmaxf(m_used, m_o);      // chain 0 always has a visible key: M is finite
        const float w_me = fast_exp2(m_used - M), w_ot = fast_exp2(m_o - M);
        const float L = l * w_me + l_o * w_ot;
        const float inv = 1.f / L;
        const float w0 = (x == 0 ? w_me : w_ot) * inv, w1 = (x == 0 ? w_ot : w_me) * inv;
        const bool two = n_sub > 1;              // chain 1 exists (uniform over the CTA)
        // each warpgroup finishes its half of the d columns of the row
        __nv_bfloat16* orow = p.O + int64_t(tok0 + tq) * p.o_stride_tok + int64_t(h) * p.o_stride_head + x * (D / 2);
        const uint32_t lane_o = tmem + C::T_O + lane_off + x * (D / 2);
#pragma unroll 1
        for (int cnk = 0; cnk < D / 64; ++cnk) {
            uint32_t a[32], b[32];
            tmem_ld32(lane_o + cnk * 32, a);
            if (two) tmem_ld32(lane_o + D + cnk * 32, b);
            tmem_wait_ld();
            if (valid) {
#pragma unroll
                for (int j = 0; j < 32; j += 8) {
                    float f[8];
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        f[e] = __uint_as_float(a[j + e]) * w0;
                        if (two) f[e] = fmaf(__uint_as_float(b[j + e]), w1, f[e]);
                    }
                    uint4 v;
                    v.x = pack_bf16(f[0], f[1]); v.y = pack_bf16(f[2], f[3]);
                    v.z = pack_bf16(f[4], f[5]); v.w = pack_bf16(f[6], f[7]);
                    *reinterpret_cast<uint4*>(orow + cnk * 32 + j) = v;
                }
            }
        }
        if (valid && x == 0)
            p.LSE[int64_t(h) * p.lse_stride + tok0 + tq] = (M + log2f(L)) * 0.6931471805599453f;
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 8) tmem_dealloc(tmem, 512);
}

}  // namespace pf
