// attn_fwd.cuh -- sm_100a attention forward with two KV sources, packed sequences.
//
//   O[t,h] = softmax_j( sigma <q[h,t], k[g,j]> ) v[g,j],   LSE[h,t] = log sum_j exp(sigma <q,k>)
//
// KV source 1 ("prefix", length Lp): every key is visible to every query (cached K1/V1, read in
// place -- no concat copy).  KV source 2 ("causal"): the keys of the query's own sequence, key j
// visible to query t iff j <= t.  Phase A / replay: Lp = 0, one sequence.  Phase B: source 1 = the
// cached prefix, the sequences are the suffixes of the wave packed along the token axis.
//
// One CTA = one query tile of 128 rows of one head:
//   warps 0-15  softmax: warpgroup q (warps 4q..4q+3) owns key columns [32q, 32q+32) of each S tile
//               (thread r of a warpgroup <-> query row r <-> TMEM lane r)
//   warp  16    TMA producer (K/V tiles through a 3-stage ring, prefix source then causal source)
//   warp  17    tcgen05.mma issuer (one thread)
// TMEM: S[0] | S[1] | O | Q  (128 + 128 + D + D/2 columns).  Q (bf16) is written to TMEM once by the
// softmax threads and is the A operand of S = Q K^T, so that per KV tile the tensor core reads only
// K and V from shared memory (an SS MMA would add 32 KB of Q per tile and make the shared-memory
// pipe the bound).  S is double-buffered: S(it+1) is computed while softmax(it) runs, P(it) (bf16)
// overwrites the start of each column quarter of S(it) and is the TMEM A operand of O += P V.  The
// four threads of a row (one per column quarter: warps w, w+4, w+8, w+12, all on one scheduler)
// exchange partial row maxima through shared memory once per KV tile behind a 128-thread named
// barrier of their own -- the four row quarters of the tile never wait for each other; O is rescaled
// lazily (only when the running max grew by more than 2^8).
//
// Measured alternatives (round 2, same GPU, alternating order): two 128-row tiles
// per CTA sharing the K/V stream with a row-per-thread softmax, and one tile walked by two independent
// KV chains with separate P columns (8 or 16 softmax warps), were 7-13 % SLOWER than this kernel: the
// softmax is bound by instruction issue (about 8 instructions per score element and thread), which
// those organisations do not reduce, and they pay more barrier round trips per key.
#pragma once
#include <cuda.h>
#include "sm100_ptx.cuh"
#include "seq_table.cuh"

namespace pf {

// Debug counter: (query row, KV tile) events in which the running-max reference was re-based after
// the row's first tile (the lazy-rescale path below).  Read through pf_counter("fwd_rescale_rows");
// the tests use it to prove that the adversarial-logit inputs really drive that path.
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

template <int B>
struct IntC {
    static constexpr int v = B;
};

template <int D>
struct FwdCfg {
    static constexpr int KS = 3;                       // K/V ring depth
    static constexpr int TILE = 128 * D * 2;           // bytes of one 128 x D bf16 tile
    static constexpr int SUB = 128 * 64 * 2;           // one 128 x 64 swizzle-128B sub-tile
    static constexpr int NSUB = D / 64;
    static constexpr int OFF_K = 0;                    // KS tiles
    static constexpr int OFF_V = KS * TILE;            // KS tiles
    static constexpr int OFF_BAR = 2 * KS * TILE;
    static constexpr int OFF_X = OFF_BAR + 256;        // row-max / row-sum exchange between column halves
    static constexpr int SMEM = OFF_X + 2 * 4 * 128 * 4;
    static constexpr int THREADS = 576;
    static constexpr int POLY16 = 6;                   // of 16 exp2 pairs, done by the polynomial on the FMA pipe
    static constexpr uint32_t T_O = 256, T_Q = 256 + D;  // TMEM columns of O and Q (S[b] at 128 b)
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
attn_fwd_kernel(const __grid_constant__ CUtensorMap tmK1, const __grid_constant__ CUtensorMap tmV1,
                const __grid_constant__ CUtensorMap tmK2, const __grid_constant__ CUtensorMap tmV2,
                const __grid_constant__ FwdParams p) {
    using C = FwdCfg<D>;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
    uint64_t* bar_Q = bars;                 // Q written to TMEM by the softmax threads
    uint64_t* bar_Kf = bars + 1;            // [KS]
    uint64_t* bar_Ke = bars + 4;
    uint64_t* bar_Vf = bars + 7;
    uint64_t* bar_Ve = bars + 10;
    uint64_t* bar_S = bars + 13;            // [2] S[b] ready (MMA -> softmax)
    uint64_t* bar_P = bars + 15;            // [2 buffers][2 halves] P half ready (softmax -> MMA)
    uint64_t* bar_PV = bars + 19;           // P.V of an iteration complete (needed before O is rescaled)
    uint64_t* bar_done = bars + 20;         // all MMAs complete
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 22);

    const int tid = threadIdx.x, warp = tid >> 5;
    if ((smem_u32(smem) & 1023u) != 0) __trap();

    // ---- work decode: sequence, then its items (rb, h') of KV head g, heaviest (largest rb) first
    const int g = blockIdx.y;
    int sq = 0, base = 0, nRB = 0;
    for (;; ++sq) {
        nRB = p.seq.ckt[sq + 1] - p.seq.ckt[sq];
        if (int(blockIdx.x) < base + nRB * p.G || sq + 1 >= p.seq.n) break;
        base += nRB * p.G;
    }
    const int tok0 = p.seq.cu[sq], Ls = p.seq.cu[sq + 1] - tok0;
    const int idx = nRB * p.G - 1 - (int(blockIdx.x) - base);
    const int rb = idx / p.G, h = g * p.G + idx % p.G;
    const int nP = p.pre.n > 0 ? p.pre.tile0[p.pre.n] : 0;
    const int n_iter = nP + rb + 1;

    // The softmax threads put their loads of Q in flight BEFORE the set-up barrier (mbarrier init,
    // TMEM allocation), so that the round trip to L2 / HBM overlaps the set-up instead of following it.
    constexpr int QW = D / 8;                    // 32-bit words of Q per softmax thread (a quarter row)
    uint32_t qv[QW];
    if (warp < 16) {
        const int r = tid & 127, qd = warp >> 2, t = rb * 128 + r;
        const uint4* qrow = reinterpret_cast<const uint4*>(
            p.Q + int64_t(tok0 + t) * p.q_stride_tok + int64_t(h) * p.q_stride_head + qd * (D / 4));
#pragma unroll
        for (int j = 0; j < QW / 4; ++j) {
            const uint4 v = t < Ls ? __ldg(qrow + j) : make_uint4(0u, 0u, 0u, 0u);
            qv[4 * j] = v.x; qv[4 * j + 1] = v.y; qv[4 * j + 2] = v.z; qv[4 * j + 3] = v.w;
        }
    }
    // one K/V tile of iteration `it` into ring stage it % KS (TMA producer thread only)
    auto load_tile = [&](int it) {
        const int st = it % C::KS;
        const uint32_t ph = (it / C::KS) & 1;
        const bool pre = it < nP;
        int row0 = tok0 + (it - nP) * 128, valid_rows;
        if (pre) p.pre.locate(it, row0, valid_rows);
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
    };
    const int n_early = n_iter < C::KS ? n_iter : C::KS;   // tiles whose loads go out before the set-up barrier
    if (tid == 0) {
        mbar_init(bar_Q, 512);
        mbar_init(&bar_S[0], 1); mbar_init(&bar_S[1], 1);
        for (int i = 0; i < 4; ++i) mbar_init(&bar_P[i], 256);
        mbar_init(bar_PV, 1);
        mbar_init(bar_done, 1);
        fence_mbar_init();
    }
    if (warp == 16) {
        // the producer initialises its own ring barriers and fills the ring right away: the first K/V
        // tiles travel while TMEM is allocated and Q is on its way
        if (elect_one()) {
            for (int s = 0; s < C::KS; ++s) {
                mbar_init(&bar_Kf[s], 1); mbar_init(&bar_Ke[s], 1);
                mbar_init(&bar_Vf[s], 1); mbar_init(&bar_Ve[s], 1);
            }
            fence_mbar_init();
            tma_prefetch_desc(&tmK1); tma_prefetch_desc(&tmV1);
            tma_prefetch_desc(&tmK2); tma_prefetch_desc(&tmV2);
            for (int it = 0; it < n_early; ++it) load_tile(it);
        }
        __syncwarp();
        tmem_alloc(tmem_slot, 512);
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp == 16) {
        // =============================== TMA producer ===============================
        if (elect_one()) {
            for (int it = n_early; it < n_iter; ++it) load_tile(it);
        }
    } else if (warp == 17) {
        // =============================== MMA issuer ===============================
        if (elect_one()) {
            constexpr uint32_t idesc_qk = make_idesc_bf16(128, 128, false, false);
            constexpr uint32_t idesc_pv = make_idesc_bf16(128, D, false, true);
            const uint32_t sK = smem_u32(smem + C::OFF_K), sV = smem_u32(smem + C::OFF_V);
            auto issue_S = [&](int b, int st) {  // S[b] = Q . K^T   (A = Q from TMEM)
                const uint64_t k = make_smem_desc_sw128(sK + st * C::TILE, 16, 1024);
#pragma unroll
                for (int kk = 0; kk < D / 16; ++kk)
                    mma_ts(tmem + b * 128, tmem + C::T_Q + kk * 8,
                           k + (((kk >> 2) * C::SUB + (kk & 3) * 32) >> 4), idesc_qk, kk > 0);
            };
            auto issue_PV = [&](int b, int st, int half, bool acc) {  // O += P[b][:, half] . V[half]
                const uint64_t v = make_smem_desc_sw128(sV + st * C::TILE, C::SUB, 1024);
#pragma unroll
                for (int kk = half * 4; kk < half * 4 + 4; ++kk)
                    mma_ts(tmem + C::T_O, tmem + b * 128 + (kk >> 1) * 32 + (kk & 1) * 8,
                           v + ((kk * 2048) >> 4), idesc_pv, (acc || kk > 0) ? 1u : 0u);
            };
            mbar_wait(bar_Q, 0);
            mbar_wait(&bar_Kf[0], 0);
            tc_fence_after();
            issue_S(0, 0);
            mma_commit(&bar_S[0]);
            mma_commit(&bar_Ke[0]);
            for (int it = 0; it < n_iter; ++it) {
                const int st = it % C::KS, b = it & 1;
                if (it + 1 < n_iter) {   // S(it+1) runs on the tensor pipe while softmax(it) works
                    const int st1 = (it + 1) % C::KS;
                    mbar_wait(&bar_Kf[st1], ((it + 1) / C::KS) & 1);
                    tc_fence_after();
                    issue_S(b ^ 1, st1);
                    mma_commit(&bar_S[b ^ 1]);
                    mma_commit(&bar_Ke[st1]);
                }
                mbar_wait(&bar_Vf[st], (it / C::KS) & 1);
                mbar_wait(&bar_P[2 * b], (it >> 1) & 1);
                tc_fence_after();
                issue_PV(b, st, 0, it > 0);
                mbar_wait(&bar_P[2 * b + 1], (it >> 1) & 1);
                tc_fence_after();
                issue_PV(b, st, 1, true);
                mma_commit(&bar_Ve[st]);
                mma_commit(bar_PV);
            }
            mma_commit(bar_done);
        }
    } else {
        // =============================== softmax warpgroups ===============================
        const int qd = warp >> 2;                // key-column quarter of the S tile / d quarter of Q and O
        const int r = tid & 127;                 // row in tile == TMEM lane
        const int t = rb * 128 + r;              // query row within its sequence
        const bool valid = t < Ls;
        constexpr int DQ = D / 4;                // d elements (O columns) per quarter
        const uint32_t lane_off = uint32_t((warp & 3) * 32) << 16;
        const uint32_t tO = tmem + C::T_O + qd * DQ + lane_off;          // this quarter of the O columns
        float* xch = reinterpret_cast<float*>(smem + C::OFF_X);          // [parity][quarter][128]
        const float c = p.scale_log2;
        // ---- Q row -> TMEM (A operand layout: lane = row, column j = elements 2j, 2j+1)
        {
            if constexpr (D == 128) tmem_st16(tmem + C::T_Q + qd * 16 + lane_off, qv);
            else tmem_st8(tmem + C::T_Q + qd * 8 + lane_off, qv);
            tmem_wait_st();
            tc_fence_before();
            mbar_arrive(bar_Q);
        }
        float m_used = -INFINITY, thr = -INFINITY;   // reference of the row and the rescale threshold m_used + 8
        float2 l2 = make_float2(0.f, 0.f);           // row sum of this column quarter, as two partial sums
        int rng = 0, next_end = nP > 0 ? p.pre.tile0[1] - 1 : -1;   // last tile of the current prefix range
        // one KV tile; the S buffer index b = it & 1 is a compile-time constant (the loop below is
        // unrolled by two): buffer addresses and barrier slots fold into immediates
        auto tile_step = [&](auto bc, const int it) {
            constexpr int b = decltype(bc)::v;
            const uint32_t tS = tmem + b * 128 + qd * 32 + lane_off;     // this quarter of S[b]; P at its start
            mbar_wait_short(&bar_S[b], (it >> 1) & 1);
            tc_fence_after();
            uint32_t x[32];
            tmem_ld32(tS, x);
            tmem_wait_ld();
            // visible keys of this tile for this row, relative to this quarter's first column: only the
            // last tile of a prefix range (ragged end) and the causal diagonal can hide any
            int limit = 32;
            if (it == n_iter - 1) {
                limit = t - rb * 128 + 1 - qd * 32;
            } else if (it == next_end) {
                limit = p.pre.len[rng] - (it - p.pre.tile0[rng]) * 128 - qd * 32;
                ++rng;
                next_end = rng < p.pre.n ? p.pre.tile0[rng + 1] - 1 : -1;
            }
            if (limit < 32) {                    // ragged prefix tail or causal diagonal
#pragma unroll
                for (int j = 0; j < 32; ++j)
                    if (j >= limit) x[j] = 0xf149f2cau;  // -1e30: exp2 -> 0, stays finite
            }
            float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
            for (int j = 0; j < 32; j += 2) {
                mx0 = fmaxf(mx0, __uint_as_float(x[j]));
                mx1 = fmaxf(mx1, __uint_as_float(x[j + 1]));
            }
            float* xm = xch + b * 512;
            float mine = fmaxf(mx0, mx1);
            xm[qd * 128 + r] = mine;
            named_bar_sync(1 + (warp & 3), 128);              // the row quarter's four warps (one per column quarter)
#pragma unroll
            for (int o = 1; o < 4; ++o) mine = fmaxf(mine, xm[((qd + o) & 3) * 128 + r]);
            const float m_new = mine * c;
            // lazy rescale: keep a stale max while the new one is within 2^8 of it
            const bool need = (it == 0) || (m_new > thr);
            const unsigned rescale_mask = __ballot_sync(0xffffffffu, need && it > 0);
            if (rescale_mask != 0u) {
                if ((tid & 31) == 0 && qd == 0)   // one of the row's four threads counts it
                    atomicAdd(&g_fwd_rescale_rows, (unsigned long long)__popc(rescale_mask));
                mbar_wait(bar_PV, (it - 1) & 1); // P.V(it-1) must have landed in O
                tc_fence_after();
                const float alpha = need ? fast_exp2(m_used - m_new) : 1.f;
                l2 = __fmul2_rn(l2, make_float2(alpha, alpha));
                uint32_t o[DQ];
                if constexpr (D == 128) tmem_ld32(tO, o); else tmem_ld16(tO, o);
                tmem_wait_ld();
#pragma unroll
                for (int j = 0; j < DQ; ++j) o[j] = __float_as_uint(__uint_as_float(o[j]) * alpha);
                if constexpr (D == 128) tmem_st32(tO, o); else tmem_st16(tO, o);
            }
            if (need) { m_used = m_new; thr = m_new + 8.f; }
            // ---- P = exp2(c S - m), packed to bf16 over the first 16 columns of this quarter of S
            const float2 c2 = make_float2(c, c), nm2 = make_float2(-m_used, -m_used);
            uint32_t pk[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                const float2 a = __ffma2_rn(make_float2(__uint_as_float(x[2 * j]),
                                                        __uint_as_float(x[2 * j + 1])), c2, nm2);
                float2 e;
                if ((j * C::POLY16) % 16 < C::POLY16) {   // POLY16 pairs in 16 on the FMA pipe
                    e = exp2_poly2(a);
                } else {
                    e.x = fast_exp2(a.x);
                    e.y = fast_exp2(a.y);
                }
                l2 = __fadd2_rn(l2, e);
                pk[j] = pack_bf16(e.x, e.y);
            }
            tmem_st16(tS, pk);
            tmem_wait_st();
            tc_fence_before();
            mbar_arrive(&bar_P[2 * b + (qd >> 1)]);   // this half (64 keys) of P: two quarters arrive
        };
        for (int it = 0; it < n_iter; it += 2) {
            tile_step(IntC<0>{}, it);
            if (it + 1 < n_iter) tile_step(IntC<1>{}, it + 1);
        }
        // combine the four quarters' row sums, then each quarter normalises its quarter of the O columns
        float* xl = xch + (n_iter & 1) * 512;
        float l = l2.x + l2.y;
        xl[qd * 128 + r] = l;
        named_bar_sync(1 + (warp & 3), 128);
#pragma unroll
        for (int o = 1; o < 4; ++o) l += xl[((qd + o) & 3) * 128 + r];
        mbar_wait(bar_done, 0);
        tc_fence_after();
        const float inv = 1.f / l;
        __nv_bfloat16* orow = p.O + int64_t(tok0 + t) * p.o_stride_tok + int64_t(h) * p.o_stride_head + qd * DQ;
        {
            uint32_t o[DQ];
            if constexpr (D == 128) tmem_ld32(tO, o); else tmem_ld16(tO, o);
            tmem_wait_ld();
            if (valid) {
#pragma unroll
                for (int j = 0; j < DQ; j += 8) {
                    uint4 v;
                    v.x = pack_bf16(__uint_as_float(o[j + 0]) * inv, __uint_as_float(o[j + 1]) * inv);
                    v.y = pack_bf16(__uint_as_float(o[j + 2]) * inv, __uint_as_float(o[j + 3]) * inv);
                    v.z = pack_bf16(__uint_as_float(o[j + 4]) * inv, __uint_as_float(o[j + 5]) * inv);
                    v.w = pack_bf16(__uint_as_float(o[j + 6]) * inv, __uint_as_float(o[j + 7]) * inv);
                    *reinterpret_cast<uint4*>(orow + j) = v;
                }
            }
        }
        if (valid && qd == 0)
            p.LSE[int64_t(h) * p.lse_stride + tok0 + t] = (m_used + log2f(l)) * 0.6931471805599453f;
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 16) tmem_dealloc(tmem, 512);
}

}  // namespace pf
