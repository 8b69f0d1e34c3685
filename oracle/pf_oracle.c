/*
 * pf_oracle.c -- fp64 CPU ORACLE for the PrefixFlow attention hot path.  TEST INFRASTRUCTURE.
 *
 * This file is test infrastructure, not product: only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no code,
 * header, table or helper with the CUDA library under paper_2606_01143_b200/csrc/.
 *
 * What it computes (the DEFINITION the schedule must reach; "changes only the order of
 * computation", "equivalent ... over real arithmetic"): plain full-sequence causal
 * attention forward and backward on ONE concatenated trajectory [P || S(i)] of T tokens, token-major
 * layout [T, H, d], GQA head map kappa(h) = h / G with G = Hq / Hkv (reading 6).
 * For q-head h, kv-head g = kappa(h), row t, keys j <= t (inclusive diagonal, reading 5):
 *
 *   s_tj   = sigma * <q[h,t], k[g,j]>              LSE[h,t] = log sum_{j<=t} exp(s_tj)  (natural log)
 *   p_tj   = exp(s_tj - LSE[h,t])                  o[h,t]   = sum_{j<=t} p_tj v[g,j]
 *   delta  = <do[h,t], o[h,t]>                     dp_tj    = <do[h,t], v[g,j]>
 *   ds_tj  = p_tj (dp_tj - delta[h,t])
 *   dq[h,t] = sigma sum_{j<=t} ds_tj k[g,j]
 *   dk[g,j] = sigma sum_{h in kappa^-1(g)} sum_{t>=j} ds_tj q[h,t]
 *   dv[g,j] =       sum_{h in kappa^-1(g)} sum_{t>=j} p_tj  do[h,t]
 *
 * Restricted to keys j < Lp and rows t >= Lp the last two lines are exactly the paper's coupling
 * gradients gK1 = (1/sqrt(d_h)) dS21^T Q2 and gV1 = P21^T dH2; the caller selects that
 * restriction through the row range [r0, r1) of pfo_cols.
 *
 * Structure: two primitives, no blocking, no fusion, one row / one key column at a time.
 *   pfo_rows: for a list of (h, t) rows -> o, LSE, delta, dq     (row of scores -> max -> exp -> sum)
 *   pfo_cols: for a list of (g, j) key columns and a row range [r0, r1) -> dk, dv contributions of
 *             rows max(j, r0) <= t < r1, recomputing p_tj from the LSE of pfo_rows.
 * OpenMP parallelises over list items only (each item is written by one thread; no reductions
 * across threads, so results do not depend on the thread count).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): central finite differences, the paper's equivalence
 * invariant against an independent matrix-form evaluation of PAPER.md:196 (1e-10), prefix isolation,
 * closed forms (row 0, Q = 0, equal keys), shift invariances, the LSE-merge identity, torch's
 * float64 CPU scaled_dot_product_attention + autograd, organisation independence, and a hand-worked
 * two-token example (tests/golden/two_token.txt).  No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int64_t T;      /* tokens in the concatenated sequence */
    int32_t Hq;     /* query heads */
    int32_t Hkv;    /* key/value heads, Hq % Hkv == 0 */
    int32_t d;      /* head dim */
    double sigma;   /* softmax scale, 1/sqrt(d) unless overridden */
} pfo_shape;

int pfo_version(void) { return 1; }

int pfo_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static inline const double* at(const double* x, int64_t t, int32_t h, int32_t H, int32_t d) {
    return x + ((size_t)t * (size_t)H + (size_t)h) * (size_t)d;
}

static double dot(const double* a, const double* b, int32_t d) {
    double s = 0.0;
    for (int32_t c = 0; c < d; ++c) s += a[c] * b[c];
    return s;
}

/*
 * Rows.  q, dO: [T, Hq, d];  k, v: [T, Hkv, d].  For item n = (hs[n], ts[n]):
 *   o[n, :], lse[n], delta[n], dq[n, :].   dO may be NULL: then delta and dq are not written.
 * Returns 0, or 1 on a bad argument.
 */
int pfo_rows(const pfo_shape* sh, const double* q, const double* k, const double* v,
             const double* dO, int64_t n_items, const int32_t* hs, const int64_t* ts,
             double* o, double* lse, double* delta, double* dq) {
    if (!sh || !q || !k || !v || sh->Hkv <= 0 || sh->Hq % sh->Hkv != 0 || sh->d <= 0) return 1;
    const int32_t d = sh->d, Hq = sh->Hq, Hkv = sh->Hkv, G = Hq / Hkv;
    const double sigma = sh->sigma;
    int bad = 0;
#pragma omp parallel
    {
        double* p = (double*)malloc(sizeof(double) * (size_t)(sh->T > 0 ? sh->T : 1));
#pragma omp for schedule(dynamic, 16)
        for (int64_t n = 0; n < n_items; ++n) {
            const int32_t h = hs[n];
            const int64_t t = ts[n];
            if (h < 0 || h >= Hq || t < 0 || t >= sh->T) {
#pragma omp atomic write
                bad = 1;
                continue;
            }
            const int32_t g = h / G;
            const double* qt = at(q, t, h, Hq, d);
            /* row of scaled scores, its maximum */
            double m = -INFINITY;
            for (int64_t j = 0; j <= t; ++j) {
                p[j] = sigma * dot(qt, at(k, j, g, Hkv, d), d);
                if (p[j] > m) m = p[j];
            }
            /* LSE = m + log sum exp(s - m);  p = exp(s - LSE) */
            double z = 0.0;
            for (int64_t j = 0; j <= t; ++j) z += exp(p[j] - m);
            const double L = m + log(z);
            for (int64_t j = 0; j <= t; ++j) p[j] = exp(p[j] - L);
            double* on = o + (size_t)n * d;
            for (int32_t c = 0; c < d; ++c) on[c] = 0.0;
            for (int64_t j = 0; j <= t; ++j) {
                const double* vj = at(v, j, g, Hkv, d);
                for (int32_t c = 0; c < d; ++c) on[c] += p[j] * vj[c];
            }
            lse[n] = L;
            if (dO) {
                const double* dot_ = at(dO, t, h, Hq, d);
                const double dl = dot(dot_, on, d);
                delta[n] = dl;
                double* dqn = dq + (size_t)n * d;
                for (int32_t c = 0; c < d; ++c) dqn[c] = 0.0;
                for (int64_t j = 0; j <= t; ++j) {
                    const double dp = dot(dot_, at(v, j, g, Hkv, d), d);
                    const double ds = p[j] * (dp - dl);
                    const double* kj = at(k, j, g, Hkv, d);
                    for (int32_t c = 0; c < d; ++c) dqn[c] += ds * kj[c];
                }
                for (int32_t c = 0; c < d; ++c) dqn[c] *= sigma;
            }
        }
        free(p);
    }
    return bad;
}

/*
 * Key columns.  lse, delta: full [Hq, T] arrays (row statistics from pfo_rows); only entries of
 * the heads of group g and rows max(j, r0) <= t < r1 are read.  For item n = (gs[n], js[n]):
 *   dk[n, :] = sigma sum_h sum_t ds_tj q[h,t],   dv[n, :] = sum_h sum_t p_tj do[h,t]
 * with h over kappa^-1(g) in increasing order and t increasing (fixed summation order).
 */
int pfo_cols(const pfo_shape* sh, const double* q, const double* k, const double* v,
             const double* dO, const double* lse, const double* delta,
             int64_t n_items, const int32_t* gs, const int64_t* js, int64_t r0, int64_t r1,
             double* dk, double* dv) {
    if (!sh || !q || !k || !v || !dO || !lse || !delta || sh->Hkv <= 0 ||
        sh->Hq % sh->Hkv != 0 || sh->d <= 0)
        return 1;
    const int32_t d = sh->d, Hq = sh->Hq, Hkv = sh->Hkv, G = Hq / Hkv;
    const double sigma = sh->sigma;
    if (r1 > sh->T) r1 = sh->T;
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t n = 0; n < n_items; ++n) {
        const int32_t g = gs[n];
        const int64_t j = js[n];
        if (g < 0 || g >= Hkv || j < 0 || j >= sh->T) {
#pragma omp atomic write
            bad = 1;
            continue;
        }
        const double* kj = at(k, j, g, Hkv, d);
        const double* vj = at(v, j, g, Hkv, d);
        double* dkn = dk + (size_t)n * d;
        double* dvn = dv + (size_t)n * d;
        for (int32_t c = 0; c < d; ++c) { dkn[c] = 0.0; dvn[c] = 0.0; }
        const int64_t tb = j > r0 ? j : r0;
        for (int32_t h = g * G; h < (g + 1) * G; ++h) {
            for (int64_t t = tb; t < r1; ++t) {
                const double* qt = at(q, t, h, Hq, d);
                const double* dot_ = at(dO, t, h, Hq, d);
                const double s = sigma * dot(qt, kj, d);
                const double p = exp(s - lse[(size_t)h * sh->T + t]);
                const double dp = dot(dot_, vj, d);
                const double ds = p * (dp - delta[(size_t)h * sh->T + t]);
                for (int32_t c = 0; c < d; ++c) {
                    dkn[c] += ds * qt[c];
                    dvn[c] += p * dot_[c];
                }
            }
        }
        for (int32_t c = 0; c < d; ++c) dkn[c] *= sigma;
    }
    return bad;
}
