// prefixflow.cu -- the C ABI declared in include/prefixflow.h: argument validation, TMA
// descriptors, workspace carving and kernel launches.  No arithmetic of the method lives on the
// host; every step runs in the kernels of attn_fwd.cuh / attn_bwd.cuh / aux_kernels.cuh.
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdarg>
#include <cstdio>
#include <cstddef>
#include <cstring>
#include <cmath>
#include <algorithm>
#include <functional>
#include <mutex>
#include <new>
#include <queue>
#include <vector>

#include "../../include/prefixflow.h"
#include "attn_fwd.cuh"
#include "attn_bwd.cuh"
#include "aux_kernels.cuh"
#include "companions.cuh"

namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

constexpr int64_t kAlign = 256;
constexpr size_t kMaxProfRecords = 1 << 16;   // unread profiling records kept per context
inline int64_t align_up(int64_t x, int64_t a) { return (x + a - 1) / a * a; }

// size of the built-in scratch of pf_causal_bwd_static (PF_STATIC_SCRATCH_BYTES in the header)
constexpr size_t kStaticScratchBytes = size_t(32) << 20;
constexpr int kMaxDevices = 64;

}  // namespace

// Built-in scratch of pf_causal_bwd_static: the backward's workspace (statistics, fp32 dQ^T tiles,
// fp32 dK/dV staging) for callers that may not allocate.  Every GPU that loads the library holds
// these 32 MiB until the process exits.  In host code this name is only a stand-in for the symbol:
// the device address comes from cudaGetSymbolAddress (pf_create, once per context = per device, with
// that device current) and is what the launches receive.
static __device__ __align__(256) unsigned char pf_static_scratch[kStaticScratchBytes];

struct ProfRec {
    cudaEvent_t a, b;
    int kind;
};

// key / value of the backward item-split model (choose_split below)
struct SplitEntry {
    int n, nPT, Hkv, G, interleave;
    int cu[pf::kMaxSeqs + 1];
    int ppcP, ppcC;
};

struct pf_ctx {
    int device = 0;
    int num_sms = 0;
    EncodeTiledFn encode = nullptr;
    uint8_t* static_scratch = nullptr;   // device address of pf_static_scratch on this context's device
    int bwd_pairs_per_item = 0;  // (seq, head) pairs per prefix-tile CTA; 0 = heuristic
    int bwd_heads_per_item = 0;  // query heads per causal-tile CTA; 0 = heuristic
    int bwd_interleave = 1;      // 1 (default): causal items launched right behind the prefix chunk that completes their sequence
    bool profile = false;
    bool zero_accumulators = true;
    bool deterministic_gkv = false;  // one CTA per key tile: gK1/gV1/dK/dV sums in a fixed order
    int64_t n_launches = 0;
    int last_ppcP = 0, last_ppcC = 0;      // split of the most recent backward launch (pf_counter)
    std::vector<SplitEntry> split_cache;   // backward item splits already modelled (pf_ctx is not thread-safe)
    std::vector<ProfRec> prof;         // recorded, not yet read
    std::vector<cudaEvent_t> ev_pool;  // recycled events
    char err[512] = {0};
};

// K and V tensor maps of one KV source with one box height
struct KvMaps {
    CUtensorMap k, v;
};

struct pf_group {
    pf_ctx* ctx;
    pf_desc desc;
    float sigma;
    int64_t Lp;
    pf_tensor K1, V1;
    float* gK1;
    float* gV1;
    uint8_t* ws;
    size_t ws_bytes;
    int64_t ws_cap;  // padded token positions the workspace holds (multiple of 64)
    pf::PrefixRanges pre;  // visible ranges of the prefix source (default: [0, Lp))
    int state;  // 0 begun, 1 A done, 2 C done
    // descriptor cache: the tensor maps of the borrowed cache tensors are encoded once per group
    KvMaps kv128;          // K1/V1 with 128-row boxes (both attention kernels)
    KvMaps acc;            // gK1 / gV1 reduce-add maps (valid when gK1 != NULL)
};

namespace {

pf_status fail(pf_ctx* ctx, pf_status st, const char* fmt, ...) {
    if (ctx) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
        va_end(ap);
    }
    return st;
}

#define PF_CUDA(ctx, call)                                                              \
    do {                                                                                \
        cudaError_t e_ = (call);                                                        \
        if (e_ != cudaSuccess)                                                          \
            return fail(ctx, PF_CUDA_ERROR, "%s failed: %s", #call, cudaGetErrorString(e_)); \
    } while (0)

cudaEvent_t prof_event(pf_ctx* ctx) {
    cudaEvent_t e = nullptr;
    if (!ctx->ev_pool.empty()) {
        e = ctx->ev_pool.back();
        ctx->ev_pool.pop_back();
    } else if (cudaEventCreate(&e) != cudaSuccess) {
        e = nullptr;
    }
    return e;
}

// RAII bracket: records an event pair around one attention kernel launch when profiling is on
struct ProfScope {
    pf_ctx* ctx;
    cudaStream_t s;
    ProfRec r{nullptr, nullptr, 0};
    ProfScope(pf_ctx* c, int kind, cudaStream_t st) : ctx(c), s(st) {
        if (!ctx->profile) return;
        if (ctx->prof.size() >= kMaxProfRecords) return;   // nobody is reading: stop recording
        r.kind = kind;
        r.a = prof_event(ctx);
        r.b = prof_event(ctx);
        if (!r.a || !r.b) {                                // keep the one that was created
            if (r.a) ctx->ev_pool.push_back(r.a);
            if (r.b) ctx->ev_pool.push_back(r.b);
            r.a = r.b = nullptr;
            return;
        }
        cudaEventRecord(r.a, s);
    }
    ~ProfScope() {
        if (!r.a || !r.b) return;
        cudaEventRecord(r.b, s);
        ctx->prof.push_back(r);
    }
};

// The context is bound to one device: launches, memsets and tensor-map encodes must run with that
// device current (the header's contract); a mismatch is the caller's phase/order error.
pf_status check_device(pf_ctx* ctx) {
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess) return fail(ctx, PF_CUDA_ERROR, "cudaGetDevice failed");
    if (cur != ctx->device)
        return fail(ctx, PF_STATE, "current CUDA device %d is not the context's device %d", cur, ctx->device);
    return PF_OK;
}

pf_status check_desc(pf_ctx* ctx, const pf_desc* d) {
    if (!d) return fail(ctx, PF_INVALID_ARG, "desc is NULL");
    if (d->n_q_heads <= 0 || d->n_kv_heads <= 0 || d->n_q_heads % d->n_kv_heads != 0)
        return fail(ctx, PF_INVALID_ARG, "n_q_heads=%d must be a positive multiple of n_kv_heads=%d",
                    d->n_q_heads, d->n_kv_heads);
    if (d->head_dim != 64 && d->head_dim != 128)
        return fail(ctx, PF_UNSUPPORTED, "head_dim=%d not in {64,128}", d->head_dim);
    if (!(d->softmax_scale >= 0.f) || std::isinf(d->softmax_scale))
        return fail(ctx, PF_INVALID_ARG, "softmax_scale must be finite and >= 0");
    if (d->n_q_heads > 65535) return fail(ctx, PF_UNSUPPORTED, "n_q_heads > 65535");
    return PF_OK;
}

// bf16 [L, H, d] strided tensor: pointer / stride rules of the TMA tiled mode
pf_status check_tensor(pf_ctx* ctx, const char* name, const pf_tensor& t, int64_t L, int H, int d) {
    if (L == 0) return PF_OK;
    if (!t.ptr) return fail(ctx, PF_INVALID_ARG, "%s.ptr is NULL", name);
    if (reinterpret_cast<uintptr_t>(t.ptr) % 16 != 0)
        return fail(ctx, PF_INVALID_ARG, "%s.ptr must be 16-byte aligned", name);
    if (t.stride_tok < d || t.stride_tok % 8 != 0)
        return fail(ctx, PF_INVALID_ARG, "%s.stride_tok=%lld must be >= d and a multiple of 8", name,
                    (long long)t.stride_tok);
    if (H > 1 && (t.stride_head < d || t.stride_head % 8 != 0))
        return fail(ctx, PF_INVALID_ARG, "%s.stride_head=%lld must be >= d and a multiple of 8", name,
                    (long long)t.stride_head);
    if (t.stride_tok * 2 >= (int64_t(1) << 40) || t.stride_head * 2 >= (int64_t(1) << 40))
        return fail(ctx, PF_INVALID_ARG, "%s strides too large", name);
    return PF_OK;
}

// 3-D map {d, H, L}, box {64, 1, rows}, swizzle-128B: one load = a [rows tokens][64 elements]
// K-major sub-tile of one head; rows past L are zero-filled.
pf_status make_map(pf_ctx* ctx, CUtensorMap* m, const char* name, const pf_tensor& t, int64_t L,
                   int H, int d, int rows = 128) {
    if (L == 0) {
        memset(m, 0, sizeof(*m));
        return PF_OK;
    }
    cuuint64_t dims[3] = {cuuint64_t(d), cuuint64_t(H), cuuint64_t(L)};
    cuuint64_t strides[2] = {cuuint64_t((H > 1 ? t.stride_head : int64_t(d)) * 2),
                             cuuint64_t(t.stride_tok * 2)};
    cuuint32_t box[3] = {64, 1, cuuint32_t(rows)};
    cuuint32_t es[3] = {1, 1, 1};
    CUresult r = ctx->encode(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, t.ptr, dims, strides, box, es,
                             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                             CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS)
        return fail(ctx, PF_CUDA_ERROR, "cuTensorMapEncodeTiled(%s) failed with CUresult %d", name,
                    int(r));
    return PF_OK;
}

// fp32 accumulator [L, H, d] contiguous: box {32, 1, 128} (128-byte rows, swizzle-128B) for the
// reduce-add of a [128 keys][32 floats] staging tile; rows past L are clipped.
pf_status make_acc_map(pf_ctx* ctx, CUtensorMap* m, const char* name, float* ptr, int64_t L, int H,
                       int d) {
    if (L == 0 || !ptr) {
        memset(m, 0, sizeof(*m));
        return PF_OK;
    }
    cuuint64_t dims[3] = {cuuint64_t(d), cuuint64_t(H), cuuint64_t(L)};
    cuuint64_t strides[2] = {cuuint64_t(d) * 4, cuuint64_t(H) * d * 4};
    cuuint32_t box[3] = {32, 1, 128};
    cuuint32_t es[3] = {1, 1, 1};
    CUresult r = ctx->encode(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, ptr, dims, strides, box, es,
                             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                             CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS)
        return fail(ctx, PF_CUDA_ERROR, "cuTensorMapEncodeTiled(%s) failed with CUresult %d", name,
                    int(r));
    return PF_OK;
}

// Workspace carving for `cap` padded token positions (multiple of 64): softmax statistics, the
// fp32 dQ^T tiles and the fp32 dK2/dV2 staging of the causal source.
struct WsLayout {
    int64_t off_lse2, off_delta, off_dq, off_ak, off_av, total;
    int64_t stat_stride;
};

int64_t ws_bytes_per_pos(const pf_desc& d) {
    return int64_t(d.n_q_heads) * 8 + int64_t(d.n_q_heads) * d.head_dim * 4 +
           int64_t(d.n_kv_heads) * d.head_dim * 8;
}

WsLayout ws_layout(const pf_desc& d, int64_t cap) {
    WsLayout w;
    w.stat_stride = cap;
    int64_t o = 0;
    w.off_lse2 = o; o += align_up(int64_t(d.n_q_heads) * cap * 4, kAlign);
    w.off_delta = o; o += align_up(int64_t(d.n_q_heads) * cap * 4, kAlign);
    w.off_dq = o; o += align_up(cap * d.n_q_heads * d.head_dim * 4, kAlign);
    w.off_ak = o; o += align_up(cap * d.n_kv_heads * d.head_dim * 4, kAlign);
    w.off_av = o; o += align_up(cap * d.n_kv_heads * d.head_dim * 4, kAlign);
    w.total = o;
    return w;
}

// largest capacity whose layout fits `bytes`
int64_t ws_capacity(const pf_desc& d, size_t bytes) {
    const int64_t slack = 6 * kAlign;
    if (int64_t(bytes) <= slack) return 0;
    return (int64_t(bytes) - slack) / ws_bytes_per_pos(d) / 64 * 64;
}

template <int MH, int BN>
bool set_gemm_attr() {
    return cudaFuncSetAttribute(pf::kv_proj_grad_kernel<MH, BN>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                pf::GemmCfg<MH, BN>::SMEM) == cudaSuccess;
}
template <int MH, int BN>
void launch_gemm(dim3 grid, cudaStream_t s, const CUtensorMap& mX, const CUtensorMap& mY, float* dW, int n_cols,
                 int n_chunks, int cps) {
    pf::kv_proj_grad_kernel<MH, BN><<<grid, pf::GemmCfg<MH, BN>::THREADS, pf::GemmCfg<MH, BN>::SMEM, s>>>(
        mX, mY, dW, n_cols, n_chunks, cps);
}

template <int D>
pf_status set_attrs() {
    cudaError_t e;
    e = cudaFuncSetAttribute(pf::attn_fwd_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             pf::FwdCfg<D>::SMEM);
    if (e != cudaSuccess) return PF_CUDA_ERROR;
    e = cudaFuncSetAttribute(pf::attn_bwd_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             pf::BwdCfg<D>::SMEM);
    if (e != cudaSuccess) return PF_CUDA_ERROR;
    return PF_OK;
}

pf::PrefixRanges whole_prefix(int64_t Lp) {
    pf::PrefixRanges r;
    memset(&r, 0, sizeof(r));
    if (Lp > 0) {
        r.n = 1;
        r.len[0] = int(Lp);
        r.tile0[1] = int((Lp + 127) / 128);
    }
    return r;
}

// Sequence table of one launch from host offsets cu[0..n] (cu[0] = 0, n <= kMaxSeqs)
pf::SeqTable make_seq_table(int n, const int64_t* cu) {
    pf::SeqTable t;
    memset(&t, 0, sizeof(t));
    t.n = n;
    for (int s = 0; s <= n; ++s) t.cu[s] = int(cu[s]);
    for (int s = 0; s < n; ++s) {
        const int Ls = t.cu[s + 1] - t.cu[s];
        t.pqs[s + 1] = t.pqs[s] + (Ls + 63) / 64;
        t.ckt[s + 1] = t.ckt[s] + (Ls + 127) / 128;
    }
    return t;
}

// ---- backward item split.  The backward launches one CTA per ITEM = (key tile, KV head, chunk of
// the (sequence, query head) pairs that see the tile); the hardware hands items to SMs in launch
// order as SMs free up (list scheduling).  Too few chunks leave SMs idle in the last round, too many
// re-load K/V, re-allocate TMEM and add more partial dK/dV tiles.  Instead of a closed-form guess the
// host SIMULATES that list scheduling for a handful of chunk sizes (cost of an item = its
// iterations + c0 for prologue and epilogue, in units of one 128 x 64 iteration) and takes the split
// with the shortest makespan.  Fitted on one-call-per-suffix launches of configs[1]: c0 = 6 predicts the
// measured kernel times of 15 splits within 1.8 % on average.  Measured against the round-1 closed form
// (fresh processes, alternating, same GPU; profiles/r2_kernel_experiments.md): configs[1] B bwd +2 %,
// C bwd +8 %, one call per suffix +4.5 %; configs[4] C bwd +14 %, whole step -9 % time.
struct SplitModel {
    const pf::SeqTable& seq;
    int n, nPT, Hkv, G, sms;
    static constexpr double kC0 = 6.0;
    // exact list scheduling in the kernel's launch order on a binary min-heap `h` of SM finish times
    static void give(std::vector<double>& h, double cost) {  // next item goes to the SM that frees up first
        const int sms = int(h.size());
        const double v = h[0] + cost;
        int i = 0;
        for (;;) {                                          // sift down
            int c = 2 * i + 1;
            if (c >= sms) break;
            if (c + 1 < sms && h[c + 1] < h[c]) ++c;
            if (h[c] >= v) break;
            h[i] = h[c];
            i = c;
        }
        h[i] = v;
    }
    void prefix_phase(int ppcP, std::vector<double>& h) const {
        h.assign(sms, 0.0);
        const int pairs = n * G;
        if (nPT == 0 || pairs == 0) return;
        for (int lo = 0; lo < pairs; lo += ppcP) {          // chunk-major: all key tiles of a chunk cost the same
            const int hi = std::min(pairs, lo + ppcP);
            double it = 0;
            for (int pr = lo; pr < hi; ++pr) it += seq.pqs[pr / G + 1] - seq.pqs[pr / G];
            int64_t cnt = int64_t(nPT) * Hkv;
            const double cost = it + kC0;
            // whole rounds of equal items give every SM one item each -- exactly what list
            // scheduling does as long as the finish times differ by no more than one item
            if (cnt >= sms && *std::max_element(h.begin(), h.end()) - h[0] <= cost) {
                const double add = cost * double(cnt / sms);
                for (double& v : h) v += add;
                cnt %= sms;
            }
            for (; cnt > 0; --cnt) give(h, cost);
        }
    }
    double causal_phase(int ppcC, std::vector<double>& h) const {
        for (int s = 0; s < n; ++s) {
            const int nqs = seq.pqs[s + 1] - seq.pqs[s], nkt = seq.ckt[s + 1] - seq.ckt[s];
            for (int kt = 0; kt < nkt; ++kt) {
                const int rows = std::max(0, nqs - 2 * kt);
                for (int g = 0; g < Hkv; ++g)
                    for (int c0 = 0; c0 < G; c0 += ppcC)
                        give(h, rows > 0 ? double(std::min(G, c0 + ppcC) - c0) * rows + kC0 : 0.5);
            }
        }
        return *std::max_element(h.begin(), h.end());
    }
    // the interleaved launch order: chunk by chunk, prefix items then the causal items of the sequences
    // the chunk completes
    double interleaved(int ppcP, int ppcC, std::vector<double>& h) const {
        h.assign(sms, 0.0);
        const int pairs = n * G;
        int s_lo = 0;
        for (int lo = 0; lo < pairs; lo += ppcP) {
            const int hi = std::min(pairs, lo + ppcP);
            double it = 0;
            for (int pr = lo; pr < hi; ++pr) it += seq.pqs[pr / G + 1] - seq.pqs[pr / G];
            int64_t cnt = int64_t(nPT) * Hkv;
            const double cost = it + kC0;
            if (cnt >= sms && *std::max_element(h.begin(), h.end()) - h[0] <= cost) {
                const double add = cost * double(cnt / sms);
                for (double& v : h) v += add;
                cnt %= sms;
            }
            for (; cnt > 0; --cnt) give(h, cost);
            const int s_hi = hi / G;
            for (int s = s_lo; s < s_hi; ++s) {
                const int nqs = seq.pqs[s + 1] - seq.pqs[s], nkt = seq.ckt[s + 1] - seq.ckt[s];
                for (int kt = 0; kt < nkt; ++kt) {
                    const int rows = std::max(0, nqs - 2 * kt);
                    for (int g = 0; g < Hkv; ++g)
                        for (int c0 = 0; c0 < G; c0 += ppcC)
                            give(h, rows > 0 ? double(std::min(G, c0 + ppcC) - c0) * rows + kC0 : 0.5);
                }
            }
            s_lo = s_hi;
        }
        return *std::max_element(h.begin(), h.end());
    }
    bool interleave = false;
    void choose(int& ppcP, int& ppcC) const {
        const int pairs = n * G;
        static const int kChunks[] = {1, 2, 3, 4, 5, 6, 7, 8, 10, 12, 14, 16, 20, 24, 28, 32, 40, 48, 56, 64, 96, 128};
        std::vector<int> as, bs;                            // candidate pairs per prefix item / heads per causal item
        if (nPT > 0 && pairs > 0) {
            const double per_chunk = double(nPT) * Hkv / sms;   // prefix items per SM and chunk
            for (int ch : kChunks) {
                if (ch > pairs) break;
                if (ch > 1 && ch * per_chunk > 16.0) break;     // more than ~16 prefix items per SM never paid
                const int a = (pairs + ch - 1) / ch;
                if (as.empty() || as.back() != a) as.push_back(a);
            }
        } else {
            as.push_back(std::max(1, pairs));
        }
        for (int b : {1, 2, (G + 1) / 2, G})                // the most even split of 1, 2, ~G/2 and G heads per item
            if (b >= 1 && b <= G && std::find(bs.begin(), bs.end(), b) == bs.end()) bs.push_back(b);
        double bm = 1e300;
        std::vector<double> after_prefix, h;
        for (int a : as) {
            if (!(interleave && nPT > 0)) prefix_phase(a, after_prefix);
            for (int b : bs) {
                double m;
                if (interleave && nPT > 0) {
                    m = interleaved(a, b, h);
                } else {
                    h = after_prefix;
                    m = causal_phase(b, h);
                }
                if (getenv("PF_SPLIT_DEBUG")) fprintf(stderr, "split a=%d b=%d makespan=%.1f\n", a, b, m);
                // ties (0.2 %): fewer, longer items -- less K/V re-loading, and CTAs that run side by
                // side then walk the same query heads, which keeps their Q / dO tiles in L2 (measured at
                // configs[4]: 2 instead of 5 heads per causal item costs Phase C 44 %)
                const bool tie = m <= bm * 1.002 && m >= bm * 0.998;
                const bool tie_better = a > ppcP || (a == ppcP && b > ppcC);
                if (m < bm * 0.998 || (tie && tie_better)) {
                    bm = std::min(bm, m); ppcP = a; ppcC = b;
                }
            }
        }
    }
};

// ---- forward launch over n sequences packed along the token axis: the queries of sequence s
// attend to the prefix source [Lp] (all visible) + the keys of s causally
// `prefix`: cached maps of the prefix source (NULL when Lp = 0); `causal`: cached maps of the causal
// source when it is the group's own K1/V1 (Phase A), else NULL and K2/V2 are encoded here.
template <int D>
pf_status launch_fwd(pf_group* g, const pf_tensor& Q, const KvMaps* prefix, int64_t Lp,
                     const KvMaps* causal, const pf_tensor& K2, const pf_tensor& V2, const pf_tensor& O,
                     float* LSE, int64_t lse_stride, int n, const int64_t* cu, int prof_kind,
                     cudaStream_t s) {
    pf_ctx* ctx = g->ctx;
    const int Hq = g->desc.n_q_heads, Hkv = g->desc.n_kv_heads;
    const int64_t total = cu[n];
    KvMaps own;
    pf_status st;
    if (!causal) {
        if ((st = make_map(ctx, &own.k, "K", K2, total, Hkv, D))) return st;
        if ((st = make_map(ctx, &own.v, "V", V2, total, Hkv, D))) return st;
        causal = &own;
    }
    if (Lp == 0 || !prefix) prefix = causal;
    const CUtensorMap &mK1 = prefix->k, &mV1 = prefix->v, &mK2 = causal->k, &mV2 = causal->v;
    pf::FwdParams p;
    p.Q = static_cast<const __nv_bfloat16*>(Q.ptr);
    p.q_stride_tok = Q.stride_tok;
    p.q_stride_head = Q.stride_head;
    p.O = static_cast<__nv_bfloat16*>(O.ptr);
    p.o_stride_tok = O.stride_tok;
    p.o_stride_head = O.stride_head;
    p.LSE = LSE;
    p.lse_stride = lse_stride;
    p.pre = Lp > 0 ? g->pre : whole_prefix(0);
    p.Hq = Hq;
    p.Hkv = Hkv;
    p.G = Hq / Hkv;
    p.scale_log2 = g->sigma * 1.4426950408889634f;
    p.seq = make_seq_table(n, cu);
    int ctas = 0;   // one CTA per (128-row block, query head of the KV head's group)
    for (int i = 0; i < n; ++i) ctas += (p.seq.ckt[i + 1] - p.seq.ckt[i]) * p.G;
    if (ctas == 0) return PF_OK;
    dim3 grid(ctas, Hkv);
    {
        ProfScope prof(ctx, prof_kind, s);
        pf::attn_fwd_kernel<D><<<grid, pf::FwdCfg<D>::THREADS, pf::FwdCfg<D>::SMEM, s>>>(
            mK1, mV1, mK2, mV2, p);
    }
    PF_CUDA(ctx, cudaGetLastError());
    ctx->n_launches += 1;
    return PF_OK;
}

// ---- backward launch over a wave of n sequences packed along the token axis.  Keys of the prefix
// source accumulate into accK1/accV1 (fp32, +=), keys of the causal source into accK2/accV2
// (fp32 [total, Hkv, d], +=); dQ goes through the fp32 tile workspace and is rounded to bf16 once
// all key tiles have contributed.  zero_acc2: accK2/accV2 are scratch and are zero-filled here (by the
// pre-processing launch) instead of accumulated onto.
// `prefix` / `prefix_acc`: cached maps of the prefix source and of its accumulators (NULL when
// Lp = 0); `causal` / `causal_acc`: cached maps when the causal source is the group's own K1/V1 and
// gK1/gV1 (Phase C), else NULL and K2/V2/accK2/accV2 are encoded here.
template <int D>
pf_status launch_bwd(pf_group* g, const pf_tensor& Q, const KvMaps* prefix, const KvMaps* prefix_acc,
                     int64_t Lp, const KvMaps* causal, const KvMaps* causal_acc, const pf_tensor& K2,
                     const pf_tensor& V2, const pf_tensor& O, const float* LSE, int64_t lse_stride,
                     const pf_tensor& dO, float* accK2, float* accV2, const pf_tensor& dQ, int n,
                     const int64_t* cu, int prof_kind, bool zero_acc2, cudaStream_t s) {
    pf_ctx* ctx = g->ctx;
    const int Hq = g->desc.n_q_heads, Hkv = g->desc.n_kv_heads, G = Hq / Hkv;
    const pf::SeqTable seq = make_seq_table(n, cu);
    const int64_t total = cu[n];
    const int nQS = seq.pqs[n];
    const int64_t npad = int64_t(nQS) * 64;
    if (npad > g->ws_cap)
        return fail(ctx, PF_WORKSPACE, "workspace too small: %lld padded positions, capacity %lld",
                    (long long)npad, (long long)g->ws_cap);
    const WsLayout w = ws_layout(g->desc, g->ws_cap);
    float* lse2 = reinterpret_cast<float*>(g->ws + w.off_lse2);
    float* delta = reinterpret_cast<float*>(g->ws + w.off_delta);
    float* dqacc = reinterpret_cast<float*>(g->ws + w.off_dq);

    CUtensorMap mQ, mdO;
    KvMaps own, own_acc;
    pf_status st;
    if ((st = make_map(ctx, &mQ, "Q", Q, total, Hq, D, 64))) return st;
    if ((st = make_map(ctx, &mdO, "dO", dO, total, Hq, D, 64))) return st;
    if (!causal) {
        if ((st = make_map(ctx, &own.k, "K", K2, total, Hkv, D))) return st;
        if ((st = make_map(ctx, &own.v, "V", V2, total, Hkv, D))) return st;
        causal = &own;
    }
    if (!causal_acc) {
        if ((st = make_acc_map(ctx, &own_acc.k, "accK2", accK2, total, Hkv, D))) return st;
        if ((st = make_acc_map(ctx, &own_acc.v, "accV2", accV2, total, Hkv, D))) return st;
        causal_acc = &own_acc;
    }
    if (Lp == 0 || !prefix) {
        prefix = causal;
        prefix_acc = causal_acc;
    }
    const CUtensorMap &mK1 = prefix->k, &mV1 = prefix->v, &mK2 = causal->k, &mV2 = causal->v;
    const CUtensorMap &mAK1 = prefix_acc->k, &mAV1 = prefix_acc->v, &mAK2 = causal_acc->k, &mAV2 = causal_acc->v;
    {   // delta / lse2 and the zero fill of dqacc (npad * Hq * D floats) in one launch
        const int64_t threads = npad * (D / 8);
        dim3 grid(unsigned((threads + 255) / 256), Hq);
        pf::bwd_preprocess_kernel<D><<<grid, 256, 0, s>>>(
            static_cast<const __nv_bfloat16*>(O.ptr), O.stride_tok, O.stride_head,
            static_cast<const __nv_bfloat16*>(dO.ptr), dO.stride_tok, dO.stride_head, LSE, lse_stride,
            lse2, delta, w.stat_stride, reinterpret_cast<float4*>(dqacc),
            reinterpret_cast<float4*>(zero_acc2 ? accK2 : nullptr), reinterpret_cast<float4*>(zero_acc2 ? accV2 : nullptr),
            total * Hkv * (D / 4), seq);
        PF_CUDA(ctx, cudaGetLastError());
        ctx->n_launches += 1;
    }
    pf::BwdParams p;
    p.dQacc = dqacc;
    p.lse2 = lse2; p.delta = delta; p.stat_stride = w.stat_stride;
    p.pre = Lp > 0 ? g->pre : whole_prefix(0);
    p.Hq = Hq; p.Hkv = Hkv; p.G = G;
    p.nPT = p.pre.n > 0 ? p.pre.tile0[p.pre.n] : 0;
    p.nQS = nQS;
    p.seq = seq;
    // ---- item sizing (SplitModel above); options and deterministic_gkv override the model
    const int pairs = n * G;
    int ppcP = pairs > 0 ? pairs : 1, ppcC = (G + 1) / 2;
    if (ctx->deterministic_gkv) {
        ppcC = G;
    } else {
        SplitEntry key;
        memset(&key, 0, sizeof(key));
        key.n = n; key.nPT = p.nPT; key.Hkv = Hkv; key.G = G; key.interleave = ctx->bwd_interleave;
        for (int i = 0; i <= n; ++i) key.cu[i] = seq.cu[i];
        const SplitEntry* hit = nullptr;
        for (const SplitEntry& e : ctx->split_cache)
            if (memcmp(&e, &key, offsetof(SplitEntry, ppcP)) == 0) { hit = &e; break; }
        if (!hit) {
            key.ppcP = ppcP; key.ppcC = ppcC;
            SplitModel model{seq, n, p.nPT, Hkv, G, ctx->num_sms};
            model.interleave = ctx->bwd_interleave != 0;
            model.choose(key.ppcP, key.ppcC);
            if (ctx->split_cache.size() >= 64) ctx->split_cache.erase(ctx->split_cache.begin());
            ctx->split_cache.push_back(key);
            hit = &ctx->split_cache.back();
        }
        ppcP = hit->ppcP; ppcC = hit->ppcC;
        if (ctx->bwd_pairs_per_item > 0) ppcP = ctx->bwd_pairs_per_item;
        if (ctx->bwd_heads_per_item > 0) ppcC = ctx->bwd_heads_per_item;
    }
    ppcP = ppcP < 1 ? 1 : (ppcP > pairs && pairs > 0 ? pairs : ppcP);
    ppcC = ppcC < 1 ? 1 : (ppcC > G ? G : ppcC);
    ctx->last_ppcP = ppcP; ctx->last_ppcC = ppcC;
    p.ppcP = ppcP; p.chunksP = (pairs + ppcP - 1) / ppcP;
    p.ppcC = ppcC; p.chunksC = (G + ppcC - 1) / ppcC;
    p.nItemsP = p.nPT * Hkv * p.chunksP;
    p.interleave = ctx->bwd_interleave && !ctx->deterministic_gkv;
    p.scale_log2 = g->sigma * 1.4426950408889634f;
    p.sigma = g->sigma;
    const int64_t items = int64_t(p.nItemsP) + int64_t(seq.ckt[n]) * Hkv * p.chunksC;
    if (items > 0) {
        {
            ProfScope prof(ctx, prof_kind, s);
            pf::attn_bwd_kernel<D><<<unsigned(items), pf::BwdCfg<D>::THREADS, pf::BwdCfg<D>::SMEM, s>>>(
                mQ, mdO, mK1, mV1, mK2, mV2, mAK1, mAV1, mAK2, mAV2, p);
        }
        PF_CUDA(ctx, cudaGetLastError());
        ctx->n_launches += 1;
    }
    if (nQS > 0) {
        pf::dq_finish_kernel<D><<<dim3(nQS, Hq), 256, 0, s>>>(
            dqacc, static_cast<__nv_bfloat16*>(dQ.ptr), dQ.stride_tok, dQ.stride_head, g->sigma, seq);
        PF_CUDA(ctx, cudaGetLastError());
        ctx->n_launches += 1;
    }
    return PF_OK;
}

// dK, dV fp32 accumulators -> bf16 outputs, one launch for the pair
template <int D>
pf_status launch_convert_kv2(pf_group* g, const float* accK, const pf_tensor& dK, const float* accV,
                             const pf_tensor& dV, int64_t L, cudaStream_t s) {
    const int Hkv = g->desc.n_kv_heads;
    const int64_t threads = L * Hkv * (D / 8);
    if (threads == 0) return PF_OK;
    pf::acc2_to_bf16_kernel<D><<<dim3(unsigned((threads + 255) / 256), 2), 256, 0, s>>>(
        accK, static_cast<__nv_bfloat16*>(dK.ptr), dK.stride_tok, dK.stride_head, accV,
        static_cast<__nv_bfloat16*>(dV.ptr), dV.stride_tok, dV.stride_head, L, Hkv);
    PF_CUDA(g->ctx, cudaGetLastError());
    g->ctx->n_launches += 1;
    return PF_OK;
}

pf_status check_cu(pf_ctx* ctx, int32_t n_seqs, const int32_t* cu) {
    if (n_seqs < 0) return fail(ctx, PF_INVALID_ARG, "n_seqs < 0");
    if (!cu) return fail(ctx, PF_INVALID_ARG, "cu_seqlens_host is NULL");
    if (cu[0] != 0) return fail(ctx, PF_INVALID_ARG, "cu_seqlens_host[0] must be 0");
    for (int i = 0; i < n_seqs; ++i)
        if (cu[i + 1] < cu[i]) return fail(ctx, PF_INVALID_ARG, "cu_seqlens_host not monotone at %d", i);
    return PF_OK;
}

inline pf_tensor tok_offset(const pf_tensor& t, int64_t tok) {
    pf_tensor r = t;
    r.ptr = static_cast<__nv_bfloat16*>(t.ptr) + tok * t.stride_tok;
    return r;
}

}  // namespace

// =================================================================================================
// C ABI
// =================================================================================================
extern "C" {

int32_t pf_version(void) { return 100; }

pf_status pf_create(pf_ctx** out, int32_t device) {
    if (!out) return PF_INVALID_ARG;
    *out = nullptr;
    pf_ctx* ctx = new (std::nothrow) pf_ctx();
    if (!ctx) return PF_CUDA_ERROR;
    ctx->device = device;
    int prev = -1;
    cudaError_t e = cudaGetDevice(&prev);
    if (e == cudaSuccess) e = cudaSetDevice(device);
    cudaDeviceProp prop;
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, device);
    if (e != cudaSuccess) {
        if (prev >= 0) cudaSetDevice(prev);
        delete ctx;
        return PF_CUDA_ERROR;
    }
    // the caller's current device is restored on every exit path below
    struct Restore { int d; ~Restore() { if (d >= 0) cudaSetDevice(d); } } restore{prev};
    if (prop.major != 10) {  // the kernels are sm_100a only: no fallback path exists
        delete ctx;
        return PF_UNSUPPORTED;
    }
    ctx->num_sms = prop.multiProcessorCount;
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q);
    if (e != cudaSuccess || !fn || q != cudaDriverEntryPointSuccess) {
        delete ctx;
        return PF_CUDA_ERROR;
    }
    ctx->encode = reinterpret_cast<EncodeTiledFn>(fn);
    if (set_attrs<64>() != PF_OK || set_attrs<128>() != PF_OK || !set_gemm_attr<1, 128>() ||
        !set_gemm_attr<1, 256>() || !set_gemm_attr<2, 128>() || !set_gemm_attr<2, 256>()) {
        delete ctx;
        return PF_CUDA_ERROR;
    }
    {   // device address of the built-in scratch: looked up once per device (this context's device is
        // current here), remembered for later contexts on the same device
        static std::mutex mu;
        static void* addr[kMaxDevices] = {nullptr};
        std::lock_guard<std::mutex> lock(mu);
        void* scratch = device >= 0 && device < kMaxDevices ? addr[device] : nullptr;
        if (!scratch) {
            e = cudaGetSymbolAddress(&scratch, pf_static_scratch);
            if (e != cudaSuccess || !scratch) {
                delete ctx;
                return PF_CUDA_ERROR;
            }
            if (device >= 0 && device < kMaxDevices) addr[device] = scratch;
        }
        ctx->static_scratch = static_cast<uint8_t*>(scratch);
    }
    *out = ctx;
    return PF_OK;
}

pf_status pf_destroy(pf_ctx* ctx) {
    if (!ctx) return PF_INVALID_ARG;
    for (auto& r : ctx->prof) {
        cudaEventDestroy(r.a);
        cudaEventDestroy(r.b);
    }
    for (auto e : ctx->ev_pool) cudaEventDestroy(e);
    delete ctx;
    return PF_OK;
}

const char* pf_last_error(const pf_ctx* ctx) { return ctx ? ctx->err : "pf_ctx is NULL"; }

pf_status pf_set_option(pf_ctx* ctx, const char* name, int64_t value) {
    if (!ctx || !name) return PF_INVALID_ARG;
    if (strcmp(name, "bwd_interleave") == 0) {
        ctx->bwd_interleave = value != 0;
        return PF_OK;
    }
    if (strcmp(name, "bwd_pairs_per_item") == 0 || strcmp(name, "bwd_heads_per_item") == 0) {
        if (value < 0 || value > (1 << 20)) return fail(ctx, PF_INVALID_ARG, "%s must be >= 0", name);
        (name[4] == 'p' ? ctx->bwd_pairs_per_item : ctx->bwd_heads_per_item) = int(value);
        return PF_OK;
    }
    if (strcmp(name, "zero_accumulators") == 0) {
        ctx->zero_accumulators = value != 0;
        return PF_OK;
    }
    if (strcmp(name, "deterministic_gkv") == 0) {
        ctx->deterministic_gkv = value != 0;
        return PF_OK;
    }
    if (strcmp(name, "profile") == 0) {
        ctx->profile = value != 0;
        return PF_OK;
    }
    return fail(ctx, PF_INVALID_ARG, "unknown option '%s'", name);
}

int64_t pf_counter(const pf_ctx* ctx, const char* name) {
    if (!ctx || !name) return -1;
    if (strcmp(name, "kernel_launches") == 0) return ctx->n_launches;
    if (strcmp(name, "last_bwd_pairs_per_item") == 0) return ctx->last_ppcP;
    if (strcmp(name, "last_bwd_heads_per_item") == 0) return ctx->last_ppcC;
    if (strcmp(name, "fwd_rescale_rows") == 0) {   // device-side debug counter (synchronises)
        unsigned long long v = 0;
        if (cudaMemcpyFromSymbol(&v, pf::g_fwd_rescale_rows, sizeof(v)) != cudaSuccess) return -1;
        return int64_t(v);
    }
    return -1;
}

pf_status pf_bwd_split_model(const pf_desc* desc, int64_t Lp, int32_t n_seqs, const int32_t* cu_seqlens_host,
                             int32_t n_sms, int32_t* pairs_per_item, int32_t* heads_per_item) {
    if (!desc || !cu_seqlens_host || !pairs_per_item || !heads_per_item) return PF_INVALID_ARG;
    if (desc->n_q_heads <= 0 || desc->n_kv_heads <= 0 || desc->n_q_heads % desc->n_kv_heads != 0 ||
        n_seqs < 0 || n_seqs > pf::kMaxSeqs || n_sms <= 0 || Lp < 0 || cu_seqlens_host[0] != 0)
        return PF_INVALID_ARG;
    int64_t cu[pf::kMaxSeqs + 1];
    for (int i = 0; i <= n_seqs; ++i) {
        if (i > 0 && cu_seqlens_host[i] < cu_seqlens_host[i - 1]) return PF_INVALID_ARG;
        cu[i] = cu_seqlens_host[i];
    }
    const pf::SeqTable seq = make_seq_table(n_seqs, cu);
    const int G = desc->n_q_heads / desc->n_kv_heads;
    int a = n_seqs * G > 0 ? n_seqs * G : 1, b = (G + 1) / 2;
    SplitModel model{seq, n_seqs, int((Lp + 127) / 128), desc->n_kv_heads, G, n_sms};
    model.interleave = true;   // the default launch order ("bwd_interleave" = 1)
    model.choose(a, b);
    *pairs_per_item = a;
    *heads_per_item = b;
    return PF_OK;
}

pf_status pf_profile_read(pf_ctx* ctx, int32_t kind, int64_t* launches, double* total_ms) {
    if (!ctx) return PF_INVALID_ARG;
    if (!launches || !total_ms) return fail(ctx, PF_INVALID_ARG, "pf_profile_read: NULL output");
    int64_t n = 0;
    double ms = 0.0;
    // first pass reads (no state is changed if a CUDA call fails), second pass recycles
    for (auto& r : ctx->prof) {
        if (r.kind != kind) continue;
        PF_CUDA(ctx, cudaEventSynchronize(r.b));
        float t = 0.f;
        PF_CUDA(ctx, cudaEventElapsedTime(&t, r.a, r.b));
        ms += t;
        n += 1;
    }
    std::vector<ProfRec> keep;
    for (auto& r : ctx->prof) {
        if (r.kind != kind) {
            keep.push_back(r);
            continue;
        }
        ctx->ev_pool.push_back(r.a);
        ctx->ev_pool.push_back(r.b);
    }
    ctx->prof.swap(keep);
    *launches = n;
    *total_ms = ms;
    return PF_OK;
}

size_t pf_workspace_bytes(const pf_desc* desc, int64_t Lp, int64_t max_Ls) {
    if (!desc || Lp < 0 || max_Ls < 0 || desc->n_q_heads <= 0 || desc->n_kv_heads <= 0 ||
        desc->head_dim <= 0)
        return 0;
    // every sequence of a packed wave is padded to a multiple of 64 rows: room for 16 ragged tails
    const int64_t Lmax = Lp > max_Ls ? Lp : max_Ls;
    const int64_t cap = align_up(Lmax, 64) + 64 * 16;
    return size_t(cap * ws_bytes_per_pos(*desc)) + size_t(8 * kAlign);
}

pf_status pf_group_begin(pf_ctx* ctx, const pf_desc* desc, int64_t Lp, pf_tensor K1, pf_tensor V1,
                         pf_tensor gK1, pf_tensor gV1, void* workspace, size_t workspace_bytes,
                         void* stream, pf_group** out) {
    if (!ctx) return PF_INVALID_ARG;
    if (!out) return fail(ctx, PF_INVALID_ARG, "out is NULL");
    *out = nullptr;
    pf_status st;
    if ((st = check_device(ctx))) return st;
    if ((st = check_desc(ctx, desc))) return st;
    if (Lp < 0 || Lp > (int64_t(1) << 30)) return fail(ctx, PF_INVALID_ARG, "Lp=%lld out of range", (long long)Lp);
    const int Hkv = desc->n_kv_heads, d = desc->head_dim;
    if ((st = check_tensor(ctx, "K1", K1, Lp, Hkv, d))) return st;
    if ((st = check_tensor(ctx, "V1", V1, Lp, Hkv, d))) return st;
    if ((gK1.ptr == nullptr) != (gV1.ptr == nullptr))
        return fail(ctx, PF_INVALID_ARG, "gK1 and gV1 must both be given or both be NULL");
    if (gK1.ptr) {
        const pf_tensor* acc[2] = {&gK1, &gV1};
        for (int i = 0; i < 2; ++i) {
            if (reinterpret_cast<uintptr_t>(acc[i]->ptr) % 16 != 0)
                return fail(ctx, PF_INVALID_ARG, "gK1/gV1 must be 16-byte aligned");
            if (Lp > 0 && (acc[i]->stride_head != d || acc[i]->stride_tok != int64_t(Hkv) * d))
                return fail(ctx, PF_UNSUPPORTED, "gK1/gV1 must be contiguous [Lp,Hkv,d] fp32");
        }
    }
    if (!workspace || reinterpret_cast<uintptr_t>(workspace) % kAlign != 0)
        return fail(ctx, PF_WORKSPACE, "workspace is NULL or not 256-byte aligned");
    // the capacity each call needs (Phase C: Lp rows; Phase B / segment: the wave's rows) is checked
    // by that call; here only a workspace that could not serve any call is refused
    if (workspace_bytes < pf_workspace_bytes(desc, 0, 0))
        return fail(ctx, PF_WORKSPACE, "workspace of %zu bytes < the minimum pf_workspace_bytes(desc, 0, 0) = %zu",
                    workspace_bytes, pf_workspace_bytes(desc, 0, 0));
    pf_group* g = new (std::nothrow) pf_group();
    if (!g) return fail(ctx, PF_CUDA_ERROR, "out of host memory");
    g->ctx = ctx;
    g->desc = *desc;
    g->sigma = desc->softmax_scale > 0.f ? desc->softmax_scale : 1.0f / sqrtf(float(d));
    g->Lp = Lp;
    g->K1 = K1;
    g->V1 = V1;
    g->gK1 = static_cast<float*>(gK1.ptr);
    g->gV1 = static_cast<float*>(gV1.ptr);
    g->ws = static_cast<uint8_t*>(workspace);
    g->ws_bytes = workspace_bytes;
    g->ws_cap = ws_capacity(*desc, workspace_bytes);
    g->pre = whole_prefix(Lp);
    g->state = 0;
    if (Lp > 0) {
        pf_status ms;
        if ((ms = make_map(ctx, &g->kv128.k, "K1", K1, Lp, Hkv, d, 128)) || (ms = make_map(ctx, &g->kv128.v, "V1", V1, Lp, Hkv, d, 128)) ||
            (ms = make_acc_map(ctx, &g->acc.k, "gK1", g->gK1, Lp, Hkv, d)) || (ms = make_acc_map(ctx, &g->acc.v, "gV1", g->gV1, Lp, Hkv, d))) {
            delete g;
            return ms;
        }
    }
    if (g->gK1 && Lp > 0 && ctx->zero_accumulators) {
        cudaStream_t s = static_cast<cudaStream_t>(stream);
        const size_t bytes = size_t(Lp) * Hkv * d * 4;
        cudaError_t e = cudaMemsetAsync(g->gK1, 0, bytes, s);
        if (e == cudaSuccess) e = cudaMemsetAsync(g->gV1, 0, bytes, s);
        if (e != cudaSuccess) {
            delete g;
            return fail(ctx, PF_CUDA_ERROR, "cudaMemsetAsync(gK1/gV1) failed: %s", cudaGetErrorString(e));
        }
    }
    *out = g;
    return PF_OK;
}

pf_status pf_group_end(pf_group* grp) {
    if (!grp) return PF_INVALID_ARG;
    delete grp;
    return PF_OK;
}

pf_status pf_phaseA_fwd(pf_group* grp, pf_tensor Q1, pf_tensor O1, float* LSE1, void* stream) {
    if (!grp) return PF_INVALID_ARG;
    pf_ctx* ctx = grp->ctx;
    if (grp->state != 0) return fail(ctx, PF_STATE, "pf_phaseA_fwd: Phase A already ran for this group");
    const int Hq = grp->desc.n_q_heads, d = grp->desc.head_dim;
    const int64_t Lp = grp->Lp;
    pf_status st;
    if ((st = check_device(ctx))) return st;
    if ((st = check_tensor(ctx, "Q1", Q1, Lp, Hq, d))) return st;
    if ((st = check_tensor(ctx, "O1", O1, Lp, Hq, d))) return st;
    if (Lp > 0 && !LSE1) return fail(ctx, PF_INVALID_ARG, "LSE1 is NULL");
    if (Lp > 0) {
        cudaStream_t s = static_cast<cudaStream_t>(stream);
        const int64_t cu[2] = {0, Lp};
        st = d == 64 ? launch_fwd<64>(grp, Q1, nullptr, 0, &grp->kv128, grp->K1, grp->V1, O1, LSE1, Lp, 1, cu, 0, s)
                     : launch_fwd<128>(grp, Q1, nullptr, 0, &grp->kv128, grp->K1, grp->V1, O1, LSE1, Lp, 1, cu, 0, s);
        if (st) return st;
    }
    grp->state = 1;
    return PF_OK;
}

pf_status pf_phaseB_fwd(pf_group* grp, int32_t n_seqs, const int32_t* cu_seqlens_host,
                        pf_tensor Q2, pf_tensor K2, pf_tensor V2, pf_tensor O2, float* LSE2,
                        void* stream) {
    if (!grp) return PF_INVALID_ARG;
    pf_ctx* ctx = grp->ctx;
    if (grp->state != 1) return fail(ctx, PF_STATE, "pf_phaseB_fwd needs Phase A done and Phase C not yet run");
    pf_status st;
    if ((st = check_device(ctx))) return st;
    if ((st = check_cu(ctx, n_seqs, cu_seqlens_host))) return st;
    const int Hq = grp->desc.n_q_heads, Hkv = grp->desc.n_kv_heads, d = grp->desc.head_dim;
    const int64_t total = cu_seqlens_host[n_seqs];
    if ((st = check_tensor(ctx, "Q2", Q2, total, Hq, d))) return st;
    if ((st = check_tensor(ctx, "K2", K2, total, Hkv, d))) return st;
    if ((st = check_tensor(ctx, "V2", V2, total, Hkv, d))) return st;
    if ((st = check_tensor(ctx, "O2", O2, total, Hq, d))) return st;
    if (total > 0 && !LSE2) return fail(ctx, PF_INVALID_ARG, "LSE2 is NULL");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int i = 0;
    while (i < n_seqs) {   // launches of <= kMaxSeqs non-empty sequences
        int64_t cu[pf::kMaxSeqs + 1];
        int n = 0;
        int64_t t0 = 0;
        for (; i < n_seqs && n < pf::kMaxSeqs; ++i) {
            const int64_t b = cu_seqlens_host[i], Ls = cu_seqlens_host[i + 1] - b;
            if (Ls == 0) continue;
            if (n == 0) { t0 = b; cu[0] = 0; }
            cu[++n] = b + Ls - t0;
        }
        if (n == 0) break;
        const pf_tensor q = tok_offset(Q2, t0), k = tok_offset(K2, t0), v = tok_offset(V2, t0),
                        o = tok_offset(O2, t0);
        st = d == 64 ? launch_fwd<64>(grp, q, &grp->kv128, grp->Lp, nullptr, k, v, o, LSE2 + t0, total, n, cu, 1, s)
                     : launch_fwd<128>(grp, q, &grp->kv128, grp->Lp, nullptr, k, v, o, LSE2 + t0, total, n, cu, 1, s);
        if (st) return st;
    }
    return PF_OK;
}

pf_status pf_phaseB_bwd(pf_group* grp, int32_t n_seqs, const int32_t* cu_seqlens_host,
                        pf_tensor Q2, pf_tensor K2, pf_tensor V2, pf_tensor O2, const float* LSE2,
                        pf_tensor dO2, pf_tensor dQ2, pf_tensor dK2, pf_tensor dV2, void* stream) {
    if (!grp) return PF_INVALID_ARG;
    pf_ctx* ctx = grp->ctx;
    if (grp->state != 1) return fail(ctx, PF_STATE, "pf_phaseB_bwd needs Phase A done and Phase C not yet run");
    if (!grp->gK1 && grp->Lp > 0)
        return fail(ctx, PF_STATE, "pf_phaseB_bwd: the group was opened without gK1/gV1");
    pf_status st;
    if ((st = check_device(ctx))) return st;
    if ((st = check_cu(ctx, n_seqs, cu_seqlens_host))) return st;
    const int Hq = grp->desc.n_q_heads, Hkv = grp->desc.n_kv_heads, d = grp->desc.head_dim;
    const int64_t total = cu_seqlens_host[n_seqs];
    if ((st = check_tensor(ctx, "Q2", Q2, total, Hq, d))) return st;
    if ((st = check_tensor(ctx, "K2", K2, total, Hkv, d))) return st;
    if ((st = check_tensor(ctx, "V2", V2, total, Hkv, d))) return st;
    if ((st = check_tensor(ctx, "O2", O2, total, Hq, d))) return st;
    if ((st = check_tensor(ctx, "dO2", dO2, total, Hq, d))) return st;
    if ((st = check_tensor(ctx, "dQ2", dQ2, total, Hq, d))) return st;
    if ((st = check_tensor(ctx, "dK2", dK2, total, Hkv, d))) return st;
    if ((st = check_tensor(ctx, "dV2", dV2, total, Hkv, d))) return st;
    if (total > 0 && !LSE2) return fail(ctx, PF_INVALID_ARG, "LSE2 is NULL");
    // every suffix must fit the workspace on its own (a wave is cut between suffixes, never inside
    // one): checked for the whole call BEFORE anything is enqueued, so that a PF_WORKSPACE return
    // leaves gK1/gV1 and the outputs untouched
    for (int i = 0; i < n_seqs; ++i) {
        const int64_t Ls = int64_t(cu_seqlens_host[i + 1]) - cu_seqlens_host[i];
        if (align_up(Ls, 64) > grp->ws_cap)
            return fail(ctx, PF_WORKSPACE, "workspace too small for suffix %d of %lld tokens (capacity %lld padded positions)",
                        i, (long long)Ls, (long long)grp->ws_cap);
    }
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const WsLayout w = ws_layout(grp->desc, grp->ws_cap);
    float* ak = reinterpret_cast<float*>(grp->ws + w.off_ak);
    float* av = reinterpret_cast<float*>(grp->ws + w.off_av);
    // the wave is cut into launches of <= kMaxSeqs non-empty sequences that fit the workspace
    int i = 0;
    while (i < n_seqs) {
        int64_t cu[pf::kMaxSeqs + 1];
        int n = 0;
        int64_t t0 = 0, npad = 0;
        for (; i < n_seqs && n < pf::kMaxSeqs; ++i) {
            const int64_t b = cu_seqlens_host[i], Ls = cu_seqlens_host[i + 1] - b;
            if (Ls == 0) continue;
            const int64_t pad = align_up(Ls, 64);
            if (n > 0 && npad + pad > grp->ws_cap) break;
            if (n == 0) { t0 = b; cu[0] = 0; }
            npad += pad;
            cu[++n] = b + Ls - t0;
        }
        if (n == 0) break;
        if (npad > grp->ws_cap)
            return fail(ctx, PF_WORKSPACE, "workspace too small for a suffix of %lld tokens", (long long)cu[1]);
        const int64_t tot = cu[n];
        const pf_tensor q = tok_offset(Q2, t0), k = tok_offset(K2, t0), v = tok_offset(V2, t0),
                        o = tok_offset(O2, t0), dout = tok_offset(dO2, t0), dq = tok_offset(dQ2, t0);
        if (d == 64) {
            st = launch_bwd<64>(grp, q, &grp->kv128, &grp->acc, grp->Lp, nullptr, nullptr, k, v, o,
                                LSE2 + t0, total, dout, ak, av, dq, n, cu, 2, true, s);
            if (!st) st = launch_convert_kv2<64>(grp, ak, tok_offset(dK2, t0), av, tok_offset(dV2, t0), tot, s);
        } else {
            st = launch_bwd<128>(grp, q, &grp->kv128, &grp->acc, grp->Lp, nullptr, nullptr, k, v, o,
                                 LSE2 + t0, total, dout, ak, av, dq, n, cu, 2, true, s);
            if (!st) st = launch_convert_kv2<128>(grp, ak, tok_offset(dK2, t0), av, tok_offset(dV2, t0), tot, s);
        }
        if (st) return st;
    }
    return PF_OK;
}

pf_status pf_group_set_prefix_ranges(pf_group* grp, int32_t n_ranges, const int64_t* starts_host,
                                     const int64_t* lens_host) {
    if (!grp) return PF_INVALID_ARG;
    pf_ctx* ctx = grp->ctx;
    if (n_ranges < 0 || n_ranges > pf::kMaxRanges)
        return fail(ctx, PF_UNSUPPORTED, "n_ranges=%d not in [0, %d]", n_ranges, pf::kMaxRanges);
    if (n_ranges > 0 && (!starts_host || !lens_host)) return fail(ctx, PF_INVALID_ARG, "ranges are NULL");
    pf::PrefixRanges r;
    memset(&r, 0, sizeof(r));
    int64_t end = 0;
    for (int i = 0; i < n_ranges; ++i) {
        if (lens_host[i] <= 0) continue;   // empty ranges are dropped
        if (starts_host[i] < end || starts_host[i] + lens_host[i] > grp->Lp)
            return fail(ctx, PF_INVALID_ARG, "prefix range %d = [%lld, +%lld) is out of [0, Lp) or not ascending",
                        i, (long long)starts_host[i], (long long)lens_host[i]);
        r.start[r.n] = int(starts_host[i]);
        r.len[r.n] = int(lens_host[i]);
        r.tile0[r.n + 1] = r.tile0[r.n] + int((lens_host[i] + 127) / 128);
        end = starts_host[i] + lens_host[i];
        ++r.n;
    }
    grp->pre = r;
    return PF_OK;
}

pf_status pf_group_mark_cached(pf_group* grp) {
    if (!grp) return PF_INVALID_ARG;
    if (grp->state != 0) return fail(grp->ctx, PF_STATE, "pf_group_mark_cached: the group already left its initial state");
    grp->state = 1;
    return PF_OK;
}

pf_status pf_segment_bwd(pf_group* grp, int64_t Ls, pf_tensor Q, pf_tensor K, pf_tensor V, pf_tensor O,
                         const float* LSE, pf_tensor dO, pf_tensor dQ, float* accK, float* accV,
                         pf_tensor dK, pf_tensor dV, void* stream) {
    if (!grp) return PF_INVALID_ARG;
    pf_ctx* ctx = grp->ctx;
    if (grp->state != 1) return fail(ctx, PF_STATE, "pf_segment_bwd needs the cache marked valid (Phase A or pf_group_mark_cached)");
    if (!grp->gK1 && grp->Lp > 0) return fail(ctx, PF_STATE, "pf_segment_bwd: the group was opened without gK1/gV1");
    if (Ls < 0) return fail(ctx, PF_INVALID_ARG, "Ls < 0");
    if (Ls == 0) return PF_OK;
    const int Hq = grp->desc.n_q_heads, Hkv = grp->desc.n_kv_heads, d = grp->desc.head_dim;
    pf_status st;
    if ((st = check_device(ctx))) return st;
    if ((st = check_tensor(ctx, "Q", Q, Ls, Hq, d))) return st;
    if ((st = check_tensor(ctx, "K", K, Ls, Hkv, d))) return st;
    if ((st = check_tensor(ctx, "V", V, Ls, Hkv, d))) return st;
    if ((st = check_tensor(ctx, "O", O, Ls, Hq, d))) return st;
    if ((st = check_tensor(ctx, "dO", dO, Ls, Hq, d))) return st;
    if ((st = check_tensor(ctx, "dQ", dQ, Ls, Hq, d))) return st;
    if ((st = check_tensor(ctx, "dK", dK, Ls, Hkv, d))) return st;
    if ((st = check_tensor(ctx, "dV", dV, Ls, Hkv, d))) return st;
    if (!LSE || !accK || !accV) return fail(ctx, PF_INVALID_ARG, "LSE / accK / accV is NULL");
    if (reinterpret_cast<uintptr_t>(accK) % 16 != 0 || reinterpret_cast<uintptr_t>(accV) % 16 != 0)
        return fail(ctx, PF_INVALID_ARG, "accK/accV must be 16-byte aligned");
    if (align_up(Ls, 64) > grp->ws_cap)
        return fail(ctx, PF_WORKSPACE, "workspace too small for a segment of %lld tokens", (long long)Ls);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int64_t cu[2] = {0, Ls};
    if (d == 64) {
        st = launch_bwd<64>(grp, Q, &grp->kv128, &grp->acc, grp->Lp, nullptr, nullptr, K, V, O, LSE, Ls,
                            dO, accK, accV, dQ, 1, cu, 2, false, s);
        if (!st) st = launch_convert_kv2<64>(grp, accK, dK, accV, dV, Ls, s);
    } else {
        st = launch_bwd<128>(grp, Q, &grp->kv128, &grp->acc, grp->Lp, nullptr, nullptr, K, V, O, LSE, Ls,
                             dO, accK, accV, dQ, 1, cu, 2, false, s);
        if (!st) st = launch_convert_kv2<128>(grp, accK, dK, accV, dV, Ls, s);
    }
    return st;
}

pf_status pf_phaseC_bwd(pf_group* grp, pf_tensor Q1, pf_tensor O1, const float* LSE1,
                        pf_tensor dO1, pf_tensor dQ1, pf_tensor dK1, pf_tensor dV1, void* stream) {
    if (!grp) return PF_INVALID_ARG;
    pf_ctx* ctx = grp->ctx;
    if (grp->state != 1) return fail(ctx, PF_STATE, "pf_phaseC_bwd needs Phase A done and runs once");
    const int Hq = grp->desc.n_q_heads, Hkv = grp->desc.n_kv_heads, d = grp->desc.head_dim;
    const int64_t Lp = grp->Lp;
    pf_status st;
    if ((st = check_device(ctx))) return st;
    if ((st = check_tensor(ctx, "Q1", Q1, Lp, Hq, d))) return st;
    if ((st = check_tensor(ctx, "O1", O1, Lp, Hq, d))) return st;
    if ((st = check_tensor(ctx, "dO1", dO1, Lp, Hq, d))) return st;
    if ((st = check_tensor(ctx, "dQ1", dQ1, Lp, Hq, d))) return st;
    if ((st = check_tensor(ctx, "dK1", dK1, Lp, Hkv, d))) return st;
    if ((st = check_tensor(ctx, "dV1", dV1, Lp, Hkv, d))) return st;
    if (Lp > 0 && !LSE1) return fail(ctx, PF_INVALID_ARG, "LSE1 is NULL");
    if (Lp > 0) {
        cudaStream_t s = static_cast<cudaStream_t>(stream);
        float* ak = grp->gK1;
        float* av = grp->gV1;
        if (!ak) {  // replay baseline: no injection, accumulate in the workspace
            const WsLayout w = ws_layout(grp->desc, grp->ws_cap);
            if (align_up(Lp, 64) > grp->ws_cap) return fail(ctx, PF_WORKSPACE, "workspace too small");
            ak = reinterpret_cast<float*>(grp->ws + w.off_ak);
            av = reinterpret_cast<float*>(grp->ws + w.off_av);
        }
        const int64_t cu[2] = {0, Lp};
        const KvMaps* cacc = grp->gK1 ? &grp->acc : nullptr;   // replay: workspace accumulators, encoded per call
        if (d == 64) {
            st = launch_bwd<64>(grp, Q1, nullptr, nullptr, 0, &grp->kv128, cacc, grp->K1, grp->V1, O1, LSE1,
                                Lp, dO1, ak, av, dQ1, 1, cu, 3, !grp->gK1, s);
            if (!st) st = launch_convert_kv2<64>(grp, ak, dK1, av, dV1, Lp, s);
        } else {
            st = launch_bwd<128>(grp, Q1, nullptr, nullptr, 0, &grp->kv128, cacc, grp->K1, grp->V1, O1, LSE1,
                                 Lp, dO1, ak, av, dQ1, 1, cu, 3, !grp->gK1, s);
            if (!st) st = launch_convert_kv2<128>(grp, ak, dK1, av, dV1, Lp, s);
        }
        if (st) return st;
    }
    grp->state = 2;
    return PF_OK;
}

pf_status pf_rope(pf_ctx* ctx, int32_t n_seqs, const int32_t* cu_seqlens_host, int64_t pos0,
                  pf_tensor X, int32_t n_heads, int32_t head_dim, float theta_base, int32_t inverse,
                  void* stream) {
    if (!ctx) return PF_INVALID_ARG;
    pf_status st;
    if ((st = check_device(ctx))) return st;
    if ((st = check_cu(ctx, n_seqs, cu_seqlens_host))) return st;
    if (n_heads <= 0 || n_heads > 65535) return fail(ctx, PF_INVALID_ARG, "pf_rope: n_heads=%d", n_heads);
    if (head_dim < 16 || head_dim > 2 * pf::kRopeMaxHalf || head_dim % 16 != 0)
        return fail(ctx, PF_UNSUPPORTED, "pf_rope: head_dim=%d must be a multiple of 16 in [16, %d]", head_dim,
                    2 * pf::kRopeMaxHalf);
    if (pos0 < 0 || pos0 > (int64_t(1) << 40)) return fail(ctx, PF_INVALID_ARG, "pf_rope: pos0 out of range");
    if (!(theta_base > 1.f) || std::isinf(theta_base))
        return fail(ctx, PF_INVALID_ARG, "pf_rope: theta_base must be finite and > 1");
    const int64_t total = cu_seqlens_host[n_seqs];
    if ((st = check_tensor(ctx, "X", X, total, n_heads, head_dim))) return st;
    if (total == 0) return PF_OK;
    pf::RopeFreq fr;
    memset(&fr, 0, sizeof(fr));
    for (int j = 0; j < head_dim / 2; ++j) fr.inv[j] = std::pow(double(theta_base), -2.0 * j / head_dim);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int i = 0;
    while (i < n_seqs) {   // launches of <= kMaxSeqs non-empty sequences
        int64_t cu[pf::kMaxSeqs + 1];
        int n = 0;
        int64_t t0 = 0;
        for (; i < n_seqs && n < pf::kMaxSeqs; ++i) {
            const int64_t b = cu_seqlens_host[i], Ls = cu_seqlens_host[i + 1] - b;
            if (Ls == 0) continue;
            if (n == 0) { t0 = b; cu[0] = 0; }
            cu[++n] = b + Ls - t0;
        }
        if (n == 0) break;
        const pf_tensor x = tok_offset(X, t0);
        pf::rope_kernel<<<unsigned(cu[n]), 128, 0, s>>>(static_cast<__nv_bfloat16*>(x.ptr), x.stride_tok,
                                                        x.stride_head, n_heads, head_dim, pos0, inverse != 0,
                                                        make_seq_table(n, cu), fr);
        PF_CUDA(ctx, cudaGetLastError());
        ctx->n_launches += 1;
    }
    return PF_OK;
}

pf_status pf_kv_proj_grad(pf_ctx* ctx, int64_t L, int32_t d_model, int32_t n_cols, const void* X,
                          int64_t ldx, const void* dY, int64_t ldy, float* dW, void* stream) {
    if (!ctx) return PF_INVALID_ARG;
    pf_status st;
    if ((st = check_device(ctx))) return st;
    if (L < 0 || L > (int64_t(1) << 30)) return fail(ctx, PF_INVALID_ARG, "pf_kv_proj_grad: L out of range");
    if (d_model <= 0 || n_cols <= 0 || d_model % 128 != 0 || n_cols % 128 != 0)
        return fail(ctx, PF_UNSUPPORTED, "pf_kv_proj_grad: d_model=%d and n_cols=%d must be positive multiples of 128",
                    d_model, n_cols);
    if (L == 0) return PF_OK;
    if (!X || !dY || !dW) return fail(ctx, PF_INVALID_ARG, "pf_kv_proj_grad: NULL pointer");
    if (reinterpret_cast<uintptr_t>(X) % 16 || reinterpret_cast<uintptr_t>(dY) % 16 || reinterpret_cast<uintptr_t>(dW) % 16)
        return fail(ctx, PF_INVALID_ARG, "pf_kv_proj_grad: X, dY and dW must be 16-byte aligned");
    if (ldx < d_model || ldy < n_cols || ldx % 8 != 0 || ldy % 8 != 0)
        return fail(ctx, PF_INVALID_ARG, "pf_kv_proj_grad: ldx=%lld / ldy=%lld must be >= the row length and multiples of 8",
                    (long long)ldx, (long long)ldy);
    CUtensorMap mX, mY;
    const void* ptr[2] = {X, dY};
    const int64_t ld[2] = {ldx, ldy};
    const int cols[2] = {d_model, n_cols};
    CUtensorMap* maps[2] = {&mX, &mY};
    for (int i = 0; i < 2; ++i) {   // 2-D map {features, tokens}, box {64, 64}, swizzle-128B; tokens past L read as 0
        cuuint64_t dims[2] = {cuuint64_t(cols[i]), cuuint64_t(L)};
        cuuint64_t strides[1] = {cuuint64_t(ld[i]) * 2};
        cuuint32_t box[2] = {64, 64};
        cuuint32_t es[2] = {1, 1};
        CUresult r = ctx->encode(maps[i], CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(ptr[i]), dims, strides,
                                 box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                 CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS)
            return fail(ctx, PF_CUDA_ERROR, "cuTensorMapEncodeTiled(%s) failed with CUresult %d", i ? "dY" : "X", int(r));
    }
    // the largest tile the shape divides into (256 x 256 halves the L2 -> shared-memory bytes per flop
    // of 128 x 128); the token range is split so that one round of CTAs about fills the SMs
    const int mh = d_model % 256 == 0 ? 2 : 1, bn = n_cols % 256 == 0 ? 256 : 128;
    const int tiles = (d_model / (128 * mh)) * (n_cols / bn);
    const int n_chunks = int((L + 63) / 64);
    int splits = ctx->num_sms / tiles;
    splits = splits < 1 ? 1 : (splits > n_chunks ? n_chunks : splits);
    const int cps = (n_chunks + splits - 1) / splits;
    splits = (n_chunks + cps - 1) / cps;                           // no empty split
    const dim3 grid(d_model / (128 * mh), n_cols / bn, splits);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (mh == 2 && bn == 256) launch_gemm<2, 256>(grid, s, mX, mY, dW, n_cols, n_chunks, cps);
    else if (mh == 2) launch_gemm<2, 128>(grid, s, mX, mY, dW, n_cols, n_chunks, cps);
    else if (bn == 256) launch_gemm<1, 256>(grid, s, mX, mY, dW, n_cols, n_chunks, cps);
    else launch_gemm<1, 128>(grid, s, mX, mY, dW, n_cols, n_chunks, cps);
    PF_CUDA(ctx, cudaGetLastError());
    ctx->n_launches += 1;
    return PF_OK;
}

pf_status pf_offload(pf_ctx* ctx, const void* src_dev, void* dst_pinned_host, size_t bytes,
                     void* side_stream) {
    if (!ctx) return PF_INVALID_ARG;
    if (bytes == 0) return PF_OK;
    if (!src_dev || !dst_pinned_host) return fail(ctx, PF_INVALID_ARG, "pf_offload: NULL pointer");
    PF_CUDA(ctx, cudaMemcpyAsync(dst_pinned_host, src_dev, bytes, cudaMemcpyDeviceToHost,
                                 static_cast<cudaStream_t>(side_stream)));
    return PF_OK;
}

pf_status pf_prefetch(pf_ctx* ctx, const void* src_pinned_host, void* dst_dev, size_t bytes,
                      void* side_stream) {
    if (!ctx) return PF_INVALID_ARG;
    if (bytes == 0) return PF_OK;
    if (!src_pinned_host || !dst_dev) return fail(ctx, PF_INVALID_ARG, "pf_prefetch: NULL pointer");
    PF_CUDA(ctx, cudaMemcpyAsync(dst_dev, src_pinned_host, bytes, cudaMemcpyHostToDevice,
                                 static_cast<cudaStream_t>(side_stream)));
    return PF_OK;
}

size_t pf_static_scratch_bytes(void) { return kStaticScratchBytes; }

int64_t pf_causal_bwd_static_max_tokens(const pf_desc* desc) {
    if (!desc || desc->n_q_heads <= 0 || desc->n_kv_heads <= 0 || desc->head_dim <= 0) return 0;
    return ws_capacity(*desc, kStaticScratchBytes);
}

pf_status pf_causal_bwd_static(pf_ctx* ctx, const pf_desc* desc, int64_t L, pf_tensor Q, pf_tensor K,
                               pf_tensor V, pf_tensor O, const float* LSE, pf_tensor dO, pf_tensor dQ,
                               pf_tensor dK, pf_tensor dV, void* stream) {
    if (!ctx) return PF_INVALID_ARG;
    pf_status st;
    if ((st = check_device(ctx))) return st;
    if ((st = check_desc(ctx, desc))) return st;
    if (L < 0) return fail(ctx, PF_INVALID_ARG, "pf_causal_bwd_static: L < 0");
    if (L == 0) return PF_OK;
    if (ctx->profile)   // the profiling bracket creates events: not an allocation-free call
        return fail(ctx, PF_STATE, "pf_causal_bwd_static: switch the \"profile\" option off (it creates CUDA events)");
    if (!ctx->static_scratch) return fail(ctx, PF_STATE, "pf_causal_bwd_static: the built-in scratch has no device address");
    const int64_t cap = ws_capacity(*desc, kStaticScratchBytes);
    if (align_up(L, 64) > cap)
        return fail(ctx, PF_WORKSPACE,
                    "pf_causal_bwd_static: L=%lld exceeds the %lld tokens the built-in %zu-byte scratch holds for "
                    "%d/%d heads of dim %d; use pf_group_begin with a workspace of your own",
                    (long long)L, (long long)cap, kStaticScratchBytes, desc->n_q_heads, desc->n_kv_heads, desc->head_dim);
    const int Hkv = desc->n_kv_heads, d = desc->head_dim;
    if ((st = check_tensor(ctx, "K", K, L, Hkv, d))) return st;
    if ((st = check_tensor(ctx, "V", V, L, Hkv, d))) return st;
    // a group on the stack in the state pf_phaseC_bwd expects for the replay baseline (no gK1/gV1
    // injection, dK/dV accumulated in the workspace): the workspace is the built-in scratch
    pf_group g{};
    g.ctx = ctx;
    g.desc = *desc;
    g.sigma = desc->softmax_scale > 0.f ? desc->softmax_scale : 1.0f / sqrtf(float(d));
    g.Lp = L;
    g.K1 = K;
    g.V1 = V;
    g.gK1 = nullptr;
    g.gV1 = nullptr;
    g.ws = ctx->static_scratch;
    g.ws_bytes = kStaticScratchBytes;
    g.ws_cap = cap;
    g.pre = whole_prefix(L);
    g.state = 1;
    if ((st = make_map(ctx, &g.kv128.k, "K", K, L, Hkv, d, 128))) return st;
    if ((st = make_map(ctx, &g.kv128.v, "V", V, L, Hkv, d, 128))) return st;
    return pf_phaseC_bwd(&g, Q, O, LSE, dO, dQ, dK, dV, stream);
}

}  // extern "C"
