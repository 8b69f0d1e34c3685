/* prefixflow.h -- C ABI of the B200-native attention hot path of PrefixFlow's training-time KV
 * cache (arxiv/paper_2606_01143).  Citations are PAPER.md:<line> of the paper text.
 *
 * A GRPO rollout group is N trajectories [P || S(1)] ... [P || S(N)] that share one prefix P of
 * Lp tokens.  The three-phase schedule runs, per attention
 * layer:
 *   Phase A  one causal forward over P; its K1/V1 become the training-time KV cache  (:152)
 *   Phase B  for every suffix S(i): attention forward and backward whose queries read the cached
 *            K1/V1 plus their own causal K2/V2 (:154-158, eq. :192); the gradients that reach the
 *            prefix,  gV1 = P21^T dO2,  gK1 = sigma dS21^T Q2  (eq. :196), are ACCUMULATED over
 *            the N suffixes (:162, :212)
 *   Phase C  one delayed causal backward over P whose dK1/dV1 = own-prefix term + accumulated
 *            gK1/gV1 (:160, :222)
 * Only K1,V1 (read) and gK1,gV1 (written) cross the prefix/suffix boundary (Property 1, :190-200).
 *
 * Conventions:
 *   - all pointers are DEVICE pointers unless a parameter name ends in _host; the library never
 *     allocates or frees user tensors; every call only enqueues work on `stream`
 *     (a cudaStream_t passed as void*), never synchronises, never allocates device memory;
 *   - activations are bf16, token-major [L, H, d] with d contiguous and explicit token / head
 *     strides in ELEMENTS (pf_tensor); base pointers and strides must be multiples of 8 elements
 *     (16 bytes, a TMA requirement) -> PF_INVALID_ARG otherwise;
 *   - LSE is fp32 [Hq, L] row-major (row stride = L), natural log of the sum of exp of the SCALED
 *     scores; GQA head mapping kappa(h) = h / (Hq/Hkv); causal = key j <= query t (inclusive);
 *   - gK1 / gV1 are fp32, contiguous [Lp, Hkv, d], borrowed for the lifetime of the group;
 *   - head_dim in {64, 128}; softmax_scale 0 means 1/sqrt(head_dim);
 *   - functions return a pf_status; nothing throws or aborts across this boundary; validation
 *     happens before any launch; Ls = 0 and Lp = 0 are legal;
 *   - every element of the tensors a call reads must be FINITE, including rows of K1/V1 that a
 *     prefix-range restriction (pf_group_set_prefix_ranges) hides and rows of a packed wave that
 *     belong to another sequence: masked keys get probability exactly 0 but their values still
 *     pass through the tensor cores (0 x NaN = NaN);
 *   - a context is bound to one CUDA device, which must be the current device of the calling
 *     thread for every call that takes the context or one of its groups (PF_STATE otherwise).
 */
#ifndef PREFIXFLOW_H_
#define PREFIXFLOW_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pf_ctx pf_ctx;     /* opaque: device properties, driver entry points, options */
typedef struct pf_group pf_group; /* opaque: one rollout group's training-time KV cache (:164) */
typedef int32_t pf_status;

enum {
    PF_OK = 0,
    PF_INVALID_ARG = 1, /* NULL / negative size / misaligned pointer or stride / Hq % Hkv != 0 */
    PF_UNSUPPORTED = 2, /* head_dim not in {64,128}, non-contiguous accumulator, ... */
    PF_CUDA_ERROR = 3,  /* a CUDA runtime / driver call failed; see pf_last_error */
    PF_WORKSPACE = 4,   /* workspace NULL, misaligned or smaller than pf_workspace_bytes */
    PF_STATE = 5        /* phase order violated (B or C before A, anything after C / end) */
};

typedef struct {
    int32_t n_q_heads;   /* Hq */
    int32_t n_kv_heads;  /* Hkv, divides Hq */
    int32_t head_dim;    /* d: 64 or 128 */
    float softmax_scale; /* sigma; 0 -> 1/sqrt(d) */
} pf_desc;

typedef struct {
    void* ptr;           /* device pointer, element [0,0,0] */
    int64_t stride_tok;  /* elements between consecutive tokens */
    int64_t stride_head; /* elements between consecutive heads */
} pf_tensor;

int32_t pf_version(void);

/* Create / destroy a context bound to CUDA device `device` (host-side state only; the caller's
 * current device is left as it was). */
pf_status pf_create(pf_ctx** out, int32_t device);
pf_status pf_destroy(pf_ctx* ctx);
/* Message of the last failing call on this context (valid until the next call). */
const char* pf_last_error(const pf_ctx* ctx);
/* Options (host-side, take effect at the next launch):
 *   "bwd_pairs_per_item" : backward work split.  A CTA owns one tile of 128 prefix keys of one KV
 *                      head and this many (sequence, query head) pairs of the wave (0 = heuristic).
 *                      All pairs in one CTA = that key tile's gK1/gV1 rows are added by one CTA
 *                      (no contention); 1 = maximal parallelism, most reduce-add traffic.
 *   "bwd_heads_per_item" : the same for the tiles of a suffix's own (causal) keys: query heads of
 *                      the KV head per CTA (0 = heuristic).
 *   "bwd_interleave"     : launch order of the backward's items.  1 (default) = chunk by chunk: the
 *                      prefix-tile items of a chunk of (sequence, head) pairs are followed by the
 *                      causal-tile items of the sequences that chunk completes, so those items find
 *                      the sequences' Q / dO and dQ^T tiles in L2 (35 % less DRAM traffic at
 *                      configs[1], same time).  0 = all prefix-tile items first, then all causal-tile
 *                      items.  Results are the same up to the order of the fp32 reduce-adds.
 *   "deterministic_gkv"  : 1 = every key tile (prefix and causal) is owned by ONE CTA per launch, which
 *                      sums all its (sequence, query head) pairs in TMEM in a fixed order and adds the
 *                      result once: gK1 / gV1 / dK / dV are then bit-reproducible from run to run (the
 *                      launches of a group are stream-ordered).  Fewer, longer CTAs: slower when the
 *                      launch has few key tiles.  dQ still sums its key tiles in arrival order.
 *                      0 (default) = the heuristic split (several CTAs may add into one key tile; the
 *                      fp32 adds happen at L2 in arrival order, "agreement within datatype
 *                      tolerance rather than bitwise").
 *   "zero_accumulators"  : 1 (default) = pf_group_begin zeroes gK1/gV1; 0 = it leaves them as they
 *                      are (segment-by-segment training, where they already hold the contributions
 *                      of later segments). */
pf_status pf_set_option(pf_ctx* ctx, const char* name, int64_t value);

/*   "profile"        : 1 = bracket every attention kernel launch (not the elementwise helpers)
 *                      with a pair of CUDA events on the launch stream; read with pf_profile_read.
 *                      Used by bench.py for the roofline of the dominant kernel.  0 = off. */

/* Counters; -1 for an unknown name.
 *   "kernel_launches"  : kernels this context has launched so far (host-side bookkeeping).
 *   "fwd_rescale_rows" : process-wide count of (query row, KV tile) events in which the forward kernel
 *                        re-based the running softmax maximum after the row's first tile (the lazy
 *                        rescale of the O accumulator).  Debug evidence for the tests; reading it
 *                        synchronises the device.
 *   "last_bwd_pairs_per_item", "last_bwd_heads_per_item" : the item split the most recent backward
 *                        launch used ((sequence, query head) pairs per prefix-tile CTA, query heads
 *                        per causal-tile CTA): the options of the same names if set, else the split
 *                        with the shortest simulated list-scheduling makespan over the SMs. */
int64_t pf_counter(const pf_ctx* ctx, const char* name);

/* Host-only: the backward item split the model picks for a launch of n_seqs packed sequences
 * (cu_seqlens_host) against a prefix of Lp fully visible keys on a GPU with n_sms SMs -- what
 * "last_bwd_*_per_item" would report after that launch with no option set.  No CUDA call is made. */
pf_status pf_bwd_split_model(const pf_desc* desc, int64_t Lp, int32_t n_seqs, const int32_t* cu_seqlens_host,
                             int32_t n_sms, int32_t* pairs_per_item, int32_t* heads_per_item);

/* Profiling read-out (needs option "profile" = 1).  kind: the call that launched the attention
 * kernel -- 0 = pf_phaseA_fwd, 1 = pf_phaseB_fwd, 2 = pf_phaseB_bwd, 3 = pf_phaseC_bwd (forward
 * kernel for 0/1, backward kernel for 2/3).  Synchronises on the recorded events, adds up their durations,
 * writes the number of launches and the total milliseconds since the previous read of that kind,
 * and recycles the events. */
pf_status pf_profile_read(pf_ctx* ctx, int32_t kind, int64_t* launches, double* total_ms);

/* Bytes of caller-provided scratch needed by a group with prefix length Lp whose longest Phase-B
 * call carries max_Ls suffix tokens (fp32 dQ / dK2 / dV2 staging and softmax statistics). */
size_t pf_workspace_bytes(const pf_desc* desc, int64_t Lp, int64_t max_Ls);

/* Open a group: register the cache K1,V1 [Lp,Hkv,d] bf16 (borrowed, immutable until
 * pf_group_end) and the accumulators gK1,gV1 [Lp,Hkv,d] fp32 contiguous (borrowed; zeroed here,
 * asynchronously on `stream`).  gK1.ptr and gV1.ptr may both be NULL: then
 * Phase B is not allowed and Phase C runs without injection (the N-times replay baseline).
 * `workspace` must be 256-byte aligned device memory of >= pf_workspace_bytes(desc, Lp, max_Ls)
 * for every later call of this group (each call checks the capacity it needs: Phase C Lp rows, a
 * Phase-B wave or a segment its own rows -> PF_WORKSPACE); it may be shared by groups that never overlap in time. */
pf_status pf_group_begin(pf_ctx* ctx, const pf_desc* desc, int64_t Lp, pf_tensor K1, pf_tensor V1,
                         pf_tensor gK1, pf_tensor gV1, void* workspace, size_t workspace_bytes,
                         void* stream, pf_group** out);

/* Phase A: O1[t,h] = softmax_{j<=t}(sigma q1[h,t].k1[g,j]) v1[g,j], LSE1 [Hq,Lp].
 * Q1, O1: [Lp,Hq,d] bf16. */
pf_status pf_phaseA_fwd(pf_group* grp, pf_tensor Q1, pf_tensor O1, float* LSE1, void* stream);

/* Phase B forward: for each of the n_seqs suffixes packed back to back along
 * the token axis (cu_seqlens_host[n_seqs+1], cu[0] = 0; the usual case is n_seqs = 1), the
 * queries of suffix i attend to all Lp cached prefix keys and causally to the keys of suffix i
 * only.  Q2,O2: [sumLs,Hq,d]; K2,V2: [sumLs,Hkv,d]; LSE2: [Hq,sumLs].  K1/V1 are read in place
 * (no concatenation copy).  The sequence offsets are a HOST array: the launch
 * geometry depends on them, and the kernels receive them by value (no device copy is read). */
pf_status pf_phaseB_fwd(pf_group* grp, int32_t n_seqs, const int32_t* cu_seqlens_host,
                        pf_tensor Q2, pf_tensor K2, pf_tensor V2, pf_tensor O2, float* LSE2,
                        void* stream);

/* Phase B backward: dQ2 [sumLs,Hq,d], dK2, dV2 [sumLs,Hkv,d] bf16 of the
 * suffix tokens, and   gK1 += sigma dS21^T Q2,  gV1 += P21^T dO2   (summed over the G query heads
 * of each KV head; fp32; the accumulators persist across calls).  Calls of one
 * group must be stream-ordered or on streams the caller orders. */
pf_status pf_phaseB_bwd(pf_group* grp, int32_t n_seqs, const int32_t* cu_seqlens_host,
                        pf_tensor Q2, pf_tensor K2, pf_tensor V2, pf_tensor O2, const float* LSE2,
                        pf_tensor dO2, pf_tensor dQ2, pf_tensor dK2, pf_tensor dV2, void* stream);

/* Phase C: causal backward over the prefix; dQ1 [Lp,Hq,d] and
 * dK1 = bf16(own-prefix term + gK1), dV1 = bf16(own-prefix term + gV1), the sum taken in fp32
 * and rounded once.  Side effect: on return gK1/gV1 hold that fp32 sum. */
pf_status pf_phaseC_bwd(pf_group* grp, pf_tensor Q1, pf_tensor O1, const float* LSE1,
                        pf_tensor dO1, pf_tensor dQ1, pf_tensor dK1, pf_tensor dV1, void* stream);

/* Segment-by-segment training of ONE long sequence ("a long single sequence can train
 * segment by segment, accumulating gK/gV into earlier segments as Proposition 3.1 prescribes").
 * Segment k is the "suffix" of a group whose prefix [0, Lp) is the concatenation of segments < k:
 * K1/V1 = their keys/values (borrowed in place), gK1/gV1 = rows [0, Lp) of a sequence-wide fp32
 * accumulator [L, Hkv, d] (open the group with option "zero_accumulators" = 0).
 *   pf_group_mark_cached : declares K1/V1 valid without running Phase A (they were produced when the
 *                          earlier segments ran), so that pf_phaseB_fwd may be called for the segment.
 *   pf_segment_bwd       : backward of the segment.  dQ [Ls,Hq,d] bf16; gK1/gV1 += the gradients that
 *                          reach the earlier segments' keys (exactly pf_phaseB_bwd); the segment's own
 *                          key rows accumulate into accK/accV (fp32, contiguous [Ls,Hkv,d]: the
 *                          accumulator rows of THIS segment, which hold the contributions of the later
 *                          segments on entry) and dK, dV = bf16(accK), bf16(accV) on exit -- one rounding.
 * Run the segments in order for the forward and in reverse order for the backward. */
pf_status pf_group_mark_cached(pf_group* grp);

/* Tree-structured data ("each internal node of tree-structured RL data can carry its own
 * K/V cache and gK/gV accumulator"): restrict the prefix that later pf_phaseB_fwd / pf_phaseB_bwd /
 * pf_segment_bwd calls of this group see to n_ranges <= 8 ascending, non-overlapping row ranges
 * [start, start+len) of the K1/V1 (and gK1/gV1) buffers -- the ancestors of the node being processed
 * when all nodes of the tree are stored in one buffer in depth-first order.  Keys outside the ranges
 * are invisible and receive no gradient.  n_ranges = 0 hides the whole prefix.  Host-side only. */
pf_status pf_group_set_prefix_ranges(pf_group* grp, int32_t n_ranges, const int64_t* starts_host,
                                     const int64_t* lens_host);
pf_status pf_segment_bwd(pf_group* grp, int64_t Ls, pf_tensor Q, pf_tensor K, pf_tensor V, pf_tensor O,
                         const float* LSE, pf_tensor dO, pf_tensor dQ, float* accK, float* accV,
                         pf_tensor dK, pf_tensor dV, void* stream);

/* Close the group (host-side; frees the handle only; enqueued work keeps running). */
pf_status pf_group_end(pf_group* grp);

/* Companion 1 -- rotary position embedding with positions that CONTINUE after the prefix
 * ("Position IDs must match the baseline sequence [P||S(i)]; in particular, RoPE
 * positions for suffix tokens continue after the prefix length rather than restarting from zero").
 * X is a packed bf16 tensor [total, n_heads, head_dim] (pf_tensor strides), rotated IN PLACE:
 * row r of sequence s (cu_seqlens_host[s] <= r < cu_seqlens_host[s+1]) has position
 * pos0 + (r - cu_seqlens_host[s]) -- pos0 = 0 for the prefix, pos0 = Lp for a wave of suffixes.
 * Rotate-half convention, theta_j = theta_base^(-2j/d), a = position * theta_j (angle formed in
 * fp64, reduced mod 2 pi, then fp32 sin/cos):
 *     y[j] = x[j] cos a - x[j+d/2] sin a,   y[j+d/2] = x[j+d/2] cos a + x[j] sin a,   j < d/2,
 * computed in fp32 and rounded once to bf16.  inverse != 0 applies the transpose rotation
 * (a -> -a): the backward of the map, to be applied to dQ / dK.  head_dim even, <= 256, multiple
 * of 16; n_seqs >= 0 (longer tables are cut into launches of 32 sequences). */
pf_status pf_rope(pf_ctx* ctx, int32_t n_seqs, const int32_t* cu_seqlens_host, int64_t pos0,
                  pf_tensor X, int32_t n_heads, int32_t head_dim, float theta_base, int32_t inverse,
                  void* stream);

/* Companion 2 -- the K/V-projection weight gradient keeps the baseline's prefix-plus-suffix split
 * (PAPER.md:212): dW_K = X1^T dK1 + sum_i X2(i)^T dK2(i); Phase B accumulates the suffix terms,
 * Phase C adds the prefix term once from a dK1 that already contains every gK1(i).  One call adds
 * one term:  dW[d_model, n_cols] (fp32, row-major, contiguous) += X[L, d_model]^T dY[L, n_cols]
 * with X, dY bf16 row-major (row strides ldx, ldy in elements; dY = dK or dV viewed as
 * [L, Hkv*d]).  A hand-written sm_100a kernel (tcgen05, fp32 accumulation in TMEM, TMA-staged
 * tiles, split over L with a reduce-add into dW); L = 0 is a no-op. d_model and n_cols multiples
 * of 128; X, dY 16-byte aligned, ldx, ldy multiples of 8; dW 16-byte aligned. */
pf_status pf_kv_proj_grad(pf_ctx* ctx, int64_t L, int32_t d_model, int32_t n_cols, const void* X,
                          int64_t ldx, const void* dY, int64_t ldy, float* dW, void* stream);

/* Optional memory lifecycle: move a dormant prefix tensor (contiguous bytes)
 * to / from PINNED host memory on a side stream while Phase B runs.  Plain async copies; the
 * caller orders them against compute with events. */
pf_status pf_offload(pf_ctx* ctx, const void* src_dev, void* dst_pinned_host, size_t bytes,
                     void* side_stream);
pf_status pf_prefetch(pf_ctx* ctx, const void* src_pinned_host, void* dst_dev, size_t bytes,
                      void* side_stream);

/* Allocation-free entry point, for callers that cannot call cudaMalloc (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it): the backward of plain causal
 * self-attention over ONE sequence of L tokens (the oracle's full-sequence causal pass,
 * PAPER.md:194-198 with no prefix; the same kernels and the same result as pf_group_begin(Lp = L,
 * K1 = K, V1 = V, no gK1/gV1, workspace) + pf_group_mark_cached + pf_phaseC_bwd), but with the
 * workspace (softmax statistics, fp32 dQ^T tiles, fp32 dK/dV staging) in a scratch array built into
 * the library: PF_STATIC_SCRATCH_BYTES = 32 MiB of device memory that every GPU loading the library
 * holds until the process exits.  The call makes no cudaMalloc / cudaFree / event or stream
 * creation and takes no caller workspace; inputs Q, O, dO [L, Hq, d], K, V [L, Hkv, d] bf16, LSE
 * [Hq, L] fp32 (row stride L) and outputs dQ [L, Hq, d], dK, dV [L, Hkv, d] bf16 are the caller's
 * device buffers as everywhere else.
 *   Limit: align_up(L, 64) <= pf_causal_bwd_static_max_tokens(desc) (1792 tokens for 28/4 heads of
 *   dim 128; 32 MiB / (8 Hq + 4 Hq d + 8 Hkv d) bytes per token); beyond it the call returns
 *   PF_WORKSPACE with a message and enqueues nothing -- use pf_group_begin with your own workspace.
 *   PF_STATE when the "profile" option is on (its bracket creates events).  L = 0 is a no-op.
 *   The scratch keeps the previous call's contents; what must start at zero (dQ^T tiles, dK/dV
 *   staging) is cleared by the call's own first kernel.  All calls, from every context and stream
 *   of a device, share the one array: two calls that overlap on the GPU race; calls on one stream,
 *   or ordered by events, are safe.  Its device address is taken once per device in pf_create. */
#define PF_STATIC_SCRATCH_BYTES (32u << 20)
size_t pf_static_scratch_bytes(void);
int64_t pf_causal_bwd_static_max_tokens(const pf_desc* desc);
pf_status pf_causal_bwd_static(pf_ctx* ctx, const pf_desc* desc, int64_t L, pf_tensor Q, pf_tensor K,
                               pf_tensor V, pf_tensor O, const float* LSE, pf_tensor dO, pf_tensor dQ,
                               pf_tensor dK, pf_tensor dV, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* PREFIXFLOW_H_ */
