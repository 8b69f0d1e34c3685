"""The three-phase call order of PAPER.md:148-160 on one GPU, and the N-times replay baseline.

Host-side orchestration only: allocates device buffers with torch and issues the C-ABI calls of
`binding` in the paper's order (Phase A once, Phase B fwd+bwd per suffix, Phase C once).  The
replay baseline (BASELINE.json north_star item 3) runs the SAME kernels on each concatenated
[P || S(i)]: a group opened with Lp = T_i and no gK1/gV1, `pf_phaseA_fwd` then `pf_phaseC_bwd`
(one launch pair per trajectory), or all N trajectories packed into one launch pair.  The memory
lifecycle (offload / prefetch of the dormant Phase-A set) lives in `lifecycle.py`.
"""
from __future__ import annotations

import dataclasses
from typing import List, Optional, Sequence

import torch

from . import binding as pf


@dataclasses.dataclass
class DeviceGroup:
    """Device-resident inputs and outputs of one rollout group (token-major [L, H, d])."""

    Hq: int
    Hkv: int
    d: int
    Lp: int
    Ls: List[int]
    Q1: torch.Tensor; K1: torch.Tensor; V1: torch.Tensor; dO1: torch.Tensor
    Q2: List[torch.Tensor]; K2: List[torch.Tensor]; V2: List[torch.Tensor]; dO2: List[torch.Tensor]
    # outputs
    O1: torch.Tensor = None; LSE1: torch.Tensor = None
    O2: List[torch.Tensor] = None; LSE2: List[torch.Tensor] = None
    dQ2: List[torch.Tensor] = None; dK2: List[torch.Tensor] = None; dV2: List[torch.Tensor] = None
    gK1: torch.Tensor = None; gV1: torch.Tensor = None
    dQ1: torch.Tensor = None; dK1: torch.Tensor = None; dV1: torch.Tensor = None
    workspace: torch.Tensor = None
    desc: pf.pf_desc = None
    wave: int = 1
    packed: list = None   # per wave: cu offsets, suffix indices and the packed tensors


def _waves(n: int, wave: int) -> List[List[int]]:
    b = max(1, int(wave))
    return [list(range(i, min(n, i + b))) for i in range(0, n, b)]


def to_device(inp, device="cuda", suffixes: Optional[Sequence[int]] = None, wave: int = 1) -> DeviceGroup:
    """Copy a `inputs.GroupInputs` to the device and allocate every output buffer.

    `wave` = b packs b consecutive suffixes back to back along the token axis (the suffix
    microbatch of PAPER.md:158, 242); Phase B then issues one call per wave.  The per-suffix
    entries of Q2, O2, ... are views of the packed wave tensors."""
    s = inp.shape
    idx = list(range(s.N)) if suffixes is None else list(suffixes)
    dev = torch.device(device)
    mv = lambda t: t.to(dev)
    g = DeviceGroup(
        s.n_q_heads, s.n_kv_heads, s.head_dim, s.Lp, [s.Ls[i] for i in idx],
        mv(inp.Q1), mv(inp.K1), mv(inp.V1), mv(inp.dO1), [], [], [], [])
    g.wave = max(1, int(wave))
    g.packed = []
    for w in _waves(len(idx), g.wave):
        cu = [0]
        for k in w:
            cu.append(cu[-1] + g.Ls[k])
        pk = {"cu": cu, "idx": w}
        for name, src in (("Q2", inp.Q2), ("K2", inp.K2), ("V2", inp.V2), ("dO2", inp.dO2)):
            pk[name] = torch.cat([src[idx[k]] for k in w], 0).contiguous().to(dev)
            getattr(g, name).extend(pk[name][cu[j]:cu[j + 1]] for j in range(len(w)))
        g.packed.append(pk)
    alloc_outputs(g)
    return g


def alloc_outputs(g: DeviceGroup) -> None:
    dev = g.Q1.device
    bf, f32 = torch.bfloat16, torch.float32
    e = lambda L, H, dt=bf: torch.empty((L, H, g.d), dtype=dt, device=dev)
    g.O1 = e(g.Lp, g.Hq); g.LSE1 = torch.empty((g.Hq, g.Lp), dtype=f32, device=dev)
    g.O2, g.LSE2, g.dQ2, g.dK2, g.dV2 = [], [], [], [], []
    max_tok = 0
    for pk in g.packed:
        cu = pk["cu"]
        tot = cu[-1]
        max_tok = max(max_tok, tot)
        pk["O2"] = e(tot, g.Hq); pk["dQ2"] = e(tot, g.Hq)
        pk["dK2"] = e(tot, g.Hkv); pk["dV2"] = e(tot, g.Hkv)
        pk["LSE2"] = torch.empty((g.Hq, tot), dtype=f32, device=dev)
        for j in range(len(pk["idx"])):
            sl = slice(cu[j], cu[j + 1])
            g.O2.append(pk["O2"][sl]); g.dQ2.append(pk["dQ2"][sl])
            g.dK2.append(pk["dK2"][sl]); g.dV2.append(pk["dV2"][sl])
            g.LSE2.append(pk["LSE2"][:, sl])
    g.gK1 = e(g.Lp, g.Hkv, f32); g.gV1 = e(g.Lp, g.Hkv, f32)
    g.dQ1 = e(g.Lp, g.Hq); g.dK1 = e(g.Lp, g.Hkv); g.dV1 = e(g.Lp, g.Hkv)
    g.desc = pf.make_desc(g.Hq, g.Hkv, g.d)
    nbytes = pf.pf_workspace_bytes(g.desc, g.Lp, max_tok)
    g.workspace = torch.empty(nbytes, dtype=torch.uint8, device=dev)


def run_prefixflow_step(ctx, g: DeviceGroup, stream=None, after_each_suffix=None,
                        order: Optional[Sequence[int]] = None, fwd_stream=None) -> None:
    """Phase A -> Phase B (fwd, bwd) per suffix wave -> Phase C.
    `order` permutes the waves (= the suffixes when wave == 1).

    `fwd_stream` (a torch.cuda.Stream other than `stream`): the Phase-B forwards are enqueued there
    instead.  They read only Q2/K2/V2 and the cached K1/V1 (inputs of the step), so the
    forward of wave i+1 may run while the backward of wave i does, and the first one beside Phase A:
    the SMs a launch leaves idle in its last round of CTAs are picked up by the other stream's launch.
    Every backward waits for its own forward; the forwards of a step wait for everything enqueued on
    `stream` before it (the previous step's backward still reads O2 / LSE2)."""
    main = stream if isinstance(stream, torch.cuda.Stream) else None
    if fwd_stream is not None:
        if main is None:
            if stream is not None:
                raise ValueError("fwd_stream needs `stream` as a torch.cuda.Stream (or None = the current stream)")
            main = torch.cuda.current_stream()
        fwd_stream.wait_stream(main)
    grp = pf.pf_group_begin(ctx, g.desc, g.Lp, g.K1, g.V1, g.gK1, g.gV1, g.workspace, stream)
    try:
        pf.pf_phaseA_fwd(grp, g.Q1, g.O1, g.LSE1, stream)
        for i in (range(len(g.packed)) if order is None else order):
            pk = g.packed[i]
            cu = pk["cu"]
            pf.pf_phaseB_fwd(grp, cu, pk["Q2"], pk["K2"], pk["V2"], pk["O2"], pk["LSE2"],
                             stream if fwd_stream is None else fwd_stream)
            if fwd_stream is not None:
                main.wait_stream(fwd_stream)   # (an event recorded on fwd_stream here; later forwards are not waited for)
            pf.pf_phaseB_bwd(grp, cu, pk["Q2"], pk["K2"], pk["V2"], pk["O2"], pk["LSE2"], pk["dO2"],
                             pk["dQ2"], pk["dK2"], pk["dV2"], stream)
            if after_each_suffix is not None:
                after_each_suffix(pk["idx"][-1])
        pf.pf_phaseC_bwd(grp, g.Q1, g.O1, g.LSE1, g.dO1, g.dQ1, g.dK1, g.dV1, stream)
    finally:
        pf.pf_group_end(grp)


def run_prefixflow_step_partials(ctx, g: DeviceGroup, partial_K: torch.Tensor, partial_V: torch.Tensor,
                                 stream=None) -> None:
    """The REJECTED alternative of BASELINE.json north_star item (2), kept only so that it can be
    measured next to the shipped accumulation: every Phase-B wave adds its prefix
    gradients into a partial accumulator of its own (`partial_K/V` fp32 [n_waves, Lp, Hkv, d], zeroed
    by the wave's pf_group_begin), and a reduce pass sums the partials into gK1/gV1 before Phase C.
    The reduce is a plain elementwise torch.sum: an HBM-bound pass over n_waves x 2 x Lp x Hkv x d x 4 B."""
    main = pf.pf_group_begin(ctx, g.desc, g.Lp, g.K1, g.V1, g.gK1, g.gV1, g.workspace, stream)
    try:
        pf.pf_phaseA_fwd(main, g.Q1, g.O1, g.LSE1, stream)
        for i, pk in enumerate(g.packed):
            grp = pf.pf_group_begin(ctx, g.desc, g.Lp, g.K1, g.V1, partial_K[i], partial_V[i], g.workspace, stream)
            try:
                pf.pf_group_mark_cached(grp)
                cu = pk["cu"]
                pf.pf_phaseB_fwd(grp, cu, pk["Q2"], pk["K2"], pk["V2"], pk["O2"], pk["LSE2"], stream)
                pf.pf_phaseB_bwd(grp, cu, pk["Q2"], pk["K2"], pk["V2"], pk["O2"], pk["LSE2"], pk["dO2"],
                                 pk["dQ2"], pk["dK2"], pk["dV2"], stream)
            finally:
                pf.pf_group_end(grp)
        with torch.cuda.stream(stream) if isinstance(stream, torch.cuda.Stream) else _nullctx():
            torch.sum(partial_K[:len(g.packed)], 0, out=g.gK1)
            torch.sum(partial_V[:len(g.packed)], 0, out=g.gV1)
        pf.pf_phaseC_bwd(main, g.Q1, g.O1, g.LSE1, g.dO1, g.dQ1, g.dK1, g.dV1, stream)
    finally:
        pf.pf_group_end(main)


class _nullctx:
    def __enter__(self):
        return None

    def __exit__(self, *a):
        return False


def capture_step(ctx, g: DeviceGroup, order: Optional[Sequence[int]] = None,
                 fwd_stream=None) -> "torch.cuda.CUDAGraph":
    """One A -> B -> C step captured into a CUDA graph.  Every C-ABI call only enqueues memsets and
    kernels on the caller's stream (tensor maps and kernel parameters are baked in at capture), so a
    training loop whose buffers keep their addresses replays the whole step with one launch; the
    launch gaps between the ~18 (one packed wave) to ~60 (one call per suffix) dependent kernels of
    a step go away.  The profile option must be off during capture.  With `fwd_stream` the fork to and
    the joins from the forwards' stream are captured too (every forward is joined by its backward)."""
    side = torch.cuda.Stream(g.Q1.device)
    side.wait_stream(torch.cuda.current_stream(g.Q1.device))
    with torch.cuda.stream(side):                 # warm-up outside the capture (lazy module loads)
        run_prefixflow_step(ctx, g, side, order=order, fwd_stream=fwd_stream)
    torch.cuda.current_stream(g.Q1.device).wait_stream(side)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        run_prefixflow_step(ctx, g, torch.cuda.current_stream(g.Q1.device), order=order, fwd_stream=fwd_stream)
    return graph


def head_shard(g: DeviceGroup, world: int, rank: int) -> DeviceGroup:
    """KV-head shard `rank` of `world` of a device group (the paper's TP rule: each
    rank caches its own head shard, no communication): the bf16 inputs and outputs are head slices
    of the full group's tensors IN PLACE (strided views: the C ABI takes token / head strides), the
    fp32 accumulators, LSE and workspace of the shard are its own.  Running `run_prefixflow_step` on
    every shard fills the full group's bf16 outputs; LSE / gK1 / gV1 are per shard."""
    if g.Hkv % world != 0:
        raise ValueError(f"{g.Hkv} KV heads do not shard over {world} ranks")
    G = g.Hq // g.Hkv
    kv = slice(rank * (g.Hkv // world), (rank + 1) * (g.Hkv // world))
    qh = slice(kv.start * G, kv.stop * G)
    q = lambda t: t[:, qh]
    k = lambda t: t[:, kv]
    sh = DeviceGroup(qh.stop - qh.start, kv.stop - kv.start, g.d, g.Lp, list(g.Ls),
                     q(g.Q1), k(g.K1), k(g.V1), q(g.dO1), [], [], [], [])
    sh.wave = g.wave
    sh.packed = []
    dev = g.Q1.device
    f32 = torch.float32
    sh.O1, sh.dQ1, sh.dK1, sh.dV1 = q(g.O1), q(g.dQ1), k(g.dK1), k(g.dV1)
    sh.LSE1 = torch.empty((sh.Hq, g.Lp), dtype=f32, device=dev)
    sh.gK1 = torch.empty((g.Lp, sh.Hkv, g.d), dtype=f32, device=dev)
    sh.gV1 = torch.empty_like(sh.gK1)
    sh.O2, sh.LSE2, sh.dQ2, sh.dK2, sh.dV2 = [], [], [], [], []
    max_tok = 0
    for pk in g.packed:
        cu = pk["cu"]
        max_tok = max(max_tok, cu[-1])
        spk = {"cu": cu, "idx": pk["idx"]}
        for name in ("Q2", "dO2", "O2", "dQ2"):
            spk[name] = q(pk[name])
        for name in ("K2", "V2", "dK2", "dV2"):
            spk[name] = k(pk[name])
        spk["LSE2"] = torch.empty((sh.Hq, cu[-1]), dtype=f32, device=dev)
        for j in range(len(pk["idx"])):
            sl = slice(cu[j], cu[j + 1])
            for name in ("Q2", "K2", "V2", "dO2", "O2", "dQ2", "dK2", "dV2"):
                getattr(sh, name).append(spk[name][sl])
            sh.LSE2.append(spk["LSE2"][:, sl])
        sh.packed.append(spk)
    sh.desc = pf.make_desc(sh.Hq, sh.Hkv, g.d)
    sh.workspace = torch.empty(pf.pf_workspace_bytes(sh.desc, g.Lp, max_tok), dtype=torch.uint8, device=dev)
    return sh


@dataclasses.dataclass
class ReplayBuffers:
    """Concatenated [P || S(i)] tensors of the N-times replay baseline (one set per trajectory)."""

    T: List[int]
    Q: List[torch.Tensor]; K: List[torch.Tensor]; V: List[torch.Tensor]; dO: List[torch.Tensor]
    O: List[torch.Tensor]; LSE: List[torch.Tensor]
    dQ: List[torch.Tensor]; dK: List[torch.Tensor]; dV: List[torch.Tensor]
    workspace: torch.Tensor
    desc: pf.pf_desc


def make_replay(g: DeviceGroup, prefix_weight: Optional[float] = None) -> ReplayBuffers:
    """Replay i sees dO = [w_i * dO1 ; dO2(i)], w_i = 1/N by default (reading 1)."""
    n = len(g.Ls)
    w = (1.0 / n if n else 1.0) if prefix_weight is None else prefix_weight
    cat = lambda a, b: torch.cat([a, b], 0).contiguous()
    Q = [cat(g.Q1, q) for q in g.Q2]; K = [cat(g.K1, k) for k in g.K2]
    V = [cat(g.V1, v) for v in g.V2]
    dO = [cat((g.dO1.float() * w).to(torch.bfloat16), x) for x in g.dO2]
    T = [g.Lp + L for L in g.Ls]
    dev = g.Q1.device
    e = lambda L, H: torch.empty((L, H, g.d), dtype=torch.bfloat16, device=dev)
    nbytes = pf.pf_workspace_bytes(g.desc, max(T, default=0), 0)
    return ReplayBuffers(
        T, Q, K, V, dO, [e(t, g.Hq) for t in T],
        [torch.empty((g.Hq, t), dtype=torch.float32, device=dev) for t in T],
        [e(t, g.Hq) for t in T], [e(t, g.Hkv) for t in T], [e(t, g.Hkv) for t in T],
        torch.empty(nbytes, dtype=torch.uint8, device=dev), g.desc)


def run_replay_step(ctx, r: ReplayBuffers, stream=None) -> None:
    """N independent full-sequence causal fwd+bwd passes with the same kernels."""
    for i, T in enumerate(r.T):
        grp = pf.pf_group_begin(ctx, r.desc, T, r.K[i], r.V[i], None, None, r.workspace, stream)
        try:
            pf.pf_phaseA_fwd(grp, r.Q[i], r.O[i], r.LSE[i], stream)
            pf.pf_phaseC_bwd(grp, r.Q[i], r.O[i], r.LSE[i], r.dO[i], r.dQ[i], r.dK[i], r.dV[i], stream)
        finally:
            pf.pf_group_end(grp)


# --------------------------------------------------------------------------------------------------
# The same replay with all N full sequences packed into ONE launch pair (Lp = 0, n_seqs = N): the
# fair "same kernels" baseline when the step under test packs its suffixes too -- both pay one launch
# tail per kernel.
# --------------------------------------------------------------------------------------------------
@dataclasses.dataclass
class PackedReplay:
    cu: List[int]
    Q: torch.Tensor; K: torch.Tensor; V: torch.Tensor; dO: torch.Tensor
    O: torch.Tensor; LSE: torch.Tensor; dQ: torch.Tensor; dK: torch.Tensor; dV: torch.Tensor
    workspace: torch.Tensor
    desc: pf.pf_desc


def make_replay_packed(g: DeviceGroup, prefix_weight: Optional[float] = None) -> PackedReplay:
    """[P || S(1)] ... [P || S(N)] back to back along the token axis; replay i sees the prefix-row
    adjoint w_i dO1, w_i = 1/N by default (reading 1; input preparation of the baseline)."""
    n = len(g.Ls)
    w = (1.0 / n if n else 1.0) if prefix_weight is None else prefix_weight
    dO1w = (g.dO1.float() * w).to(torch.bfloat16)
    cat = lambda first, rest: torch.cat([t for r in rest for t in (first, r)], 0).contiguous()
    Q, K, V, dO = cat(g.Q1, g.Q2), cat(g.K1, g.K2), cat(g.V1, g.V2), cat(dO1w, g.dO2)
    cu = [0]
    for L in g.Ls:
        cu.append(cu[-1] + g.Lp + L)
    dev = g.Q1.device
    e = lambda t: torch.empty_like(t)
    nbytes = pf.pf_workspace_bytes(g.desc, 0, cu[-1])
    return PackedReplay(cu, Q, K, V, dO, e(Q), torch.empty((g.Hq, cu[-1]), dtype=torch.float32, device=dev),
                        e(Q), e(K), e(V), torch.empty(nbytes, dtype=torch.uint8, device=dev), g.desc)


def run_replay_packed_step(ctx, r: PackedReplay, stream=None) -> None:
    """One forward and one backward launch over the N packed full sequences (plain causal attention:
    a group without a prefix whose `suffixes` are the whole trajectories)."""
    grp = pf.pf_group_begin(ctx, r.desc, 0, None, None, None, None, r.workspace, stream)
    try:
        pf.pf_group_mark_cached(grp)
        pf.pf_phaseB_fwd(grp, r.cu, r.Q, r.K, r.V, r.O, r.LSE, stream)
        pf.pf_phaseB_bwd(grp, r.cu, r.Q, r.K, r.V, r.O, r.LSE, r.dO, r.dQ, r.dK, r.dV, stream)
    finally:
        pf.pf_group_end(grp)


def random_device_group(shape, device="cuda", wave: int = 1, seed: int = 0) -> DeviceGroup:
    """A rollout group of the given shape drawn directly on the device (N(0,1)/sqrt(d) -> bf16):
    for timing sweeps over many configurations, where values do not matter and the CPU generator
    of `inputs.make_group` would dominate the run.  Parity tests never use this."""
    dev = torch.device(device)
    gen = torch.Generator(device=dev)
    gen.manual_seed(seed)
    d, sc = shape.head_dim, shape.head_dim ** -0.5
    draw = lambda L, H: (torch.randn((L, H, d), generator=gen, device=dev, dtype=torch.float32) * sc).to(torch.bfloat16)
    Hq, Hkv = shape.n_q_heads, shape.n_kv_heads
    g = DeviceGroup(Hq, Hkv, d, shape.Lp, list(shape.Ls), draw(shape.Lp, Hq), draw(shape.Lp, Hkv),
                    draw(shape.Lp, Hkv), draw(shape.Lp, Hq), [], [], [], [])
    g.wave = max(1, int(wave))
    g.packed = []
    for w in _waves(shape.N, g.wave):
        cu = [0]
        for k in w:
            cu.append(cu[-1] + shape.Ls[k])
        pk = {"cu": cu, "idx": w}
        for name, H in (("Q2", Hq), ("K2", Hkv), ("V2", Hkv), ("dO2", Hq)):
            pk[name] = draw(cu[-1], H)
            getattr(g, name).extend(pk[name][cu[j]:cu[j + 1]] for j in range(len(w)))
        g.packed.append(pk)
    alloc_outputs(g)
    return g


# --------------------------------------------------------------------------------------------------
# Segment-by-segment training of one long sequence: causal
# attention over [S_0 | S_1 | ... | S_m-1] computed one segment at a time.  Forward in order: segment k
# attends to the cached K/V of segments < k (in place, rows [0, Lp_k) of the sequence's K/V) and
# causally to itself.  Backward in reverse order: segment k's gradient reaches the earlier segments'
# keys through the sequence-wide fp32 accumulator (gK/gV superposition, Proposition 3.1) and its
# own key rows add onto what the later segments left there, rounded to bf16 once.
# --------------------------------------------------------------------------------------------------
def run_segmented_sequence(ctx, Q, K, V, dO, seg_lens: Sequence[int], stream=None) -> dict:
    """Q, dO [L,Hq,d], K, V [L,Hkv,d] bf16 device tensors; returns O, LSE, dQ, dK, dV of the whole
    sequence (identical, up to rounding order, to one full causal pass)."""
    L, Hq, d = Q.shape
    Hkv = K.shape[1]
    assert sum(seg_lens) == L
    dev = Q.device
    desc = pf.make_desc(Hq, Hkv, d)
    O = torch.empty_like(Q); dQ = torch.empty_like(Q)
    dK = torch.empty_like(K); dV = torch.empty_like(V)
    LSE = [torch.empty((Hq, n), dtype=torch.float32, device=dev) for n in seg_lens]
    accK = torch.zeros((L, Hkv, d), dtype=torch.float32, device=dev)   # sequence-wide gK / gV
    accV = torch.zeros((L, Hkv, d), dtype=torch.float32, device=dev)
    ws = torch.empty(pf.pf_workspace_bytes(desc, 0, max(seg_lens)), dtype=torch.uint8, device=dev)
    starts = [sum(seg_lens[:k]) for k in range(len(seg_lens))]
    pf.pf_set_option(ctx, "zero_accumulators", 0)
    try:
        def open_group(k):
            lo = starts[k]
            g = pf.pf_group_begin(ctx, desc, lo, K[:lo], V[:lo], accK[:lo], accV[:lo], ws, stream)
            pf.pf_group_mark_cached(g)
            return g, slice(lo, lo + seg_lens[k])
        for k in range(len(seg_lens)):                       # forward, in order
            g, sl = open_group(k)
            try:
                pf.pf_phaseB_fwd(g, [0, seg_lens[k]], Q[sl], K[sl], V[sl], O[sl], LSE[k], stream)
            finally:
                pf.pf_group_end(g)
        for k in range(len(seg_lens) - 1, -1, -1):           # backward, in reverse order
            g, sl = open_group(k)
            try:
                pf.pf_segment_bwd(g, Q[sl], K[sl], V[sl], O[sl], LSE[k], dO[sl], dQ[sl],
                                  accK[sl], accV[sl], dK[sl], dV[sl], stream)
            finally:
                pf.pf_group_end(g)
    finally:
        pf.pf_set_option(ctx, "zero_accumulators", 1)
    return dict(O=O, LSE=torch.cat(LSE, 1), dQ=dQ, dK=dK, dV=dV)


# --------------------------------------------------------------------------------------------------
# Tree-structured data: all nodes of a prefix tree stored in ONE
# [L, H, d] buffer in depth-first order; a node attends to its ancestors (row ranges of the buffer
# before it, `pf_group_set_prefix_ranges`) and causally to itself.  Forward in DFS order; backward in
# reverse DFS order, every node adding into its ancestors' rows of the tree-wide fp32 gK/gV
# accumulator and finishing its own rows (children first, so all contributions have arrived).
# --------------------------------------------------------------------------------------------------
def tree_ranges(nodes: Sequence[Sequence[int]]):
    """nodes[i] = (parent index or -1, length), in DFS order.  Returns (starts, per-node ancestor
    ranges [(start, len), ...] with adjacent ranges merged)."""
    starts, out = [], []
    pos = 0
    for parent, n in nodes:
        starts.append(pos)
        pos += n
    for i, (parent, n) in enumerate(nodes):
        path = []
        a = parent
        while a >= 0:
            path.append(a)
            a = nodes[a][0]
        rs = []
        for a in reversed(path):
            if nodes[a][1] == 0:
                continue
            if rs and rs[-1][0] + rs[-1][1] == starts[a]:
                rs[-1] = (rs[-1][0], rs[-1][1] + nodes[a][1])
            else:
                rs.append((starts[a], nodes[a][1]))
        out.append(rs)
    return starts, out


def run_tree(ctx, Q, K, V, dO, nodes: Sequence[Sequence[int]], stream=None) -> dict:
    """Attention forward + backward over a prefix tree (see above); returns O, LSE (per node), dQ, dK, dV."""
    L, Hq, d = Q.shape
    Hkv = K.shape[1]
    lens = [n for _, n in nodes]
    assert sum(lens) == L
    dev = Q.device
    desc = pf.make_desc(Hq, Hkv, d)
    starts, ranges = tree_ranges(nodes)
    O = torch.empty_like(Q); dQ = torch.empty_like(Q)
    dK = torch.empty_like(K); dV = torch.empty_like(V)
    LSE = [torch.empty((Hq, n), dtype=torch.float32, device=dev) for n in lens]
    accK = torch.zeros((L, Hkv, d), dtype=torch.float32, device=dev)   # tree-wide gK / gV
    accV = torch.zeros((L, Hkv, d), dtype=torch.float32, device=dev)
    ws = torch.empty(pf.pf_workspace_bytes(desc, 0, max(lens)), dtype=torch.uint8, device=dev)
    pf.pf_set_option(ctx, "zero_accumulators", 0)
    try:
        def open_group(i):
            lo = starts[i]
            g = pf.pf_group_begin(ctx, desc, lo, K[:lo], V[:lo], accK[:lo], accV[:lo], ws, stream)
            pf.pf_group_set_prefix_ranges(g, ranges[i])
            pf.pf_group_mark_cached(g)
            return g, slice(lo, lo + lens[i])
        for i in range(len(nodes)):
            if lens[i] == 0:
                continue
            g, sl = open_group(i)
            try:
                pf.pf_phaseB_fwd(g, [0, lens[i]], Q[sl], K[sl], V[sl], O[sl], LSE[i], stream)
            finally:
                pf.pf_group_end(g)
        for i in range(len(nodes) - 1, -1, -1):
            if lens[i] == 0:
                continue
            g, sl = open_group(i)
            try:
                pf.pf_segment_bwd(g, Q[sl], K[sl], V[sl], O[sl], LSE[i], dO[sl], dQ[sl],
                                  accK[sl], accV[sl], dK[sl], dV[sl], stream)
            finally:
                pf.pf_group_end(g)
    finally:
        pf.pf_set_option(ctx, "zero_accumulators", 1)
    return dict(O=O, LSE=LSE, dQ=dQ, dK=dK, dV=dV, starts=starts)
