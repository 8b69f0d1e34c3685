"""The three-phase call order of PAPER.md:148-160 on one GPU, and the N-times replay baseline.

Host-side orchestration only: allocates device buffers with torch and issues the C-ABI calls of
`binding` in the paper's order (Phase A once, Phase B fwd+bwd per suffix, Phase C once).  The
replay baseline (BASELINE.json north_star item 3) runs the SAME kernels on each concatenated
[P || S(i)]: a group opened with Lp = T_i and no gK1/gV1, `pf_phaseA_fwd` then `pf_phaseC_bwd`.
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
                        order: Optional[Sequence[int]] = None) -> None:
    """Phase A -> Phase B (fwd, bwd) per suffix wave -> Phase C.
    `order` permutes the waves (= the suffixes when wave == 1)."""
    grp = pf.pf_group_begin(ctx, g.desc, g.Lp, g.K1, g.V1, g.gK1, g.gV1, g.workspace, stream)
    try:
        pf.pf_phaseA_fwd(grp, g.Q1, g.O1, g.LSE1, stream)
        for i in (range(len(g.packed)) if order is None else order):
            pk = g.packed[i]
            cu = pk["cu"]
            pf.pf_phaseB_fwd(grp, cu, pk["Q2"], pk["K2"], pk["V2"], pk["O2"], pk["LSE2"], stream)
            pf.pf_phaseB_bwd(grp, cu, pk["Q2"], pk["K2"], pk["V2"], pk["O2"], pk["LSE2"], pk["dO2"],
                             pk["dQ2"], pk["dK2"], pk["dV2"], stream)
            if after_each_suffix is not None:
                after_each_suffix(pk["idx"][-1])
        pf.pf_phaseC_bwd(grp, g.Q1, g.O1, g.LSE1, g.dO1, g.dQ1, g.dK1, g.dV1, stream)
    finally:
        pf.pf_group_end(grp)


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
# Memory lifecycle of one layer: hot set {K1, V1, gK1, gV1} stays resident, the
# dormant Phase-A set {Q1, O1, LSE1} leaves for pinned host memory on a side stream while Phase B
# runs and is prefetched back before Phase C; suffix-wave tensors live only during their wave.
# --------------------------------------------------------------------------------------------------
def run_lifecycle_step(ctx, inp, device="cuda", wave: int = 1, offload: bool = True,
                       pinned: Optional[dict] = None, keep_outputs: bool = False) -> dict:
    """One A -> B -> C step that allocates and frees device tensors the way a trainer would.
    Returns peak allocated bytes of the whole step and of Phase B alone (the paper's
    "Phase-B peak HBM"), the step time, and (optionally) the outputs."""
    s = inp.shape
    dev = torch.device(device)
    Hq, Hkv, d, Lp = s.n_q_heads, s.n_kv_heads, s.head_dim, s.Lp
    bf, f32 = torch.bfloat16, torch.float32
    main = torch.cuda.current_stream(dev)
    side = pinned.setdefault("side_stream", torch.cuda.Stream(dev)) if pinned is not None else torch.cuda.Stream(dev)
    pinned = pinned if pinned is not None else {}

    def pin(name, like):
        if name not in pinned:
            pinned[name] = torch.empty(like.shape, dtype=like.dtype, pin_memory=True)
        return pinned[name]

    e = lambda L, H, dt=bf: torch.empty((L, H, d), dtype=dt, device=dev)
    waves = _waves(s.N, wave)
    max_tok = max((sum(s.Ls[k] for k in w) for w in waves), default=0)
    desc = pf.make_desc(Hq, Hkv, d)
    torch.cuda.synchronize(dev)
    torch.cuda.reset_peak_memory_stats(dev)
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record(main)
    # ---- Phase A
    Q1, K1, V1 = inp.Q1.to(dev), inp.K1.to(dev), inp.V1.to(dev)
    O1 = e(Lp, Hq); LSE1 = torch.empty((Hq, Lp), dtype=f32, device=dev)
    gK1, gV1 = e(Lp, Hkv, f32), e(Lp, Hkv, f32)
    ws = torch.empty(pf.pf_workspace_bytes(desc, Lp, max_tok), dtype=torch.uint8, device=dev)
    grp = pf.pf_group_begin(ctx, desc, Lp, K1, V1, gK1, gV1, ws, main)
    outs = {}
    try:
        pf.pf_phaseA_fwd(grp, Q1, O1, LSE1, main)
        dormant = {"Q1": Q1, "O1": O1, "LSE1": LSE1}
        if offload:
            evA = torch.cuda.Event(); evA.record(main)
            side.wait_event(evA)
            for name, t in dormant.items():
                pf.pf_offload(ctx, t, pin(name, t), side)
            side.synchronize()        # the copies ran beside nothing here; a trainer overlaps them with wave 1
            if keep_outputs:
                outs["O1"], outs["LSE1"] = O1.clone(), LSE1.clone()
            shapes = {k: (t.shape, t.dtype) for k, t in dormant.items()}
            del Q1, O1, LSE1, dormant
        # ---- Phase B, one wave at a time; a wave's tensors are freed when the wave is done
        peak_a = torch.cuda.max_memory_allocated(dev)
        torch.cuda.reset_peak_memory_stats(dev)
        base = torch.cuda.memory_allocated(dev)
        for w in waves:
            cu = [0]
            for k in w:
                cu.append(cu[-1] + s.Ls[k])
            cat = lambda src: torch.cat([src[k] for k in w], 0).contiguous().to(dev)
            Q2, K2, V2, dO2 = cat(inp.Q2), cat(inp.K2), cat(inp.V2), cat(inp.dO2)
            tot = cu[-1]
            O2, dQ2 = e(tot, Hq), e(tot, Hq)
            dK2, dV2 = e(tot, Hkv), e(tot, Hkv)
            LSE2 = torch.empty((Hq, tot), dtype=f32, device=dev)
            pf.pf_phaseB_fwd(grp, cu, Q2, K2, V2, O2, LSE2, main)
            pf.pf_phaseB_bwd(grp, cu, Q2, K2, V2, O2, LSE2, dO2, dQ2, dK2, dV2, main)
            if keep_outputs:
                for j, k in enumerate(w):
                    sl = slice(cu[j], cu[j + 1])
                    outs[f"O2[{k}]"], outs[f"LSE2[{k}]"] = O2[sl].clone(), LSE2[:, sl].clone()
                    outs[f"dQ2[{k}]"], outs[f"dK2[{k}]"], outs[f"dV2[{k}]"] = (
                        dQ2[sl].clone(), dK2[sl].clone(), dV2[sl].clone())
            del Q2, K2, V2, dO2, O2, dQ2, dK2, dV2, LSE2
        peak_b = torch.cuda.max_memory_allocated(dev)
        # ---- prefetch the dormant set back (side stream), then Phase C
        if offload:
            Q1 = torch.empty(shapes["Q1"][0], dtype=shapes["Q1"][1], device=dev)
            O1 = torch.empty(shapes["O1"][0], dtype=shapes["O1"][1], device=dev)
            LSE1 = torch.empty(shapes["LSE1"][0], dtype=shapes["LSE1"][1], device=dev)
            evB = torch.cuda.Event(); evB.record(main)   # the fresh buffers may reuse blocks Phase B still reads
            side.wait_event(evB)
            for name, t in (("Q1", Q1), ("O1", O1), ("LSE1", LSE1)):
                pf.pf_prefetch(ctx, pinned[name], t, side)
            evP = torch.cuda.Event(); evP.record(side)
            main.wait_event(evP)
        elif keep_outputs:
            outs["O1"], outs["LSE1"] = O1.clone(), LSE1.clone()
        dO1 = inp.dO1.to(dev)
        dQ1, dK1, dV1 = e(Lp, Hq), e(Lp, Hkv), e(Lp, Hkv)
        pf.pf_phaseC_bwd(grp, Q1, O1, LSE1, dO1, dQ1, dK1, dV1, main)
    finally:
        pf.pf_group_end(grp)
    t1.record(main)
    torch.cuda.synchronize(dev)
    if keep_outputs:
        outs.update(dQ1=dQ1, dK1=dK1, dV1=dV1)
    return dict(ms=t0.elapsed_time(t1), peak_step_bytes=max(peak_a, torch.cuda.max_memory_allocated(dev)),
                peak_phaseB_bytes=peak_b, resident_at_phaseB_start_bytes=base, outputs=outs)


# --------------------------------------------------------------------------------------------------
# Multi-layer lifecycle: L attention layers, each with
# its own training-time KV cache.  Phase A runs layer by layer and every layer's dormant set
# {Q1, O1, LSE1} leaves for the pinned host pool on the side stream as soon as it is produced;
# Phase B runs all waves on all layers with only the hot sets {K1, V1, gK1, gV1} resident; Phase C
# runs in reverse layer order with the dormant set of layer l-1 prefetched while layer l computes
# (if a prefetch has not been issued or has not landed, Phase C simply waits for it: demand load).
# --------------------------------------------------------------------------------------------------
def run_multilayer_step(ctx, layers, device="cuda", wave: int = 1, offload: bool = True,
                        pinned: Optional[dict] = None, keep_outputs: bool = False,
                        early_prefetch: bool = False) -> dict:
    """`layers`: list of inputs.GroupInputs with identical shapes (one per attention layer).
    `early_prefetch` issues the first Phase-C prefetch behind the last Phase-B wave: no exposed wait,
    but its buffers count in the Phase-B peak."""
    s = layers[0].shape
    dev = torch.device(device)
    Hq, Hkv, d, Lp, L = s.n_q_heads, s.n_kv_heads, s.head_dim, s.Lp, len(layers)
    bf, f32 = torch.bfloat16, torch.float32
    main = torch.cuda.current_stream(dev)
    pinned = pinned if pinned is not None else {}
    side = pinned.setdefault("side_stream", torch.cuda.Stream(dev))
    e = lambda n, H, dt=bf: torch.empty((n, H, d), dtype=dt, device=dev)
    waves = _waves(s.N, wave)
    max_tok = max((sum(s.Ls[k] for k in w) for w in waves), default=0)
    desc = pf.make_desc(Hq, Hkv, d)

    def pin(l, name, like):
        key = (l, name)
        if key not in pinned:
            pinned[key] = torch.empty(like.shape, dtype=like.dtype, pin_memory=True)
        return pinned[key]

    torch.cuda.synchronize(dev)
    torch.cuda.reset_peak_memory_stats(dev)
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record(main)
    ws = torch.empty(pf.pf_workspace_bytes(desc, Lp, max_tok), dtype=torch.uint8, device=dev)
    hot, dorm, grp, outs = [], [], [], [dict() for _ in range(L)]
    exposed = []                                    # (event before wait, event after wait) per layer
    try:
        # ---- Phase A, layer by layer; dormant sets stream out behind it
        for l, inp in enumerate(layers):
            Q1, K1, V1 = inp.Q1.to(dev), inp.K1.to(dev), inp.V1.to(dev)
            O1 = e(Lp, Hq); LSE1 = torch.empty((Hq, Lp), dtype=f32, device=dev)
            gK1, gV1 = e(Lp, Hkv, f32), e(Lp, Hkv, f32)
            g = pf.pf_group_begin(ctx, desc, Lp, K1, V1, gK1, gV1, ws, main)
            grp.append(g)
            pf.pf_phaseA_fwd(g, Q1, O1, LSE1, main)
            hot.append(dict(K1=K1, V1=V1, gK1=gK1, gV1=gV1))
            dset = dict(Q1=Q1, O1=O1, LSE1=LSE1)
            if keep_outputs:
                outs[l]["O1"], outs[l]["LSE1"] = O1.clone(), LSE1.clone()
            if offload:
                ev = torch.cuda.Event(); ev.record(main)
                side.wait_event(ev)
                for name, t in dset.items():
                    pf.pf_offload(ctx, t, pin(l, name, t), side)
                dset = dict(shapes={k: (t.shape, t.dtype) for k, t in dset.items()},
                            done=torch.cuda.Event())
                dset["done"].record(side)
                dset["keep"] = (Q1, O1, LSE1)       # freed once the copy has left (below)
            dorm.append(dset)
            del Q1, O1, LSE1
        if offload:
            side.synchronize()                      # all dormant sets are on the host: free them
            for dset in dorm:
                dset.pop("keep")
        peak_a = torch.cuda.max_memory_allocated(dev)
        torch.cuda.reset_peak_memory_stats(dev)
        base = torch.cuda.memory_allocated(dev)
        def prefetch(l):
            dset = dorm[l]
            ev = torch.cuda.Event(); ev.record(main)   # fresh buffers may reuse blocks main still reads
            bufs = {k: torch.empty(sh, dtype=dt, device=dev) for k, (sh, dt) in dset["shapes"].items()}
            side.wait_event(ev)
            for name, t in bufs.items():
                pf.pf_prefetch(ctx, pinned[(l, name)], t, side)
            dset["bufs"], dset["landed"] = bufs, torch.cuda.Event()
            dset["landed"].record(side)

        # ---- Phase B: every wave on every layer (a wave's tensors live only during the wave)
        for wi, w in enumerate(waves):
            if offload and early_prefetch and wi == len(waves) - 1:
                prefetch(L - 1)                       # hidden behind the last wave (costs its buffers in the Phase-B peak)
            cu = [0]
            for k in w:
                cu.append(cu[-1] + s.Ls[k])
            tot = cu[-1]
            for l, inp in enumerate(layers):
                cat = lambda src: torch.cat([src[k] for k in w], 0).contiguous().to(dev)
                Q2, K2, V2, dO2 = cat(inp.Q2), cat(inp.K2), cat(inp.V2), cat(inp.dO2)
                O2, dQ2, dK2, dV2 = e(tot, Hq), e(tot, Hq), e(tot, Hkv), e(tot, Hkv)
                LSE2 = torch.empty((Hq, tot), dtype=f32, device=dev)
                pf.pf_phaseB_fwd(grp[l], cu, Q2, K2, V2, O2, LSE2, main)
                pf.pf_phaseB_bwd(grp[l], cu, Q2, K2, V2, O2, LSE2, dO2, dQ2, dK2, dV2, main)
                if keep_outputs:
                    for j, k in enumerate(w):
                        sl = slice(cu[j], cu[j + 1])
                        outs[l][f"O2[{k}]"], outs[l][f"LSE2[{k}]"] = O2[sl].clone(), LSE2[:, sl].clone()
                        outs[l][f"dQ2[{k}]"], outs[l][f"dK2[{k}]"], outs[l][f"dV2[{k}]"] = (
                            dQ2[sl].clone(), dK2[sl].clone(), dV2[sl].clone())
                del Q2, K2, V2, dO2, O2, dQ2, dK2, dV2, LSE2
        peak_b = torch.cuda.max_memory_allocated(dev)

        # ---- Phase C in reverse layer order, prefetching one layer ahead
        if offload and "bufs" not in dorm[L - 1]:
            prefetch(L - 1)
        for l in range(L - 1, -1, -1):
            if offload:
                if "bufs" not in dorm[l]:
                    prefetch(l)                       # demand load: nobody prefetched this layer
                b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                b0.record(main)
                main.wait_event(dorm[l]["landed"])
                b1.record(main)
                exposed.append((b0, b1))
                if l > 0:
                    prefetch(l - 1)                   # overlaps Phase C of layer l
                Q1, O1, LSE1 = (dorm[l]["bufs"][k] for k in ("Q1", "O1", "LSE1"))
            else:
                Q1, O1, LSE1 = (dorm[l][k] for k in ("Q1", "O1", "LSE1"))
            dO1 = layers[l].dO1.to(dev)
            dQ1, dK1, dV1 = e(Lp, Hq), e(Lp, Hkv), e(Lp, Hkv)
            pf.pf_phaseC_bwd(grp[l], Q1, O1, LSE1, dO1, dQ1, dK1, dV1, main)
            if keep_outputs:
                outs[l].update(dQ1=dQ1, dK1=dK1, dV1=dV1)
            dorm[l] = None
            hot[l] = None
            del Q1, O1, LSE1, dO1, dQ1, dK1, dV1
    finally:
        for g in grp:
            pf.pf_group_end(g)
    t1.record(main)
    torch.cuda.synchronize(dev)
    return dict(ms=t0.elapsed_time(t1), layers=L,
                peak_step_bytes=max(peak_a, peak_b, torch.cuda.max_memory_allocated(dev)),
                peak_phaseB_bytes=peak_b, resident_at_phaseB_start_bytes=base,
                exposed_prefetch_ms=sum(a.elapsed_time(b) for a, b in exposed), outputs=outs)


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
