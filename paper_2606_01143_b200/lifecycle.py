"""Memory lifecycle of the training-time KV cache over L attention layers.

Per layer the HOT set {K1, V1, gK1, gV1} stays in HBM from Phase A to the end of Phase C; the
DORMANT Phase-A set {Q1, O1, LSE1} is only needed again by Phase C, so it leaves for a pinned host
pool on a side stream as soon as Phase A has produced it and is prefetched back one layer ahead of
Phase C ("the pool is sized at about 1.5x the measured Phase-A saved-tensor footprint
... prefetch falls back to demand-load when HBM headroom is short, so correctness never depends on
overlap").  Suffix-wave tensors live only during their wave.

Host-side orchestration only: device memory comes from torch's caching allocator, copies and
kernels go through the C ABI (`pf_offload`, `pf_prefetch`, `pf_phase*`).  Nothing here synchronises
the host with the main stream; the one host wait (`offload="wait"`) is on the LAST offload copy's
event, because torch's allocator can only hand freed blocks to later allocations once the host has
seen the copy complete (a block freed behind `record_stream` stays allocated until its event has
been observed).  `offload="overlap"` never waits: the dormant buffers are released at the first wave
boundary at which their copy is seen complete, so the first waves of Phase B run beside the copy and
still see the dormant set in HBM.
"""
from __future__ import annotations

import dataclasses
from typing import Dict, List, Optional, Sequence

import torch

from . import binding as pf
from .schedule import _waves


class PinnedPool:
    """One pinned host allocation carved into 256-byte aligned blocks (bump allocation, reset per
    step).  `alloc` returns None when the pool is full: the caller then keeps that tensor in HBM."""

    def __init__(self, capacity_bytes: int):
        self.capacity = int(capacity_bytes)
        self.buf = torch.empty(max(1, self.capacity), dtype=torch.uint8, pin_memory=True)
        self.offset = 0
        self.high_water = 0

    def alloc(self, nbytes: int) -> Optional[torch.Tensor]:
        start = (self.offset + 255) // 256 * 256
        if start + nbytes > self.capacity:
            return None
        self.offset = start + nbytes
        self.high_water = max(self.high_water, self.offset)
        return self.buf[start:start + nbytes]

    def reset(self) -> None:
        self.offset = 0


def dormant_bytes(shape) -> int:
    """{Q1, O1} bf16 [Lp, Hq, d] + LSE1 fp32 [Hq, Lp] of one layer."""
    return 2 * shape.Lp * shape.n_q_heads * shape.head_dim * 2 + shape.n_q_heads * shape.Lp * 4


class RandomSource:
    """Layer inputs drawn on the device when the schedule asks for them, as if the preceding
    projection had just produced them (timing and memory runs: values do not matter, shapes do).
    N(0,1)/sqrt(d) -> bf16, seeded per (layer, tensor)."""

    def __init__(self, shape, n_layers: int, device, seed: int = 0):
        self.shape, self.n_layers, self.dev, self.seed = shape, n_layers, torch.device(device), seed
        self.gen = torch.Generator(device=self.dev)

    def _draw(self, key: int, L: int, H: int) -> torch.Tensor:
        self.gen.manual_seed(self.seed * 1000003 + key)
        x = torch.randn((L, H, self.shape.head_dim), generator=self.gen, device=self.dev, dtype=torch.float32)
        return (x * self.shape.head_dim ** -0.5).to(torch.bfloat16)

    def prefix(self, l: int):
        s = self.shape
        return (self._draw(16 * l, s.Lp, s.n_q_heads), self._draw(16 * l + 1, s.Lp, s.n_kv_heads),
                self._draw(16 * l + 2, s.Lp, s.n_kv_heads))

    def dO1(self, l: int):
        return self._draw(16 * l + 3, self.shape.Lp, self.shape.n_q_heads)

    def wave(self, l: int, w: Sequence[int]):
        s = self.shape
        tot = sum(s.Ls[k] for k in w)
        base = 16 * l + 4 + 4096 * (w[0] + 1)
        return (self._draw(base, tot, s.n_q_heads), self._draw(base + 1, tot, s.n_kv_heads),
                self._draw(base + 2, tot, s.n_kv_heads), self._draw(base + 3, tot, s.n_q_heads))


class HostSource:
    """Layer inputs uploaded from `inputs.GroupInputs` (parity tests: the oracle sees the same bits)."""

    def __init__(self, layers, device):
        self.layers, self.dev = list(layers), torch.device(device)
        self.shape, self.n_layers = self.layers[0].shape, len(self.layers)

    def prefix(self, l: int):
        i = self.layers[l]
        return i.Q1.to(self.dev), i.K1.to(self.dev), i.V1.to(self.dev)

    def dO1(self, l: int):
        return self.layers[l].dO1.to(self.dev)

    def wave(self, l: int, w: Sequence[int]):
        i = self.layers[l]
        cat = lambda src: torch.cat([src[k] for k in w], 0).contiguous().to(self.dev)
        return cat(i.Q2), cat(i.K2), cat(i.V2), cat(i.dO2)


@dataclasses.dataclass
class _Dormant:
    """The Phase-A set of one layer while it is away (or on its way)."""
    dev: Optional[Dict[str, torch.Tensor]]      # device copies (None once released)
    host: Dict[str, torch.Tensor]               # pool blocks (empty dict: kept resident)
    meta: Dict[str, tuple]
    nbytes: int = 0
    copied: Optional[torch.cuda.Event] = None   # D2H finished
    back: Optional[Dict[str, torch.Tensor]] = None
    landed: Optional[torch.cuda.Event] = None   # H2D finished


def run_layers(ctx, source, device="cuda", wave: int = 1, offload: str = "wait",
               pool: Optional[PinnedPool] = None, keep_outputs: bool = False,
               early_prefetch: bool = False, hbm_headroom_bytes: int = 0,
               side: Optional[torch.cuda.Stream] = None) -> dict:
    """One A -> B -> C step over `source.n_layers` attention layers (each with its own
    training-time KV cache), allocating and freeing device tensors the way a trainer would.

    offload: "none"    - the dormant sets stay in HBM (the baseline);
             "wait"    - they leave behind Phase A on the side stream; the host waits for the last
                         copy before Phase B is enqueued (exposed: `exposed_offload_ms`), so every
                         wave of Phase B runs with the dormant sets out of HBM;
             "overlap" - no wait: buffers are released at the first wave boundary that sees their
                         copy complete.
    Prefetch: the dormant set of layer l-1 comes back on the side stream while Phase C of layer l
    computes (`early_prefetch`: the first one is issued behind the last Phase-B wave).  If the device
    buffers for an early prefetch do not fit under `hbm_headroom_bytes` of free HBM the load is done
    on demand, right before the layer's Phase C (exposed).
    Returns times, peaks (torch.cuda.max_memory_allocated, "CUDA allocated HBM") and,
    with keep_outputs, every output per layer."""
    assert offload in ("none", "wait", "overlap")
    s = source.shape
    dev = torch.device(device)
    Hq, Hkv, d, Lp, L = s.n_q_heads, s.n_kv_heads, s.head_dim, s.Lp, source.n_layers
    bf, f32 = torch.bfloat16, torch.float32
    main = torch.cuda.current_stream(dev)
    side = side or torch.cuda.Stream(dev)
    e = lambda n, H, dt=bf: torch.empty((n, H, d), dtype=dt, device=dev)
    waves = _waves(s.N, wave)
    max_tok = max((sum(s.Ls[k] for k in w) for w in waves), default=0)
    desc = pf.make_desc(Hq, Hkv, d)
    if pool is not None:
        pool.reset()
    ev = lambda timing=False: torch.cuda.Event(enable_timing=timing)

    torch.cuda.synchronize(dev)
    torch.cuda.reset_peak_memory_stats(dev)
    t0, t1 = ev(True), ev(True)
    t0.record(main)
    ws = torch.empty(pf.pf_workspace_bytes(desc, Lp, max_tok), dtype=torch.uint8, device=dev)
    hot, dorm, grp, outs = [], [], [], [dict() for _ in range(L)]
    exposed_pre, kept_resident, demand_loads = [], 0, 0
    exposed_off = None

    def release_copied(block: bool) -> None:
        """Drop the device copies of dormant sets whose D2H copy the host has seen complete."""
        for ds in dorm:
            if ds.dev is not None and ds.copied is not None:
                if block:
                    ds.copied.synchronize()
                if ds.copied.query():
                    ds.dev = None

    def prefetch(l: int) -> None:
        ds = dorm[l]
        if ds.dev is not None or ds.back is not None:     # still (or already) in HBM
            return
        gate = ev(); gate.record(main)                    # fresh buffers may reuse blocks main still reads
        ds.back = {k: torch.empty(sh, dtype=dt, device=dev) for k, (sh, dt) in ds.meta.items()}
        side.wait_event(gate)
        for k, t in ds.back.items():
            pf.pf_prefetch(ctx, ds.host[k].view(t.dtype)[:t.numel()].view(t.shape), t, side)
        ds.landed = ev(); ds.landed.record(side)

    def fits_early(l: int) -> bool:
        need = dorm[l].nbytes
        free, _ = torch.cuda.mem_get_info(dev)
        cached = torch.cuda.memory_reserved(dev) - torch.cuda.memory_allocated(dev)
        return free + cached - need >= hbm_headroom_bytes

    try:
        # ---- Phase A, layer by layer; each dormant set streams out behind it
        for l in range(L):
            Q1, K1, V1 = source.prefix(l)
            O1 = e(Lp, Hq); LSE1 = torch.empty((Hq, Lp), dtype=f32, device=dev)
            gK1, gV1 = e(Lp, Hkv, f32), e(Lp, Hkv, f32)
            g = pf.pf_group_begin(ctx, desc, Lp, K1, V1, gK1, gV1, ws, main)
            grp.append(g)
            pf.pf_phaseA_fwd(g, Q1, O1, LSE1, main)
            hot.append(dict(K1=K1, V1=V1, gK1=gK1, gV1=gV1))
            if keep_outputs:
                outs[l]["O1"], outs[l]["LSE1"] = O1.clone(), LSE1.clone()
            dset = dict(Q1=Q1, O1=O1, LSE1=LSE1)
            ds = _Dormant(dev=dset, host={}, meta={k: (t.shape, t.dtype) for k, t in dset.items()},
                          nbytes=sum(t.numel() * t.element_size() for t in dset.values()))
            if offload != "none":
                blocks = {k: (pool.alloc(t.numel() * t.element_size()) if pool is not None else
                              torch.empty(t.numel() * t.element_size(), dtype=torch.uint8, pin_memory=True))
                          for k, t in dset.items()}
                if any(b is None for b in blocks.values()):
                    kept_resident += sum(t.numel() * t.element_size() for t in dset.values())   # pool full
                else:
                    produced = ev(); produced.record(main)
                    side.wait_event(produced)
                    for k, t in dset.items():
                        pf.pf_offload(ctx, t, blocks[k], side)
                        t.record_stream(side)
                    ds.host = blocks
                    ds.copied = ev(); ds.copied.record(side)
            dorm.append(ds)
            del Q1, O1, LSE1, dset
        if offload == "wait":
            a0, a1 = ev(True), ev(True)
            a0.record(main)
            release_copied(block=True)                 # host waits for the copies (not for `main`)
            last = [ds.copied for ds in dorm if ds.copied is not None]
            if last:
                main.wait_event(last[-1])
            a1.record(main)
            exposed_off = (a0, a1)
        peak_a = torch.cuda.max_memory_allocated(dev)
        torch.cuda.reset_peak_memory_stats(dev)
        base = torch.cuda.memory_allocated(dev)

        # ---- Phase B: every wave on every layer (a wave's tensors live only during the wave)
        gone_from, peak_b_head = None, 0
        for wi, w in enumerate(waves):
            if offload == "overlap" and gone_from is None:
                release_copied(block=False)
                if all(ds.dev is None or ds.copied is None for ds in dorm):
                    peak_b_head = torch.cuda.max_memory_allocated(dev)   # peak of the waves that ran beside the copies
                    torch.cuda.reset_peak_memory_stats(dev)              # from here on the dormant sets are gone
                    gone_from = wi
            if early_prefetch and offload != "none" and wi == len(waves) - 1 and fits_early(L - 1):
                prefetch(L - 1)                        # hidden behind the last wave (costs its buffers in the peak)
            cu = [0]
            for k in w:
                cu.append(cu[-1] + s.Ls[k])
            tot = cu[-1]
            for l in range(L):
                Q2, K2, V2, dO2 = source.wave(l, w)
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
        peak_b_tail = torch.cuda.max_memory_allocated(dev)
        peak_b = max(peak_b_head, peak_b_tail)
        if offload == "overlap":
            release_copied(block=True)                 # Phase C needs the bookkeeping settled

        # ---- Phase C in reverse layer order, prefetching one layer ahead
        for l in range(L - 1, -1, -1):
            ds = dorm[l]
            if ds.dev is None and ds.back is None:
                demand_loads += 1                      # nobody prefetched this layer: load it now (exposed)
                prefetch(l)
            if ds.back is not None:
                b0, b1 = ev(True), ev(True)
                b0.record(main)
                main.wait_event(ds.landed)
                b1.record(main)
                exposed_pre.append((b0, b1))
                cur = ds.back
            else:
                cur = ds.dev
            if l > 0 and offload != "none" and fits_early(l - 1):
                prefetch(l - 1)                        # overlaps Phase C of layer l
            dO1 = source.dO1(l)
            dQ1, dK1, dV1 = e(Lp, Hq), e(Lp, Hkv), e(Lp, Hkv)
            pf.pf_phaseC_bwd(grp[l], cur["Q1"], cur["O1"], cur["LSE1"], dO1, dQ1, dK1, dV1, main)
            if keep_outputs:
                outs[l].update(dQ1=dQ1, dK1=dK1, dV1=dV1)
            dorm[l] = _Dormant(dev=None, host={}, meta={})
            hot[l] = None
            del cur, ds, dO1, dQ1, dK1, dV1
    finally:
        for g in grp:
            pf.pf_group_end(g)
    t1.record(main)
    torch.cuda.synchronize(dev)
    res = dict(ms=t0.elapsed_time(t1), layers=L, offload=offload,
               peak_step_bytes=max(peak_a, peak_b, torch.cuda.max_memory_allocated(dev)),
               peak_phaseB_bytes=peak_b, resident_at_phaseB_start_bytes=base,
               exposed_prefetch_ms=sum(a.elapsed_time(b) for a, b in exposed_pre),
               exposed_offload_ms=exposed_off[0].elapsed_time(exposed_off[1]) if exposed_off else 0.0,
               kept_resident_bytes=kept_resident, demand_loads=demand_loads,
               pool_bytes=pool.capacity if pool is not None else None,
               pool_high_water_bytes=pool.high_water if pool is not None else None,
               outputs=outs)
    if offload == "overlap":
        res["dormant_gone_from_wave"] = gone_from       # None: the copies outlasted Phase B
        res["peak_phaseB_after_offload_bytes"] = peak_b_tail if gone_from is not None else None
    return res
