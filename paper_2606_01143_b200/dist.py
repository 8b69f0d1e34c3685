"""Multi-GPU execution of the path: one process per GPU, `torch.distributed` (NCCL on GPUs, gloo in
the CPU tests) for the plumbing.

Three ways the path shards:

  groups   whole rollout groups on different GPUs are independent: weak scaling, no
           data-path collective; the only collectives are the timing barrier and a MAX over ranks.
  heads    ONE group sharded by KV head -- the paper's TP rule ("each rank caches
           its own head shard"): every phase runs on the rank's heads only, zero communication.
  split    ONE group with Phase B sharded by SUFFIX -- the paper's CP rule / DP split-group fallback
           ("exchanges only compact prefix K/V plus the corresponding
           prefix-side gK/gV"): Phase A and Phase C are head-sharded; between them
               all-gather     K1, V1  (bf16 [Lp, Hkv, d])       after Phase A
               Phase B        the rank's suffixes on ALL heads into a local fp32 gK1/gV1
               reduce-scatter gK1, gV1 (fp32) over the KV-head dimension, back to the head owners
           With several layers the collectives run on a communication stream: layer l+1's all-gather
           and layer l-1's reduce-scatter overlap layer l's Phase B.

`SplitGroupRank` holds one rank's tensors and issues its C-ABI calls; the collectives are injected
(`DistComm` = torch.distributed, `LocalComm` = all ranks in one process, used to run the exact
per-rank schedule on a single GPU in the tests).
"""
from __future__ import annotations

import copy
import dataclasses
from typing import List, Optional, Sequence

import torch
import torch.distributed as dist

RANK_SEED_STRIDE = 100000


# ------------------------------------------------------------------------------------------------
# groups: weak scaling
# ------------------------------------------------------------------------------------------------
def rank_shape(shape, rank: int):
    """Rank r draws its own rollout group: same shapes, seed shifted by r * RANK_SEED_STRIDE."""
    s = copy.deepcopy(shape)
    s.seed = shape.seed + RANK_SEED_STRIDE * int(rank)
    return s


def max_over_ranks(value: float, device=None) -> float:
    """MAX over ranks of a per-rank scalar (the timed milliseconds); identity when not distributed."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank: float, ms_max: float, world: int) -> float:
    """Whole-job throughput: units all ranks processed / the slowest rank's time."""
    return world * units_per_rank / (ms_max * 1e-3)


# ------------------------------------------------------------------------------------------------
# plan of a sharded group (host side, no tensors)
# ------------------------------------------------------------------------------------------------
@dataclasses.dataclass
class SplitPlan:
    world: int
    rank: int
    kv_heads: range        # KV heads this rank owns (Phase A, Phase C, head sharding)
    q_heads: range         # their query heads: kappa^-1(kv_heads)
    suffixes: List[int]    # suffixes whose Phase B this rank runs ("split" mode)


def split_plan(shape, world: int, rank: int) -> SplitPlan:
    """KV heads in contiguous blocks of Hkv / world; suffixes by longest-processing-time-first onto
    the least loaded rank (cost of suffix i ~ Ls_i * Lp + Ls_i^2 / 2 attended pairs), ties to the
    lower rank -- deterministic, identical on every rank."""
    Hkv, G = shape.n_kv_heads, shape.G
    if world < 1 or not 0 <= rank < world:
        raise ValueError(f"rank {rank} outside world {world}")
    if Hkv % world != 0:
        raise ValueError(f"{Hkv} KV heads do not shard over {world} ranks")
    per = Hkv // world
    kv = range(rank * per, (rank + 1) * per)
    cost = lambda i: shape.Ls[i] * shape.Lp + shape.Ls[i] * (shape.Ls[i] + 1) // 2
    load = [0] * world
    owner = {}
    for i in sorted(range(shape.N), key=lambda i: (-cost(i), i)):
        r = min(range(world), key=lambda r: (load[r], r))
        owner[i] = r
        load[r] += cost(i)
    return SplitPlan(world, rank, kv, range(kv.start * G, kv.stop * G),
                     sorted(i for i, r in owner.items() if r == rank))


# ------------------------------------------------------------------------------------------------
# the two exchanges of "split" mode
# ------------------------------------------------------------------------------------------------
class DistComm:
    """Collectives of the split-group schedule through torch.distributed (NCCL or gloo)."""

    def __init__(self, group=None):
        self.group = group
        self.world = dist.get_world_size(group)
        self.rank = dist.get_rank(group)

    def all_gather_heads(self, shard: torch.Tensor) -> torch.Tensor:
        """[L, H/world, d] per rank -> [L, H, d] (rank r's heads at r * H/world)."""
        shard = shard.contiguous()
        parts = [torch.empty_like(shard) for _ in range(self.world)]
        dist.all_gather(parts, shard, group=self.group)
        return torch.cat(parts, 1)

    def reduce_scatter_heads(self, full: torch.Tensor, out: Optional[torch.Tensor] = None) -> torch.Tensor:
        """SUM over ranks of [L, H, d] fp32, each rank keeping its own H/world heads."""
        per = full.shape[1] // self.world
        if dist.get_backend(self.group) == "nccl":
            chunks = full.view(full.shape[0], self.world, per, full.shape[2]).permute(1, 0, 2, 3).contiguous()
            res = torch.empty_like(chunks[0]) if out is None else out
            dist.reduce_scatter_tensor(res, chunks, op=dist.ReduceOp.SUM, group=self.group)
            return res
        tmp = full.clone()                      # gloo has no reduce-scatter: all-reduce, then slice
        dist.all_reduce(tmp, op=dist.ReduceOp.SUM, group=self.group)
        res = tmp[:, self.rank * per:(self.rank + 1) * per].contiguous()
        if out is not None:
            out.copy_(res)
            return out
        return res


class LocalComm:
    """All ranks of a split group inside ONE process: `gather` / `scatter` take the per-rank tensors
    of every rank at once.  Lets the tests drive the exact per-rank schedule on a single GPU."""

    def __init__(self, world: int):
        self.world = world

    def all_gather_heads(self, shards: Sequence[torch.Tensor]) -> List[torch.Tensor]:
        full = torch.cat([s.contiguous() for s in shards], 1)
        return [full for _ in range(self.world)]

    def reduce_scatter_heads(self, fulls: Sequence[torch.Tensor]) -> List[torch.Tensor]:
        total = torch.stack(list(fulls), 0).sum(0)
        per = total.shape[1] // self.world
        return [total[:, r * per:(r + 1) * per].contiguous() for r in range(self.world)]


# ------------------------------------------------------------------------------------------------
# one rank of a split group on its GPU
# ------------------------------------------------------------------------------------------------
class SplitGroupRank:
    """Device tensors and C-ABI calls of one rank for one layer of a split group.

    The rank holds the prefix tensors of ITS heads only (Q1, K1, V1, dO1 head slices) and the suffix
    tensors of ITS suffixes on all heads.  Call order: phase_a() -> [all-gather K1, V1] ->
    phase_b(K1_full, V1_full) -> [reduce-scatter gK1, gV1] -> phase_c(gK1_shard, gV1_shard)."""

    def __init__(self, ctx, inp, plan: SplitPlan, device="cuda", wave: int = 0, stream=None):
        from . import binding as pf
        from . import schedule
        self.pf, self.ctx, self.plan, self.stream = pf, ctx, plan, stream
        s = inp.shape
        self.shape = s
        dev = torch.device(device)
        kv, qh = plan.kv_heads, plan.q_heads
        mv = lambda t: t.contiguous().to(dev)
        self.Q1, self.dO1 = mv(inp.Q1[:, qh.start:qh.stop]), mv(inp.dO1[:, qh.start:qh.stop])
        self.K1, self.V1 = mv(inp.K1[:, kv.start:kv.stop]), mv(inp.V1[:, kv.start:kv.stop])
        Lp, d = s.Lp, s.head_dim
        self.nq, self.nkv = len(qh), len(kv)
        bf, f32 = torch.bfloat16, torch.float32
        e = lambda L, H, dt=bf: torch.empty((L, H, d), dtype=dt, device=dev)
        self.O1, self.LSE1 = e(Lp, self.nq), torch.empty((self.nq, Lp), dtype=f32, device=dev)
        self.gK1s, self.gV1s = e(Lp, self.nkv, f32), e(Lp, self.nkv, f32)      # own heads: Phase C accumulators
        self.dQ1, self.dK1, self.dV1 = e(Lp, self.nq), e(Lp, self.nkv), e(Lp, self.nkv)
        # Phase B of the rank's suffixes on all heads, packed `wave` per call (0: all in one wave)
        self.idx = list(plan.suffixes)
        b = len(self.idx) if wave <= 0 else wave
        self.waves = [self.idx[i:i + b] for i in range(0, len(self.idx), max(1, b))]
        self.pk = []
        max_tok = 0
        for w in self.waves:
            cu = [0]
            for k in w:
                cu.append(cu[-1] + s.Ls[k])
            cat = lambda src: torch.cat([src[k] for k in w], 0).contiguous().to(dev)
            pk = dict(cu=cu, idx=w, Q2=cat(inp.Q2), K2=cat(inp.K2), V2=cat(inp.V2), dO2=cat(inp.dO2))
            tot = cu[-1]
            max_tok = max(max_tok, tot)
            pk.update(O2=e(tot, s.n_q_heads), dQ2=e(tot, s.n_q_heads), dK2=e(tot, s.n_kv_heads),
                      dV2=e(tot, s.n_kv_heads), LSE2=torch.empty((s.n_q_heads, tot), dtype=f32, device=dev))
            self.pk.append(pk)
        self.gK1f, self.gV1f = e(Lp, s.n_kv_heads, f32), e(Lp, s.n_kv_heads, f32)   # local sums over own suffixes
        self.desc_s = pf.make_desc(self.nq, self.nkv, d)
        self.desc_f = pf.make_desc(s.n_q_heads, s.n_kv_heads, d)
        self.ws_s = torch.empty(pf.pf_workspace_bytes(self.desc_s, Lp, 0), dtype=torch.uint8, device=dev)
        self.ws_f = torch.empty(pf.pf_workspace_bytes(self.desc_f, 0, max_tok), dtype=torch.uint8, device=dev)
        self.grp_s = None

    def phase_a(self) -> None:
        """Head-sharded Phase A; the group stays open for Phase C (its accumulators are zeroed here)."""
        pf = self.pf
        self.grp_s = pf.pf_group_begin(self.ctx, self.desc_s, self.shape.Lp, self.K1, self.V1, self.gK1s,
                                       self.gV1s, self.ws_s, self.stream)
        pf.pf_phaseA_fwd(self.grp_s, self.Q1, self.O1, self.LSE1, self.stream)

    def phase_b(self, K1_full: torch.Tensor, V1_full: torch.Tensor) -> None:
        """Phase B of the rank's suffixes against the gathered prefix K/V; gK1f/gV1f = their sum."""
        pf = self.pf
        grp = pf.pf_group_begin(self.ctx, self.desc_f, self.shape.Lp, K1_full, V1_full, self.gK1f, self.gV1f,
                                self.ws_f, self.stream)
        try:
            pf.pf_group_mark_cached(grp)
            for pk in self.pk:
                pf.pf_phaseB_fwd(grp, pk["cu"], pk["Q2"], pk["K2"], pk["V2"], pk["O2"], pk["LSE2"], self.stream)
                pf.pf_phaseB_bwd(grp, pk["cu"], pk["Q2"], pk["K2"], pk["V2"], pk["O2"], pk["LSE2"], pk["dO2"],
                                 pk["dQ2"], pk["dK2"], pk["dV2"], self.stream)
        finally:
            pf.pf_group_end(grp)

    def phase_c(self, gK1_shard: torch.Tensor, gV1_shard: torch.Tensor) -> None:
        """Head-sharded Phase C with the reduced coupling gradients of the rank's heads injected."""
        pf = self.pf
        if gK1_shard.data_ptr() != self.gK1s.data_ptr():
            self.gK1s.copy_(gK1_shard)
            self.gV1s.copy_(gV1_shard)
        try:
            pf.pf_phaseC_bwd(self.grp_s, self.Q1, self.O1, self.LSE1, self.dO1, self.dQ1, self.dK1, self.dV1,
                             self.stream)
        finally:
            pf.pf_group_end(self.grp_s)
            self.grp_s = None


def run_split_group_local(ctx, inp, world: int, device="cuda", wave: int = 0) -> List[SplitGroupRank]:
    """The split-group schedule of all `world` ranks on ONE device, rank after rank, with `LocalComm`
    standing in for the collectives: the same per-rank calls, buffers and plan as the distributed run."""
    comm = LocalComm(world)
    ranks = [SplitGroupRank(ctx, inp, split_plan(inp.shape, world, r), device, wave) for r in range(world)]
    for r in ranks:
        r.phase_a()
    K1f = comm.all_gather_heads([r.K1 for r in ranks])
    V1f = comm.all_gather_heads([r.V1 for r in ranks])
    for r, k, v in zip(ranks, K1f, V1f):
        r.phase_b(k, v)
    gk = comm.reduce_scatter_heads([r.gK1f for r in ranks])
    gv = comm.reduce_scatter_heads([r.gV1f for r in ranks])
    for r, a, b in zip(ranks, gk, gv):
        r.phase_c(a, b)
    return ranks


def run_split_group_step(rank: SplitGroupRank, comm: DistComm, comm_stream=None) -> dict:
    """One rank's step of a split group with real collectives.  With a `comm_stream` the exchanges
    are enqueued there and ordered against the compute stream by events (the building block of the
    multi-layer overlap: a caller that interleaves several layers issues layer l+1's all-gather
    before layer l's Phase B).  Returns the events that bracket what the compute stream waited for."""
    main = rank.stream if isinstance(rank.stream, torch.cuda.Stream) else torch.cuda.current_stream()
    cs = comm_stream or main
    ev = lambda: torch.cuda.Event(enable_timing=True)
    rank.phase_a()
    a_done = ev(); a_done.record(main)
    cs.wait_event(a_done)
    with torch.cuda.stream(cs):
        K1f = comm.all_gather_heads(rank.K1)
        V1f = comm.all_gather_heads(rank.V1)
        g_done = ev(); g_done.record(cs)
    w0 = ev(); w0.record(main)
    main.wait_event(g_done)
    w1 = ev(); w1.record(main)
    rank.phase_b(K1f, V1f)
    b_done = ev(); b_done.record(main)
    cs.wait_event(b_done)
    with torch.cuda.stream(cs):
        comm.reduce_scatter_heads(rank.gK1f, out=rank.gK1s)
        comm.reduce_scatter_heads(rank.gV1f, out=rank.gV1s)
        r_done = ev(); r_done.record(cs)
    w2 = ev(); w2.record(main)
    main.wait_event(r_done)
    w3 = ev(); w3.record(main)
    rank.phase_c(rank.gK1s, rank.gV1s)
    return dict(gather_wait=(w0, w1), reduce_wait=(w2, w3))


class SelfComm:
    """world = 1: the collectives of `DistComm` as identities (a copy), with the same signatures.
    Lets the stream / event schedule of the multi-layer step run on one GPU without a process group."""
    world, rank = 1, 0

    def all_gather_heads(self, shard: torch.Tensor) -> torch.Tensor:
        return shard.clone()

    def reduce_scatter_heads(self, full: torch.Tensor, out: Optional[torch.Tensor] = None) -> torch.Tensor:
        if out is None:
            return full.clone()
        out.copy_(full)
        return out


def run_split_group_layers(layers: Sequence[SplitGroupRank], comm, comm_stream: torch.cuda.Stream) -> dict:
    """One rank's step over L attention layers of a split group with the exchanges overlapped
    ("next-layer K/V gathers and previous-layer gK/gV reductions are prefetched on a
    communication stream", :310): Phase A runs layer by layer and each layer's K1/V1 all-gather is
    enqueued on `comm_stream` right behind it -- it travels under the Phase A of the later layers and
    the Phase B of the earlier ones; each layer's gK1/gV1 reduce-scatter is enqueued right behind its
    Phase B and travels under the Phase B of the later layers; Phase C runs in reverse layer order
    and waits only for its own layer's reduction.  `layers[l]` holds the rank's tensors of layer l.
    Returns the milliseconds the compute stream spent waiting for a gather / a reduction (exposed
    communication) once the caller has synchronised."""
    main = layers[0].stream if isinstance(layers[0].stream, torch.cuda.Stream) else torch.cuda.current_stream()
    ev = lambda: torch.cuda.Event(enable_timing=True)
    gathered, g_done, r_done, waits = [], [], [], []
    for rk in layers:                                          # Phase A + gather behind it
        rk.phase_a()
        a = ev(); a.record(main)
        comm_stream.wait_event(a)
        with torch.cuda.stream(comm_stream):
            gathered.append((comm.all_gather_heads(rk.K1), comm.all_gather_heads(rk.V1)))
            e = ev(); e.record(comm_stream)
        g_done.append(e)
    for l, rk in enumerate(layers):                            # Phase B + reduction behind it
        w0 = ev(); w0.record(main)
        main.wait_event(g_done[l])
        w1 = ev(); w1.record(main)
        waits.append(("gather", l, w0, w1))
        K1f, V1f = gathered[l]
        K1f.record_stream(main); V1f.record_stream(main)
        rk.phase_b(K1f, V1f)
        b = ev(); b.record(main)
        comm_stream.wait_event(b)
        with torch.cuda.stream(comm_stream):
            comm.reduce_scatter_heads(rk.gK1f, out=rk.gK1s)
            comm.reduce_scatter_heads(rk.gV1f, out=rk.gV1s)
            e = ev(); e.record(comm_stream)
        r_done.append(e)
    for l in range(len(layers) - 1, -1, -1):                   # Phase C, reverse layer order
        w0 = ev(); w0.record(main)
        main.wait_event(r_done[l])
        w1 = ev(); w1.record(main)
        waits.append(("reduce", l, w0, w1))
        layers[l].phase_c(layers[l].gK1s, layers[l].gV1s)
    return dict(waits=waits,
                exposed_ms=lambda: {k: sum(a.elapsed_time(b) for kind, _, a, b in waits if kind == k)
                                    for k in ("gather", "reduce")})
