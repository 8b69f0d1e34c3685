#!/usr/bin/env python
"""bench.py -- one B200 (or N independent ranks): the A -> B(xN) -> C attention step of PrefixFlow's
training-time KV cache through the C ABI, against the build's own N-times replay baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 7b|ragged|32k|sweep-rR-nN|tiny]
    python bench.py --impl reference ...      # times the fp64 CPU oracle on a bounded sample

A "step" is one pass of the whole hot path over one synthetic rollout group (SURVEY.md §8a rows
a1-a4): pf_group_begin, pf_phaseA_fwd, N x (pf_phaseB_fwd, pf_phaseB_bwd), pf_phaseC_bwd.
Prints ONE JSON line (rank 0).  Keys follow the driver's contract; DESIGN.md "Measurement" explains
every number.  Nothing here reads /root/reference; every input is seeded and synthetic
(paper_2606_01143_b200/inputs.py).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = ("A+B+C attention step throughput (algorithmic TFLOP/s; step time vs N-times replay and "
          "Phase-B TFLOP/s / % of BF16 peak in extra keys)")
UNIT = "TFLOP/s"
L2_BYTES = 126 * 2 ** 20


# --------------------------------------------------------------------------------------------------
# algorithmic work (fwd = 4 d pairs Hq, bwd = 10 d pairs Hq; tile padding not counted)
# --------------------------------------------------------------------------------------------------
def tri(L: int) -> int:
    return L * (L + 1) // 2


def flops(shape) -> dict:
    Hq, d, Lp = shape.n_q_heads, shape.head_dim, shape.Lp
    pa = tri(Lp)
    pb = [Ls * Lp + tri(Ls) for Ls in shape.Ls]
    pr = [tri(Lp + Ls) for Ls in shape.Ls]
    f = dict(A=4 * d * pa * Hq, B_fwd=4 * d * sum(pb) * Hq, B_bwd=10 * d * sum(pb) * Hq,
             C=10 * d * pa * Hq, replay=14 * d * sum(pr) * Hq)
    f["B_bwd_each"] = [10 * d * p * Hq for p in pb]
    f["B_fwd_each"] = [4 * d * p * Hq for p in pb]
    f["step"] = f["A"] + f["B_fwd"] + f["B_bwd"] + f["C"]
    f["ideal_speedup"] = sum(pr) / (pa + sum(pb)) if (pa + sum(pb)) else 1.0
    return f


def pick_config(name: str):
    from paper_2606_01143_b200 import inputs
    if name == "7b":
        return inputs.config_7b()
    if name == "tiny":
        return inputs.config_tiny()
    if name == "ragged":
        return inputs.config_ragged()
    if name == "32k":
        return inputs.config_32k()
    if name.startswith("sweep-r"):
        r, n = name[len("sweep-r"):].split("-n")
        return inputs.config_sweep(int(r), int(n))
    raise SystemExit(f"unknown --config {name}")


def measured_peaks() -> dict:
    """MEASURED_PEAKS.json (driver-written) or the fallback of /opt/skills/guides/B200_PROFILING.md."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            m = json.load(f)
        return dict(burst=float(m["bf16_tflops"]), sustained=float(m["bf16_tflops_sustained"]),
                    hbm=float(m["hbm_gbs"]), source="measured (MEASURED_PEAKS.json)")
    return dict(burst=1590.0, sustained=1400.0, hbm=6650.0, source="fallback (B200_PROFILING.md)")


def ncu_traffic(kernel: str, config: str):
    """dram bytes per launch of `kernel` from the committed ncu --set full summary, else None."""
    p = os.path.join(ROOT, "profiles", "roofline_traffic.csv")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        for line in f:
            parts = [x.strip() for x in line.split(",")]
            if len(parts) >= 3 and parts[0] == kernel and parts[1] == config:
                try:
                    return float(parts[2])
                except ValueError:
                    return None
    return None


# --------------------------------------------------------------------------------------------------
# clocks sampled DURING the timed region (NVML in a thread; nvidia-smi's own start-up is too slow)
# --------------------------------------------------------------------------------------------------
class ClockSampler:
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown",
               0x4: "sw_power_cap", 0x80: "hw_power_brake", 0x2: "applications_clocks_setting"}

    def __init__(self, index: int):
        self.samples, self.reasons, self.power = [], set(), []
        self.max_mhz = None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:  # NVML missing: clocks are reported as null
            self.nv = None

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                for bit, name in self.REASONS.items():
                    if r & bit:
                        self.reasons.add(name)
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            time.sleep(0.005)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self) -> dict:
        if not self.samples:
            return dict(sm_mhz=None, sm_max_mhz=self.max_mhz, reasons=[], samples=0)
        return dict(sm_mhz=statistics.median(self.samples), sm_max_mhz=self.max_mhz,
                    reasons=sorted(self.reasons), samples=len(self.samples),
                    power_w_max=max(self.power) if self.power else None)


# --------------------------------------------------------------------------------------------------
# CPU oracle leg (cpu_baseline and --impl reference): a BOUNDED sample of the same workload
# --------------------------------------------------------------------------------------------------
def oracle_sample(shape, budget_flops: float = 6e11):
    """Phase B forward + backward of (suffix i, KV head g) units -- the G query heads of g: every
    suffix row (O2, LSE2, delta, dQ2) and every key column (gK1/gV1 of the prefix keys, dK2/dV2
    of the suffix keys) -- as many whole units as fit `budget_flops` algorithmic flops (at least
    one; if one unit alone exceeds the budget its key columns are strided).  Returns
    (seconds, algorithmic flops of what was computed, description, threads)."""
    import numpy as np
    import oracle
    from paper_2606_01143_b200 import inputs
    d, G, Lp = shape.head_dim, shape.G, shape.Lp
    units = [(i, g) for i in range(shape.N) for g in range(shape.n_kv_heads)]
    # algorithmic count 14 d per (query, key) pair and head: the row side covers S, PV, dP, dQ (8 d),
    # the column side the S recompute, dK, dV (6 d); the oracle's own extra dP recompute is not counted
    unit_flops = lambda i: 14 * d * (shape.Ls[i] * Lp + tri(shape.Ls[i])) * G
    chosen, acc = [], 0.0
    for (i, g) in units:
        if chosen and acc + unit_flops(i) > budget_flops:
            break
        chosen.append((i, g))
        acc += unit_flops(i)
    stride = 1
    if len(chosen) == 1:
        i = chosen[0][0]
        pairs = shape.Ls[i] * Lp + tri(shape.Ls[i])
        while 8 * d * pairs * G + 6 * d * pairs * G / stride > budget_flops and stride < 64:
            stride *= 2
    inp = inputs.make_group(shape, only_suffixes=sorted({i for i, _ in chosen}))
    done, dt = 0.0, 0.0
    for (i, g) in chosen:
        Ls = shape.Ls[i]
        pj = np.arange(0, Lp, stride, dtype=np.int64)
        sj = np.arange(0, Ls, stride, dtype=np.int64)
        t0 = time.perf_counter()
        oracle.sampled_phaseB(inp, i, g, pj, sj)
        dt += time.perf_counter() - t0
        col_pairs = int(len(pj) * Ls + sum(Ls - j for j in sj))
        done += 8 * d * (Ls * Lp + tri(Ls)) * G + 6 * d * col_pairs * G
    desc = (f"oracle/ fp64 (C, OpenMP), Phase B fwd+bwd of {len(chosen)} (suffix, KV head) units "
            f"[{chosen[0]}..{chosen[-1]}] x {G} q-heads: all suffix rows + every "
            f"{'' if stride == 1 else str(stride) + '-th '}key column = "
            f"{done / flops(shape)['step'] * 100:.2f}% of a step's algorithmic flops")
    return dt, float(done), desc, oracle.max_threads()


def run_reference(args, rank: int) -> None:
    if rank != 0:
        return
    shape = pick_config(args.config)
    times, work, desc, thr = [], 0.0, "", 0
    # bound the whole run to ~1.2e12 algorithmic flops (a few minutes of host time)
    budget = min(args.cpu_budget, 1.2e12 / max(1, args.warmup + args.steps))
    for i in range(args.warmup + args.steps):
        dt, work, desc, thr = oracle_sample(shape, budget)
        if i >= args.warmup:
            times.append(dt)
    ms = 1e3 * sum(times) / len(times)
    val = work / (ms * 1e-3) / 1e12
    out = dict(metric=METRIC, value=val, unit=UNIT, n_gpus=args.gpus, steps=args.steps,
               warmup=args.warmup, ms_per_step=ms, higher_is_better=True, scaling="weak",
               vs_baseline=None, dtype="f64", data="synthetic", impl="reference",
               config=workload_config(shape, args.config),
               cpu_baseline=dict(value=val, unit=UNIT, cores=thr, kind="oracle", sample=desc),
               e2e=dict(value=val, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0),
               gpu_launches=0)
    print(json.dumps(out))


def workload_config(shape, name: str) -> dict:
    Ls = shape.Ls
    return dict(workload=f"BASELINE.json configs[{ {'tiny': 0, '7b': 1, 'ragged': 2, '32k': 4}.get(name, 3) }] "
                         f"{shape.name}: {shape.n_q_heads}q/{shape.n_kv_heads}kv heads, d={shape.head_dim}, "
                         f"prefix {shape.Lp}, N={shape.N} suffixes of "
                         f"{Ls[0] if len(set(Ls)) == 1 else f'{min(Ls)}..{max(Ls)}'} tokens "
                         f"({100 * shape.Lp / (shape.Lp + sum(Ls) / max(1, len(Ls))):.0f}% prefix)",
                seed=shape.seed, dist="N(0,1)/sqrt(d) -> bf16", parallelism="1 group per GPU")


# --------------------------------------------------------------------------------------------------
# helper legs of the GPU arm
# --------------------------------------------------------------------------------------------------
def _strip(r: dict) -> dict:
    r = dict(r)
    r.pop("outputs", None)
    return r


def memory_legs(ctx, lifecycle, shape, dev, wave: int, layers: int, reps: int = 2) -> dict:
    """Lifecycle measurement of one layer and of an L-layer pipeline: dormant sets resident
    ("none"), offloaded with Phase B waiting for the copy ("wait": every wave runs with the set out
    of HBM) and offloaded without any wait ("overlap").  Inputs are drawn on the device as the
    schedule asks for them (lifecycle.RandomSource): the times hold no host upload."""
    import torch
    torch.cuda.empty_cache()
    out = dict(wave=wave, dormant_bytes_per_layer=lifecycle.dormant_bytes(shape),
               other_live_bytes_at_start=int(torch.cuda.memory_allocated(dev)),   # counted in every peak below
               note="tensors allocated and freed as a trainer would (suffix-wave tensors live only during their "
                    "wave); peaks are torch.cuda.max_memory_allocated; pinned pool = 1.5x the dormant footprint")
    for L in ([1] + ([layers] if layers > 1 else [])):
        pool = lifecycle.PinnedPool(int(1.5 * L * lifecycle.dormant_bytes(shape)))
        side = torch.cuda.Stream(dev)
        res = {}
        for mode in ("none", "wait", "overlap"):
            for _ in range(reps):
                r = lifecycle.run_layers(ctx, lifecycle.RandomSource(shape, L, dev, seed=7), dev, wave=wave,
                                         offload=mode, pool=pool, side=side, early_prefetch=(mode == "overlap"))
            res[mode] = _strip(r)
            torch.cuda.empty_cache()
        leg = dict(layers=L, resident=res["none"], offload_wait=res["wait"], offload_overlap=res["overlap"],
                   phaseB_peak_reduction_pct=100.0 * (1 - res["wait"]["peak_phaseB_bytes"] / res["none"]["peak_phaseB_bytes"]),
                   ms_ratio_wait=res["wait"]["ms"] / res["none"]["ms"],
                   ms_ratio_overlap=res["overlap"]["ms"] / res["none"]["ms"])
        out["single_layer" if L == 1 else "multilayer"] = leg
        del pool
    return out


def sweep_legs(ctx, schedule, lifecycle, inputs, dev, stream, peaks, steps: int = 3) -> dict:
    """Step time vs the packed replay at the corners of configs[3] and at configs[2] / configs[4]
    (inputs drawn on the device: timing only), plus the single-layer memory leg of configs[4]."""
    import torch
    out = {}
    legs = [(f"sweep-r{r}-n{n}", inputs.config_sweep(r, n)) for r in (20, 95) for n in (2, 16)]
    legs += [("ragged", inputs.config_ragged()), ("32k", inputs.config_32k())]
    for name, shape in legs:
        F = flops(shape)
        g = schedule.random_device_group(shape, dev, wave=max(1, shape.N), seed=shape.seed)
        step = lambda: schedule.run_prefixflow_step(ctx, g, stream)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

        def t(fn, k):
            fn()
            torch.cuda.synchronize()
            e0.record(stream)
            for _ in range(k):
                fn()
            e1.record(stream)
            torch.cuda.synchronize()
            return e0.elapsed_time(e1) / k
        ms = t(step, steps)
        rp = schedule.make_replay_packed(g)
        ms_r = t(lambda: schedule.run_replay_packed_step(ctx, rp, stream), max(1, steps - 1))
        out[name] = dict(step_ms=ms, step_tflops=F["step"] / (ms * 1e-3) / 1e12, replay_packed_ms=ms_r,
                         speedup=ms_r / ms, ideal_speedup_pair_model=F["ideal_speedup"])
        del g, rp
        torch.cuda.empty_cache()
    m = memory_legs(ctx, lifecycle, inputs.config_32k(), dev, 1, 0, reps=2)
    out["32k"]["memory_single_layer"] = m["single_layer"]
    return out


def run_sharded_group(args, shape, ctx, pf, pfd, inputs, schedule, dist, dev, rank, world, peaks) -> None:
    """N > 1, ONE rollout group over all ranks (strong scaling): --shard heads (KV-head sharding, no
    communication) or --shard split (suffix sharding with an all-gather of K1/V1
    and a reduce-scatter of gK1/gV1).  Prints the contract's JSON line."""
    import torch
    F = flops(shape)
    inp = inputs.make_group(shape)
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        dist.barrier()
        torch.cuda.synchronize()

    if args.shard == "heads":
        g = schedule.to_device(inp, dev, wave=max(1, shape.N))
        sh = schedule.head_shard(g, world, rank)
        step = lambda: schedule.run_prefixflow_step(ctx, sh, stream)
        extra = dict(parallelism=f"1 group over {world} ranks, KV-head sharded, no communication")
    else:
        plan = pfd.split_plan(shape, world, rank)
        rk = pfd.SplitGroupRank(ctx, inp, plan, dev, wave=0, stream=stream)
        comm = pfd.DistComm()
        cs = torch.cuda.Stream(dev)
        waits = []
        step = lambda: waits.append(pfd.run_split_group_step(rk, comm, cs))
        extra = dict(parallelism=f"1 group over {world} ranks: Phase A/C head-sharded, Phase B suffix-sharded, "
                                 f"all-gather K1/V1 + reduce-scatter gK1/gV1")
    for _ in range(args.warmup):
        step()
    if args.shard == "split":
        waits.clear()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    barrier()
    ms = pfd.max_over_ranks(e0.elapsed_time(e1), dev) / args.steps
    comm_ms = None
    if args.shard == "split":
        comm_ms = sum(a.elapsed_time(b) for w in waits for a, b in w.values()) / args.steps
        comm_ms = pfd.max_over_ranks(comm_ms, dev)
    cfg = workload_config(shape, args.config)
    cfg.update(extra)
    out = dict(metric=METRIC, value=F["step"] / (ms * 1e-3) / 1e12, unit=UNIT, n_gpus=world, steps=args.steps,
               warmup=args.warmup, ms_per_step=ms, higher_is_better=True, scaling="strong", vs_baseline=None,
               dtype="bf16", data="synthetic", config=cfg, shard=args.shard, exposed_comm_ms=comm_ms,
               flops=dict(step=F["step"]), peaks=peaks)
    if rank == 0:
        print(json.dumps(out))


# --------------------------------------------------------------------------------------------------
# GPU leg
# --------------------------------------------------------------------------------------------------
def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="7b")
    ap.add_argument("--replay-steps", type=int, default=-1, help="-1: max(3, steps // 4); 0: skip")
    ap.add_argument("--cpu-budget", type=float, default=6e11, help="algorithmic flops of the oracle sample")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--wave", type=int, default=0,
                    help="suffixes packed per Phase-B call (PAPER.md:158, 242 suffix microbatch); "
                         "0 = all N in one wave (default), 1 = one call per suffix")
    ap.add_argument("--no-wave1", action="store_true", help="skip the extra wave = 1 measurement")
    ap.add_argument("--no-companions", action="store_true", help="skip the pf_rope / pf_kv_proj_grad timings")
    ap.add_argument("--no-graph", action="store_true", help="skip the CUDA-graph replay of the step")
    ap.add_argument("--no-offload", action="store_true", help="skip the memory-lifecycle / offload measurement")
    ap.add_argument("--offload-wave", type=int, default=1, help="suffixes per wave in the lifecycle measurement")
    ap.add_argument("--layers", type=int, default=4, help="attention layers in the multi-layer offload pipeline (0 = skip)")
    ap.add_argument("--bwd-pairs", type=int, default=0, help="C-ABI option bwd_pairs_per_item (0 = heuristic)")
    ap.add_argument("--bwd-heads", type=int, default=0, help="C-ABI option bwd_heads_per_item (0 = model)")
    ap.add_argument("--deterministic", action="store_true", help="C-ABI option deterministic_gkv")
    ap.add_argument("--no-sweep", action="store_true", help="skip the compact prefix-ratio x N sweep / configs[2], configs[4] legs")
    ap.add_argument("--shard", default="groups", choices=["groups", "heads", "split"],
                    help="N > 1: 'groups' = one independent group per rank (weak scaling, default); 'heads' = ONE group "
                         "sharded by KV head, no communication; 'split' = ONE group, Phase B sharded by suffix with an "
                         "all-gather of K1/V1 and a reduce-scatter of gK1/gV1 (strong scaling)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist
    from paper_2606_01143_b200 import binding as pf          # raises if libprefixflow.so is missing
    from paper_2606_01143_b200 import dist as pfd
    from paper_2606_01143_b200 import inputs, lifecycle, schedule

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback of the product path)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    shape = pick_config(args.config)
    peaks = measured_peaks()
    ctx = pf.pf_create(local_rank)
    if args.bwd_pairs:
        pf.pf_set_option(ctx, "bwd_pairs_per_item", args.bwd_pairs)
    if args.bwd_heads:
        pf.pf_set_option(ctx, "bwd_heads_per_item", args.bwd_heads)
    if args.deterministic:
        pf.pf_set_option(ctx, "deterministic_gkv", 1)
    if world > 1 and args.shard != "groups":
        run_sharded_group(args, shape, ctx, pf, pfd, inputs, schedule, dist, dev, rank, world, peaks)
        pf.pf_destroy(ctx)
        dist.destroy_process_group()
        return
    # weak scaling over independent rollout groups: rank r draws its own group
    shape = pfd.rank_shape(shape, rank)
    F = flops(shape)
    inp = inputs.make_group(shape)
    wave = args.wave if args.wave > 0 else max(1, shape.N)
    g = schedule.to_device(inp, dev, wave=wave)
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def timed(fn, steps):
        """K steps between two CUDA events on the launch stream; max over ranks; returns ms/step."""
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(stream)
        for _ in range(steps):
            fn()
        e1.record(stream)
        barrier()
        return pfd.max_over_ranks(e0.elapsed_time(e1), dev) / steps

    step = lambda: schedule.run_prefixflow_step(ctx, g, stream)
    torch.cuda.reset_peak_memory_stats()
    for _ in range(args.warmup):
        step()
    n0 = pf.pf_counter(ctx, "kernel_launches")
    with ClockSampler(local_rank) as clk:
        ms_step = timed(step, args.steps)
    launches = pf.pf_counter(ctx, "kernel_launches") - n0
    peak_hbm = torch.cuda.max_memory_allocated()

    # ---- per-kernel event brackets of the C ABI: per-phase kernel time.  Two passes: (a) the same K
    # steps straight after the timed region (clocks as the long run left them: the part sags under
    # the power cap after some tens of ms of tensor load), (b) after an idle gap, a short pass of
    # <= 10 steps -- the burst regime the burst peak of MEASURED_PEAKS.json was taken in (best of 10
    # isolated GEMMs).  The rooflines use (b) against the burst peak; (a) is printed beside it.
    def profile_pass(nsteps):
        pf.pf_set_option(ctx, "profile", 1)
        for k in range(4):
            pf.pf_profile_read(ctx, k)
        ms = timed(step, nsteps)
        out = {}
        for k, name in enumerate(["A_fwd", "B_fwd", "B_bwd", "C_bwd"]):
            n, tot = pf.pf_profile_read(ctx, k)
            out[name] = dict(launches=n, ms_total=tot, ms_per_launch=tot / n if n else None)
        pf.pf_set_option(ctx, "profile", 0)
        return ms, out
    ms_step_inrun, prof_inrun = profile_pass(args.steps)
    time.sleep(1.0)
    for _ in range(2):
        step()
    psteps = min(args.steps, 10)
    ms_step_prof, prof = profile_pass(psteps)
    steps = args.steps
    ph_ms = {k: (v["ms_total"] / psteps) for k, v in prof.items()}
    ph_ms_inrun = {k: (v["ms_total"] / steps) for k, v in prof_inrun.items()}
    tf = lambda fl, ms: (fl / (ms * 1e-3) / 1e12) if ms and ms > 0 else None
    phases = dict(
        A_fwd=dict(ms=ph_ms["A_fwd"], tflops=tf(F["A"], ph_ms["A_fwd"])),
        B_fwd=dict(ms=ph_ms["B_fwd"], tflops=tf(F["B_fwd"], ph_ms["B_fwd"])),
        B_bwd=dict(ms=ph_ms["B_bwd"], tflops=tf(F["B_bwd"], ph_ms["B_bwd"])),
        C_bwd=dict(ms=ph_ms["C_bwd"], tflops=tf(F["C"], ph_ms["C_bwd"])))
    b_ms = ph_ms["B_fwd"] + ph_ms["B_bwd"]
    phaseB_tflops = tf(F["B_fwd"] + F["B_bwd"], b_ms)
    other_ms = ms_step_prof - sum(ph_ms.values())

    # roofline of the dominant kernel (attn_bwd_kernel as launched by pf_phaseB_bwd) and of the
    # forward kernel (pf_phaseB_fwd): pass (b) above (after an idle gap, <= 10 steps) against the
    # BURST peak; `achieved_in_run` is pass (a), straight after the K timed steps; the fraction of
    # the sustained peak (seconds-long GEMM loop under the power cap) is printed beside it.
    def roofline_of(kind, call, kname, fl):
        n = prof[kind]["launches"]
        ach = tf(fl * psteps / n, prof[kind]["ms_per_launch"]) if n else None
        n_in = prof_inrun[kind]["launches"]
        ach_in = tf(fl * steps / n_in, prof_inrun[kind]["ms_per_launch"]) if n_in else None
        return dict(achieved_in_run=ach_in, timing=f"CUDA events around each launch on the launch stream; "
                    f"{psteps} steps after a 1 s idle gap (burst regime); achieved_in_run = the {steps} steps "
                    "straight after the timed region",
                    bound="tensor", kernel=f"{kname} ({call})", achieved=ach, peak=peaks["burst"], unit="TFLOP/s",
                    frac=(ach / peaks["burst"]) if ach else None,
                    peak_kind="bf16 burst, " + peaks["source"],
                    frac_of_sustained=(ach / peaks["sustained"]) if ach else None, peak_sustained=peaks["sustained"],
                    frac_of_nominal=(ach / 2250.0) if ach else None,
                    flops_per_launch=fl / max(1, n // max(1, psteps)) if n else None,
                    ms_per_launch=prof[kind]["ms_per_launch"], traffic=ncu_traffic(kname, args.config))
    roofline = roofline_of("B_bwd", "pf_phaseB_bwd", f"attn_bwd_kernel<{shape.head_dim}>", F["B_bwd"])
    roofline_fwd = roofline_of("B_fwd", "pf_phaseB_fwd", f"attn_fwd_kernel<{shape.head_dim}>", F["B_fwd"])

    # ---- N-times replay baseline: the same kernels on every concatenated [P || S(i)] ----
    replay = None
    rsteps = max(3, args.steps // 4) if args.replay_steps < 0 else args.replay_steps
    if rsteps > 0:
        r = schedule.make_replay(g)
        rstep = lambda: schedule.run_replay_step(ctx, r, stream)
        for _ in range(2):
            rstep()
        ms_replay = timed(rstep, rsteps)
        del r
        torch.cuda.empty_cache()
        # the same N full sequences packed into one forward and one backward launch (Lp = 0,
        # n_seqs = N): the baseline pays one launch tail per kernel, like the step under test
        rp = schedule.make_replay_packed(g)
        rpstep = lambda: schedule.run_replay_packed_step(ctx, rp, stream)
        for _ in range(2):
            rpstep()
        ms_packed = timed(rpstep, rsteps)
        del rp
        torch.cuda.empty_cache()
        best = min(ms_replay, ms_packed)
        replay = dict(ms_per_step=best, steps=rsteps, tflops=tf(F["replay"], best),
                      speedup=best / ms_step, ideal_speedup_pair_model=F["ideal_speedup"],
                      per_sequence_ms=ms_replay, packed_ms=ms_packed,
                      note="speedup is quoted against the FASTER of the two replay organisations")

    # ---- the same step with one Phase-B call per suffix (the paper's "separate" organisation) ----
    wave1 = None
    if wave != 1 and not args.no_wave1:
        g1 = schedule.to_device(inp, dev, wave=1)
        step1 = lambda: schedule.run_prefixflow_step(ctx, g1, stream)
        for _ in range(args.warmup):
            step1()
        ms1 = timed(step1, args.steps)
        pf.pf_set_option(ctx, "profile", 1)
        for k in range(4):
            pf.pf_profile_read(ctx, k)
        timed(step1, args.steps)
        p1 = {name: pf.pf_profile_read(ctx, k) for k, name in enumerate(["A_fwd", "B_fwd", "B_bwd", "C_bwd"])}
        pf.pf_set_option(ctx, "profile", 0)
        bf_ms, bb_ms = p1["B_fwd"][1] / steps, p1["B_bwd"][1] / steps
        wave1 = dict(ms_per_step=ms1, tflops=world * F["step"] / (ms1 * 1e-3) / 1e12,
                     B_fwd=dict(ms=bf_ms, tflops=tf(F["B_fwd"], bf_ms), launches_per_step=p1["B_fwd"][0] // steps),
                     B_bwd=dict(ms=bb_ms, tflops=tf(F["B_bwd"], bb_ms), launches_per_step=p1["B_bwd"][0] // steps),
                     phaseB_tflops=tf(F["B_fwd"] + F["B_bwd"], bf_ms + bb_ms),
                     phaseB_pct_of_bf16_burst=100 * tf(F["B_fwd"] + F["B_bwd"], bf_ms + bb_ms) / peaks["burst"],
                     speedup_vs_replay=(replay["ms_per_step"] / ms1) if replay else None)
        # the same with the Phase-B forwards on a second stream (schedule.run_prefixflow_step(fwd_stream=...)):
        # the forward of suffix i+1 runs beside the backward of suffix i and fills the SMs that the
        # last round of CTAs of either launch leaves idle (224 forward CTAs on 148 SMs per suffix)
        side = torch.cuda.Stream(dev)
        step1s = lambda: schedule.run_prefixflow_step(ctx, g1, stream, fwd_stream=side)
        for _ in range(args.warmup):
            step1s()
        ms1s = timed(step1s, args.steps)
        wave1["fwd_side_stream"] = dict(ms_per_step=ms1s, tflops=world * F["step"] / (ms1s * 1e-3) / 1e12,
                                        speedup_vs_one_stream=ms1 / ms1s,
                                        speedup_vs_replay=(replay["ms_per_step"] / ms1s) if replay else None,
                                        note="Phase-B forwards enqueued on a second stream; every backward waits for its own forward")
        del step1s
        # the rejected gK/gV organisation, measured next to the shipped one: every
        # suffix adds into a partial accumulator of its own, one reduce pass before Phase C
        pK = torch.empty((shape.N, shape.Lp, shape.n_kv_heads, shape.head_dim), dtype=torch.float32, device=dev)
        pV = torch.empty_like(pK)
        stepp = lambda: schedule.run_prefixflow_step_partials(ctx, g1, pK, pV, stream)
        for _ in range(args.warmup):
            stepp()
        msp = timed(stepp, args.steps)
        wave1["gkv_partials"] = dict(ms_per_step=msp, vs_reduce_add=msp / ms1,
                                     partial_bytes=int(2 * pK.numel() * 4),
                                     note="per-suffix fp32 partials + torch.sum reduce before Phase C (rejected alternative)")
        del g1, pK, pV, stepp
        torch.cuda.empty_cache()

    # ---- the same step replayed from a CUDA graph (one launch per step: no gaps between the
    # dependent memsets / kernels); packed wave and, if measured above, one call per suffix ----
    graph = None
    if not args.no_graph:
        gr = schedule.capture_step(ctx, g)
        for _ in range(2):
            gr.replay()
        ms_g = timed(gr.replay, args.steps)
        graph = dict(ms_per_step=ms_g, tflops=world * F["step"] / (ms_g * 1e-3) / 1e12, speedup_vs_eager=ms_step / ms_g)
        del gr
        if wave1 is not None:
            g1 = schedule.to_device(inp, dev, wave=1)
            gr1 = schedule.capture_step(ctx, g1)
            for _ in range(2):
                gr1.replay()
            ms_g1 = timed(gr1.replay, args.steps)
            graph["wave1_ms_per_step"] = ms_g1
            graph["wave1_speedup_vs_eager"] = wave1["ms_per_step"] / ms_g1
            del gr1
            gr1s = schedule.capture_step(ctx, g1, fwd_stream=torch.cuda.Stream(dev))   # fork / join captured
            for _ in range(2):
                gr1s.replay()
            graph["wave1_fwd_side_stream_ms_per_step"] = timed(gr1s.replay, args.steps)
            del gr1s, g1
        torch.cuda.empty_cache()

    # ---- companions: RoPE of one wave's Q2 and K2 (HBM-bound) and the
    # dW_K terms of the step with a 7B-shaped d_model ----
    companions = None
    if not args.no_companions:
        pk = g.packed[0]
        q2, k2 = pk["Q2"].clone(), pk["K2"].clone()
        def rope_both():
            pf.pf_rope(ctx, pk["cu"], shape.Lp, q2, 10000.0, False, stream)
            pf.pf_rope(ctx, pk["cu"], shape.Lp, k2, 10000.0, False, stream)
        rope_both()
        ms_rope = timed(rope_both, args.steps)
        rope_bytes = 2 * (q2.numel() + k2.numel()) * 2
        dm = 128 * shape.n_q_heads
        X1 = torch.randn((shape.Lp, dm), device=dev).to(torch.bfloat16)
        X2 = torch.randn((pk["K2"].shape[0], dm), device=dev).to(torch.bfloat16)
        dW = torch.zeros((dm, shape.n_kv_heads * shape.head_dim), dtype=torch.float32, device=dev)
        def dwk():
            pf.pf_kv_proj_grad(ctx, X2, pk["dK2"], dW, stream)
            pf.pf_kv_proj_grad(ctx, X1, g.dK1, dW, stream)
        dwk()
        ms_dw = timed(dwk, args.steps)
        fl_dw = 2.0 * (shape.Lp + X2.shape[0]) * dm * dW.shape[1]
        companions = dict(
            rope=dict(ms=ms_rope, bytes=rope_bytes, gbs=rope_bytes / (ms_rope * 1e-3) / 1e9,
                      frac_of_hbm_peak=rope_bytes / (ms_rope * 1e-3) / 1e9 / peaks["hbm"],
                      what=f"pf_rope in place on Q2 {tuple(q2.shape)} and K2 {tuple(k2.shape)} of the wave, positions from Lp"),
            kv_proj_grad=dict(ms=ms_dw, tflops=fl_dw / (ms_dw * 1e-3) / 1e12, flops=fl_dw,
                              what=f"dW_K [{dm}, {dW.shape[1]}] += X2^T dK2 ({X2.shape[0]} tokens) + X1^T dK1 ({shape.Lp} tokens)"))
        del q2, k2, X1, X2, dW, rope_both, dwk, pk     # the closures hold the tensors: drop them too
        torch.cuda.empty_cache()

    # ---- memory lifecycle: Phase-B peak HBM with the dormant Phase-A set
    # {Q1, O1, LSE1} resident vs offloaded to a pinned host pool on a side stream ----
    memory = None
    if rank == 0 and not args.no_offload:
        del g
        torch.cuda.empty_cache()
        memory = memory_legs(ctx, lifecycle, shape, dev, args.offload_wave, args.layers)
        g = schedule.to_device(inp, dev, wave=wave)

    # ---- compact sweep: the four corners of the prefix-ratio x N sweep (configs[3]) and configs[2],
    # configs[4]: step vs replay, so that one bench line shows the trend ----
    sweep = None
    if rank == 0 and world == 1 and not args.no_sweep and args.config == "7b":
        del g
        torch.cuda.empty_cache()
        sweep = sweep_legs(ctx, schedule, lifecycle, inputs, dev, stream, peaks)
        g = schedule.to_device(inp, dev, wave=wave)

    # ---- end to end: pinned host inputs -> device, step, results -> pinned host, every step ----
    e2e = None
    if not args.no_e2e:
        pk = g.packed   # the packed wave tensors (the per-suffix entries of g.Q2 ... are views of them)
        ins = [g.Q1, g.K1, g.V1, g.dO1] + [w[k] for w in pk for k in ("Q2", "K2", "V2", "dO2")]
        outs = [g.O1, g.LSE1, g.dQ1, g.dK1, g.dV1, g.gK1, g.gV1] + \
               [w[k] for w in pk for k in ("O2", "LSE2", "dQ2", "dK2", "dV2")]
        h_in = [torch.empty(t.shape, dtype=t.dtype, pin_memory=True).copy_(t) for t in ins]
        h_out = [torch.empty(t.shape, dtype=t.dtype, pin_memory=True) for t in outs]
        bi = sum(t.numel() * t.element_size() for t in ins)
        bo = sum(t.numel() * t.element_size() for t in outs)

        def e2e_step():
            for h, t in zip(h_in, ins):
                pf.pf_prefetch(ctx, h, t, stream)          # cudaMemcpyAsync H2D through the C ABI
            schedule.run_prefixflow_step(ctx, g, stream)
            for t, h in zip(outs, h_out):
                pf.pf_offload(ctx, t, h, stream)           # cudaMemcpyAsync D2H through the C ABI

        for _ in range(2):
            e2e_step()
        ms_serial = timed(e2e_step, max(3, args.steps // 2))

        # pipelined over steps: two device buffer sets, H2D / compute / D2H on three streams, so the
        # copies of steps i+1 and i-1 overlap the kernels of step i (PCIe is full duplex)
        gb = schedule.to_device(inp, dev, wave=wave)
        sets = []
        for gg in (g, gb):
            pkk = gg.packed
            sets.append(dict(
                g=gg,
                ins=[gg.Q1, gg.K1, gg.V1, gg.dO1] + [w[k] for w in pkk for k in ("Q2", "K2", "V2", "dO2")],
                outs=[gg.O1, gg.LSE1, gg.dQ1, gg.dK1, gg.dV1, gg.gK1, gg.gV1] +
                     [w[k] for w in pkk for k in ("O2", "LSE2", "dQ2", "dK2", "dV2")],
                ev_in=torch.cuda.Event(), ev_comp=torch.cuda.Event(), ev_out=torch.cuda.Event()))
        s_in, s_out = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
        state = dict(i=0)

        def e2e_pipe_step():
            st = sets[state["i"] & 1]
            first = state["i"] < 2
            state["i"] += 1
            if not first:
                s_in.wait_event(st["ev_comp"])             # the kernels that read these inputs are done
            for h, t in zip(h_in, st["ins"]):
                pf.pf_prefetch(ctx, h, t, s_in)
            st["ev_in"].record(s_in)
            stream.wait_event(st["ev_in"])
            if not first:
                stream.wait_event(st["ev_out"])            # the previous outputs of this set were copied out
            schedule.run_prefixflow_step(ctx, st["g"], stream)
            st["ev_comp"].record(stream)
            s_out.wait_event(st["ev_comp"])
            for t, h in zip(st["outs"], h_out):
                pf.pf_offload(ctx, t, h, s_out)
            st["ev_out"].record(s_out)

        def e2e_pipe(steps_):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            state["i"] = 0
            barrier()
            e0.record(stream)
            for _ in range(steps_):
                e2e_pipe_step()
            stream.wait_stream(s_out)                      # the last results are on the host
            e1.record(stream)
            barrier()
            return pfd.max_over_ranks(e0.elapsed_time(e1), dev) / steps_

        e2e_pipe(4)
        ms_e2e = e2e_pipe(max(6, args.steps))
        e2e = dict(value=world * F["step"] / (ms_e2e * 1e-3) / 1e12, unit=UNIT, ms_per_step=ms_e2e,
                   h2d_bytes_per_step=bi, d2h_bytes_per_step=bo, serial_ms_per_step=ms_serial,
                   serial_value=world * F["step"] / (ms_serial * 1e-3) / 1e12,
                   note="every step copies all inputs from pinned host memory and all outputs back "
                        "through the C ABI; pipelined over steps on three streams (H2D | kernels | "
                        "D2H, two device buffer sets); serial_* = the same on one stream")
        del gb, sets
        del h_in, h_out

    # ---- CPU oracle on a bounded sample (rank 0, N = 1 only) ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        dt, work, desc, thr = oracle_sample(shape, args.cpu_budget)
        cpu = dict(value=work / dt / 1e12, unit=UNIT, cores=thr, kind="oracle", sample=desc,
                   seconds=dt)

    value = world * F["step"] / (ms_step * 1e-3) / 1e12
    ws_bytes = sum(t.numel() * t.element_size() for t in
                   [g.Q1, g.K1, g.V1, g.dO1, g.O1, g.dQ1, g.dK1, g.dV1, g.gK1, g.gV1] +
                   g.Q2 + g.K2 + g.V2 + g.dO2 + g.O2 + g.dQ2 + g.dK2 + g.dV2)
    cfg = workload_config(shape, args.config)
    cfg["wave"] = wave
    if args.bwd_pairs or args.deterministic:
        cfg["bwd_split"] = "deterministic_gkv" if args.deterministic else f"bwd_pairs_per_item={args.bwd_pairs}"
    cfg["l2"] = (f"no explicit flush: one step touches {ws_bytes / 2 ** 20:.0f} MiB of inputs+outputs "
                 f"(> 126 MiB L2) before any tensor is reused" if ws_bytes > L2_BYTES else
                 f"working set {ws_bytes / 2 ** 20:.0f} MiB fits L2 (parity-size config; not a bench line)")
    out = dict(
        metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
        ms_per_step=ms_step, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="bf16",
        data="synthetic", config=cfg, clocks=clk.summary(), e2e=e2e, gpu_launches=launches,
        roofline=roofline, roofline_fwd=roofline_fwd, cpu_baseline=cpu, sweep=sweep, graph=graph, companions=companions,
        phases=phases, phaseB=dict(ms=b_ms, tflops=phaseB_tflops,
                                   pct_of_bf16_burst=100 * phaseB_tflops / peaks["burst"] if phaseB_tflops else None,
                                   pct_of_bf16_sustained=100 * phaseB_tflops / peaks["sustained"] if phaseB_tflops else None,
                                   pct_of_bf16_nominal=100 * phaseB_tflops / 2250.0 if phaseB_tflops else None),
        ms_per_step_profiled=ms_step_prof, non_attention_ms=other_ms,
        phases_in_run={k: dict(ms=v, tflops=tf(F[{"A_fwd": "A", "B_fwd": "B_fwd", "B_bwd": "B_bwd", "C_bwd": "C"}[k]], v))
                       for k, v in ph_ms_inrun.items()},
        ms_per_step_profiled_in_run=ms_step_inrun,
        replay=replay, wave1=wave1, memory=memory, flops=dict(A=F["A"], B_fwd=F["B_fwd"], B_bwd=F["B_bwd"], C=F["C"], step=F["step"],
                                  replay=F["replay"]),
        peak_hbm_bytes=peak_hbm, peaks=peaks)
    pf.pf_destroy(ctx)
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
