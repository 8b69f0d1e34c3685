"""N > 1 host logic on CPU with two gloo ranks: (a) bench.py's default mode -- independent groups per
rank, MAX-over-ranks timing (weak scaling, no data-path collective); (b) the split-group mode of ONE
group: the plan, the all-gather of the
head-sharded K1/V1 and the reduce-scatter of the per-rank gK1/gV1 partial sums over the KV-head
dimension, checked against the oracle's per-suffix coupling gradients (CPU tensors stand in for what
each rank's kernels produce)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_01143_b200 import dist as pfd
from paper_2606_01143_b200 import inputs


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        shape = pfd.rank_shape(inputs.config_tiny(), rank)
        inp = inputs.make_group(shape)
        ms = pfd.max_over_ranks(1.0 + rank)                    # rank 1 is the slow one
        val = pfd.aggregate_throughput(10.0, ms, world)
        digest = float(inp.Q1.float().sum())
        gathered = [None] * world
        dist.all_gather_object(gathered, (shape.seed, digest))
        out.put((rank, ms, val, gathered))
    finally:
        dist.destroy_process_group()


def test_two_ranks_independent_groups_and_max_time():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, val, gathered in res:
        assert ms == 2.0                                        # MAX over ranks, on every rank
        assert val == world * 10.0 / 2e-3
        seeds = [g[0] for g in gathered]
        assert seeds == [0, pfd.RANK_SEED_STRIDE]               # each rank has its own group
        assert gathered[0][1] != gathered[1][1]                 # ... with different data


def test_single_process_is_identity():
    assert pfd.max_over_ranks(3.5) == 3.5
    s = pfd.rank_shape(inputs.config_7b(), 3)
    assert s.seed == 1000 + 3 * pfd.RANK_SEED_STRIDE and s.Ls == inputs.config_7b().Ls


def _split_worker(rank: int, world: int, port: int, out):
    import numpy as np
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        shape = inputs.small_case(4, 2, 16, 40, [9, 17, 5], seed=77, dist="unit")
        inp = inputs.make_group(shape)                     # every rank draws the same group
        ref = oracle.group_reference(inp)
        plan = pfd.split_plan(shape, world, rank)
        comm = pfd.DistComm()
        kv = plan.kv_heads
        # all-gather of the head-sharded cache (bf16), as after the head-sharded Phase A
        K1f = comm.all_gather_heads(inp.K1[:, kv.start:kv.stop])
        V1f = comm.all_gather_heads(inp.V1[:, kv.start:kv.stop])
        ok_gather = bool(torch.equal(K1f, inp.K1) and torch.equal(V1f, inp.V1))
        # the rank's Phase-B partial sums over ITS suffixes, all heads (fp32), then reduce-scatter
        part = lambda each: torch.from_numpy(
            sum((each[i] for i in plan.suffixes), np.zeros_like(each[0]))).to(torch.float32)
        gk = comm.reduce_scatter_heads(part(ref.gK1_each))
        gv = comm.reduce_scatter_heads(part(ref.gV1_each))
        want_k = ref.gK1_after[-1][:, kv.start:kv.stop]
        want_v = ref.gV1_after[-1][:, kv.start:kv.stop]
        err = max(float(np.abs(gk.double().numpy() - want_k).max()), float(np.abs(gv.double().numpy() - want_v).max()))
        scale = float(np.abs(want_k).max())
        out.put((rank, list(kv), list(plan.q_heads), plan.suffixes, ok_gather, tuple(gk.shape), err, scale))
    finally:
        dist.destroy_process_group()


def test_split_group_plan_and_collectives():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_split_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    suffixes = []
    for rank, kv, qh, suf, ok_gather, shp, err, scale in res:
        assert kv == [rank] and qh == [2 * rank, 2 * rank + 1]     # Hkv = 2 over 2 ranks, G = 2
        assert ok_gather and shp == (40, 1, 16)
        assert err <= 1e-6 * max(1.0, scale)                       # fp32 sum of fp64 oracle values
        suffixes += suf
    assert sorted(suffixes) == [0, 1, 2]                           # every suffix on exactly one rank
    # longest-processing-time-first: the longest suffix (index 1) alone on one rank
    assert [1] in [r[3] for r in res]


def test_split_plan_is_deterministic_and_balanced():
    shape = inputs.config_ragged()
    plans = [pfd.split_plan(shape, 4, r) for r in range(4)]
    assert sorted(i for p in plans for i in p.suffixes) == list(range(16))
    assert [list(p.kv_heads) for p in plans] == [[0], [1], [2], [3]]
    cost = lambda i: shape.Ls[i] * shape.Lp + shape.Ls[i] * (shape.Ls[i] + 1) // 2
    loads = [sum(cost(i) for i in p.suffixes) for p in plans]
    assert max(loads) <= 1.15 * (sum(loads) / 4)                   # LPT keeps the ranks within 15 %
    assert plans == [pfd.split_plan(shape, 4, r) for r in range(4)]
    import pytest
    with pytest.raises(ValueError):
        pfd.split_plan(shape, 3, 0)                                # 4 KV heads do not shard over 3 ranks
