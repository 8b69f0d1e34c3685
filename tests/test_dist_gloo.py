"""N > 1 host logic of bench.py on CPU: two gloo ranks, independent groups per rank, MAX-over-ranks
timing (the task's multi-GPU contract: weak scaling, no data-path collective)."""
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
