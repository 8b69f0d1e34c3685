"""GPU parity at BASELINE.json's full size (configs[1], 7B-shaped, 83% prefix) in the launch
configuration bench.py times (all N suffixes in one packed wave): sampled outputs the fp64 oracle
computes one by one -- every suffix row of one KV-head group for two suffixes, sampled key columns
(tile edges included) of dK2/dV2 and of the accumulated gK1/gV1, sampled prefix rows and key
columns of Phase A / Phase C."""
import numpy as np
import pytest
import torch

import oracle
from oracle import reference as oref
from paper_2606_01143_b200 import binding as pf
from paper_2606_01143_b200 import inputs, schedule
from parity_util import check

pytestmark = pytest.mark.gpu


def test_config_7b_sampled():
    shape = inputs.config_7b()
    inp = inputs.make_group(shape)
    Lp, G, d, N = shape.Lp, shape.G, shape.head_dim, shape.N
    ctx = pf.pf_create(0)
    g = schedule.to_device(inp, wave=N)
    snap = {}
    schedule.run_prefixflow_step(ctx, g, after_each_suffix=lambda i: snap.update(
        gk=g.gK1.clone(), gv=g.gV1.clone()))
    torch.cuda.synchronize()
    pf.pf_destroy(ctx)

    kv = 1                                                   # the KV-head group that is checked
    heads = list(range(kv * G, (kv + 1) * G))
    pj = np.array([0, 1, 127, 128, 129, 2047, 2048, 3000, 4095, 5000, 5118, 5119], dtype=np.int64)
    sj = np.array([0, 63, 64, 127, 128, 500, 1000, 1023], dtype=np.int64)
    gk_sum = np.zeros((len(pj), d)); gv_sum = np.zeros((len(pj), d))
    for i in range(N):
        r = oref.sampled_phaseB(inp, i, kv, pj, sj)
        gk_sum += r["gk"]; gv_sum += r["gv"]
        if i in (0, 5):                                      # every suffix row of the group, two suffixes
            check(f"O2[{i}] group {kv}", g.O2[i][:, heads].permute(1, 0, 2), r["o2"])
            check(f"LSE2[{i}] group {kv}", g.LSE2[i][heads], r["lse2"], lse=True)
            check(f"dQ2[{i}] group {kv}", g.dQ2[i][:, heads].permute(1, 0, 2), r["dq2"])
            check(f"dK2[{i}] sampled keys", g.dK2[i][sj, kv], r["dk2"])
            check(f"dV2[{i}] sampled keys", g.dV2[i][sj, kv], r["dv2"])
    check("gK1 after Phase B, sampled keys", snap["gk"][pj, kv], gk_sum)
    check("gV1 after Phase B, sampled keys", snap["gv"][pj, kv], gv_sum)

    # ---- Phase A / Phase C: rows of the prefix alone (any replay's prefix rows)
    q1, k1, v1, do1 = (oref.widen(x) for x in (inp.Q1, inp.K1, inp.V1, inp.dO1))
    ts = np.array([0, 1, 127, 128, 1000, 2559, 4096, 5119], dtype=np.int64)
    hs_s = np.repeat(np.array(heads, dtype=np.int32), len(ts)); ts_s = np.tile(ts, G)
    o, lse, delta, dq = oref.rows(q1, k1, v1, do1, hs_s, ts_s)
    check("O1 sampled rows", g.O1[ts][:, heads].permute(1, 0, 2), o.reshape(G, len(ts), d))
    check("LSE1 sampled rows", g.LSE1[heads][:, ts], lse.reshape(G, len(ts)), lse=True)
    check("dQ1 sampled rows", g.dQ1[ts][:, heads].permute(1, 0, 2), dq.reshape(G, len(ts), d))
    # own-prefix dK/dV at the sampled keys need the statistics of every prefix row of the group
    hs_a = np.repeat(np.array(heads, dtype=np.int32), Lp); ts_a = np.tile(np.arange(Lp, dtype=np.int64), G)
    _, lse_a, delta_a, _ = oref.rows(q1, k1, v1, do1, hs_a, ts_a)
    lse_f = np.full((shape.n_q_heads, Lp), np.nan); dl_f = np.full((shape.n_q_heads, Lp), np.nan)
    lse_f[heads] = lse_a.reshape(G, Lp); dl_f[heads] = delta_a.reshape(G, Lp)
    dk_own, dv_own = oref.cols(q1, k1, v1, do1, lse_f, dl_f, np.full(len(pj), kv, np.int32), pj, 0, Lp)
    check("dK1 = own + gK1, sampled keys", g.dK1[pj, kv], dk_own + gk_sum)
    check("dV1 = own + gV1, sampled keys", g.dV1[pj, kv], dv_own + gv_sum)
