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


def _phaseB_subset_sampled(shape, subset, kv, pj, sj_of):
    """Phase A + Phase B of a SUBSET of the config's suffixes in one packed wave (the prefix and the
    chosen suffixes are drawn exactly as in the full config); every suffix row of KV-head group `kv`
    and sampled key columns are compared, gK1/gV1 against the sum over the subset."""
    inp = inputs.make_group(shape, only_suffixes=subset)
    G, d = shape.G, shape.head_dim
    ctx = pf.pf_create(0)
    g = schedule.to_device(inp, suffixes=subset, wave=len(subset))
    grp = pf.pf_group_begin(ctx, g.desc, g.Lp, g.K1, g.V1, g.gK1, g.gV1, g.workspace)
    pf.pf_phaseA_fwd(grp, g.Q1, g.O1, g.LSE1)
    pk = g.packed[0]
    pf.pf_phaseB_fwd(grp, pk["cu"], pk["Q2"], pk["K2"], pk["V2"], pk["O2"], pk["LSE2"])
    pf.pf_phaseB_bwd(grp, pk["cu"], pk["Q2"], pk["K2"], pk["V2"], pk["O2"], pk["LSE2"], pk["dO2"],
                     pk["dQ2"], pk["dK2"], pk["dV2"])
    pf.pf_group_end(grp)
    torch.cuda.synchronize()
    pf.pf_destroy(ctx)
    heads = list(range(kv * G, (kv + 1) * G))
    gk_sum = np.zeros((len(pj), d)); gv_sum = np.zeros((len(pj), d))
    for n, i in enumerate(subset):
        sj = sj_of(shape.Ls[i])
        r = oref.sampled_phaseB(inp, i, kv, pj, sj)
        gk_sum += r["gk"]; gv_sum += r["gv"]
        check(f"O2[{i}]", g.O2[n][:, heads].permute(1, 0, 2), r["o2"])
        check(f"LSE2[{i}]", g.LSE2[n][heads], r["lse2"], lse=True)
        check(f"dQ2[{i}]", g.dQ2[n][:, heads].permute(1, 0, 2), r["dq2"])
        check(f"dK2[{i}] sampled keys", g.dK2[n][sj, kv], r["dk2"])
        check(f"dV2[{i}] sampled keys", g.dV2[n][sj, kv], r["dv2"])
    check("gK1 (subset), sampled keys", g.gK1[pj, kv], gk_sum)
    check("gV1 (subset), sampled keys", g.gV1[pj, kv], gv_sum)


def test_config_ragged_sampled():
    """BASELINE.json configs[2]: 28q/4kv, prefix 16384, ragged suffix lengths (three of the 16)."""
    shape = inputs.config_ragged()
    order = np.argsort(shape.Ls)
    subset = sorted(int(i) for i in (order[0], order[len(order) // 2], order[-1]))   # shortest, median, longest
    pj = np.array([0, 127, 128, 8191, 8192, 12345, 16255, 16256, 16383], dtype=np.int64)
    sj_of = lambda Ls: np.unique(np.array([0, 1, 63, 64, 127, 128, Ls // 2, Ls - 2, Ls - 1], dtype=np.int64))
    _phaseB_subset_sampled(shape, subset, kv=2, pj=pj, sj_of=sj_of)


def test_config_32k_sampled():
    """BASELINE.json configs[4]: 40q/8kv (GQA 5:1), prefix 32768, one of the 8 suffixes of 2048."""
    shape = inputs.config_32k()
    pj = np.array([0, 128, 16383, 16384, 32639, 32640, 32767], dtype=np.int64)
    sj_of = lambda Ls: np.array([0, 127, 128, 1024, Ls - 1], dtype=np.int64)
    _phaseB_subset_sampled(shape, [3], kv=5, pj=pj, sj_of=sj_of)
