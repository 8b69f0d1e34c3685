"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (all N
suffixes in one packed wave): sampled outputs the fp64 oracle computes one by one -- every suffix
row of one KV-head group for two suffixes, sampled key columns (tile edges included) of dK2/dV2
and of the accumulated gK1/gV1, sampled prefix rows and key columns of Phase A / Phase C.

  configs[1] (7B-shaped)  : N(0,1)/sqrt(d), unit-logit and the adversarial "ramp" distribution
  configs[3] (sweep)      : 32q/8kv, T = 8192: r = 83 %, N = 8, and the unaligned prefix 6799
  configs[2], configs[4]  : a subset of the suffixes in one wave; Phase A / C at Lp = 16384 / 32768
"""
import numpy as np
import pytest
import torch

import oracle
from oracle import reference as oref
from paper_2606_01143_b200 import binding as pf
from paper_2606_01143_b200 import inputs, schedule
from parity_util import RAMP_MAX_REL, RAMP_RMS_REL, STRICT_RMS_REL
from parity_util import check as _check

_grad_rms_gate = STRICT_RMS_REL


def check(name, got, ref, **kw):
    """parity_util.check with the relative-RMS gate of gradient tensors set per input distribution."""
    if name[0] in "dg":
        kw.setdefault("rms_rel_gate", _grad_rms_gate)
        if _grad_rms_gate == RAMP_RMS_REL:
            kw.setdefault("max_rel_gate", RAMP_MAX_REL)
    return _check(name, got, ref, **kw)

pytestmark = pytest.mark.gpu


def _edges(L, extra=()):
    """Sampled positions of a length-L axis: both ends, the 64/128-row tile edges next to them, the
    middle and whatever `extra` names (clipped, unique, sorted)."""
    c = [0, 1, 63, 64, 127, 128, 129, L // 2 - 1, L // 2, L - 130, L - 129, L - 128, L - 65, L - 64,
         L - 2, L - 1, *extra]
    return np.unique(np.array([x for x in c if 0 <= x < L], dtype=np.int64))


def _phaseAC_sampled(shape, inp, g, kv, gk_at, gv_at, pj_c, ts):
    """Phase A / Phase C outputs of KV-head group `kv` against the oracle: O1 / LSE1 / dQ1 at the
    sampled rows `ts`, dK1 / dV1 = own-prefix term + accumulated gK1 / gV1 at the sampled keys
    `pj_c` (gk_at / gv_at = the oracle's accumulated coupling gradients at those keys).  The
    own-prefix term of key j needs the statistics of every prefix row t >= j of the group, so the
    oracle evaluates the rows [min(pj_c), Lp)."""
    Lp, G, d = shape.Lp, shape.G, shape.head_dim
    heads = list(range(kv * G, (kv + 1) * G))
    q1, k1, v1, do1 = (oref.widen(x) for x in (inp.Q1, inp.K1, inp.V1, inp.dO1))
    hs_s = np.repeat(np.array(heads, dtype=np.int32), len(ts)); ts_s = np.tile(ts, G)
    o, lse, delta, dq = oref.rows(q1, k1, v1, do1, hs_s, ts_s)
    check("O1 sampled rows", g.O1[ts][:, heads].permute(1, 0, 2), o.reshape(G, len(ts), d))
    check("LSE1 sampled rows", g.LSE1[heads][:, ts], lse.reshape(G, len(ts)), lse=True)
    check("dQ1 sampled rows", g.dQ1[ts][:, heads].permute(1, 0, 2), dq.reshape(G, len(ts), d))
    r0 = int(pj_c.min())
    rr = np.arange(r0, Lp, dtype=np.int64)
    hs_a = np.repeat(np.array(heads, dtype=np.int32), len(rr)); ts_a = np.tile(rr, G)
    _, lse_a, delta_a, _ = oref.rows(q1, k1, v1, do1, hs_a, ts_a)
    lse_f = np.full((shape.n_q_heads, Lp), np.nan); dl_f = np.full((shape.n_q_heads, Lp), np.nan)
    lse_f[np.ix_(heads, rr)] = lse_a.reshape(G, len(rr)); dl_f[np.ix_(heads, rr)] = delta_a.reshape(G, len(rr))
    dk_own, dv_own = oref.cols(q1, k1, v1, do1, lse_f, dl_f, np.full(len(pj_c), kv, np.int32), pj_c, 0, Lp)
    check("dK1 = own + gK1, sampled keys", g.dK1[pj_c, kv], dk_own + gk_at)
    check("dV1 = own + gV1, sampled keys", g.dV1[pj_c, kv], dv_own + gv_at)


def _full_step_sampled(shape, kv, row_suffixes):
    """One whole A -> B -> C step exactly as bench.py launches it (one packed wave of all N suffixes)."""
    inp = inputs.make_group(shape)
    Lp, G, d, N = shape.Lp, shape.G, shape.head_dim, shape.N
    ctx = pf.pf_create(0)
    g = schedule.to_device(inp, wave=N)
    snap = {}
    schedule.run_prefixflow_step(ctx, g, after_each_suffix=lambda i: snap.update(
        gk=g.gK1.clone(), gv=g.gV1.clone()))
    torch.cuda.synchronize()
    pf.pf_destroy(ctx)

    heads = list(range(kv * G, (kv + 1) * G))
    pj = _edges(Lp, (2047, 2048, 3000, 4095))
    gk_sum = np.zeros((len(pj), d)); gv_sum = np.zeros((len(pj), d))
    for i in range(N):
        sj = _edges(shape.Ls[i], (500,))
        r = oref.sampled_phaseB(inp, i, kv, pj, sj)
        gk_sum += r["gk"]; gv_sum += r["gv"]
        if i in row_suffixes:                                # every suffix row of the group
            check(f"O2[{i}] group {kv}", g.O2[i][:, heads].permute(1, 0, 2), r["o2"])
            check(f"LSE2[{i}] group {kv}", g.LSE2[i][heads], r["lse2"], lse=True)
            check(f"dQ2[{i}] group {kv}", g.dQ2[i][:, heads].permute(1, 0, 2), r["dq2"])
        check(f"dK2[{i}] sampled keys", g.dK2[i][sj, kv], r["dk2"])
        check(f"dV2[{i}] sampled keys", g.dV2[i][sj, kv], r["dv2"])
    check("gK1 after Phase B, sampled keys", snap["gk"][pj, kv], gk_sum)
    check("gV1 after Phase B, sampled keys", snap["gv"][pj, kv], gv_sum)
    # Phase A / Phase C: rows of the prefix alone (any replay's prefix rows)
    _phaseAC_sampled(shape, inp, g, kv, gk_sum, gv_sum, pj, _edges(Lp, (1000, 2559, 4096)))


@pytest.mark.parametrize("dist", ["std", "unit", "ramp"])
def test_config_7b_sampled(dist):
    """BASELINE.json configs[1]: 28q/4kv, d=128, prefix 5120, N=8 x 1024 -- the bench workload -- at the
    BASELINE.json input scale, with unit logits (SURVEY.md section 8c reading 16 iii) and with the
    adversarial ramp (every row re-bases its softmax maximum ~4 times along the KV loop)."""
    global _grad_rms_gate
    ctx = pf.pf_create(0)
    n0 = pf.pf_counter(ctx, "fwd_rescale_rows")
    _grad_rms_gate = RAMP_RMS_REL if dist == "ramp" else STRICT_RMS_REL
    try:
        _full_step_sampled(inputs.config_7b(dist=dist), kv=1, row_suffixes=(0, 5))
    finally:
        _grad_rms_gate = STRICT_RMS_REL
    n1 = pf.pf_counter(ctx, "fwd_rescale_rows")
    pf.pf_destroy(ctx)
    if dist == "ramp":
        assert n1 - n0 >= (5120 + 8 * 1024) * 28, (n0, n1)


def test_config_sweep_r83_n8_sampled():
    """BASELINE.json configs[3]: 32q/8kv (G = 4), d=128, T = 8192, prefix 6784 (83 %), N = 8."""
    _full_step_sampled(inputs.config_sweep(83, 8), kv=6, row_suffixes=(2,))


def test_config_sweep_unaligned_prefix_sampled():
    """configs[3] with the unaligned prefix of SURVEY.md section 8d (6799 = 82.99 % of 8192, not a
    multiple of 64): ragged prefix tail tile and suffix rows that start mid-tile, unit logits."""
    shape = inputs.GroupShape("sweep-r83u-n4", 32, 8, 128, 6799, [8192 - 6799] * 4, seed=3834, dist="unit")
    _full_step_sampled(shape, kv=3, row_suffixes=(1,))


def _phaseABC_subset_sampled(shape, subset, kv, pj, sj_of, ts):
    """Phase A, Phase B of a SUBSET of the config's suffixes in one packed wave, and Phase C (the
    prefix and the chosen suffixes are drawn exactly as in the full config); every suffix row of
    KV-head group `kv` and sampled key columns are compared, gK1/gV1 against the sum over the subset,
    Phase A / C at sampled prefix rows and at key columns of the last 1536 prefix rows."""
    inp = inputs.make_group(shape, only_suffixes=subset)
    G, d, Lp = shape.G, shape.head_dim, shape.Lp
    ctx = pf.pf_create(0)
    g = schedule.to_device(inp, suffixes=subset, wave=len(subset))
    grp = pf.pf_group_begin(ctx, g.desc, g.Lp, g.K1, g.V1, g.gK1, g.gV1, g.workspace)
    pf.pf_phaseA_fwd(grp, g.Q1, g.O1, g.LSE1)
    pk = g.packed[0]
    pf.pf_phaseB_fwd(grp, pk["cu"], pk["Q2"], pk["K2"], pk["V2"], pk["O2"], pk["LSE2"])
    pf.pf_phaseB_bwd(grp, pk["cu"], pk["Q2"], pk["K2"], pk["V2"], pk["O2"], pk["LSE2"], pk["dO2"],
                     pk["dQ2"], pk["dK2"], pk["dV2"])
    torch.cuda.synchronize()
    gk_dev, gv_dev = g.gK1.clone(), g.gV1.clone()
    pf.pf_phaseC_bwd(grp, g.Q1, g.O1, g.LSE1, g.dO1, g.dQ1, g.dK1, g.dV1)
    pf.pf_group_end(grp)
    torch.cuda.synchronize()
    pf.pf_destroy(ctx)
    heads = list(range(kv * G, (kv + 1) * G))
    pj_c = np.array([Lp - 1536, Lp - 1025, Lp - 1024, Lp - 129, Lp - 128, Lp - 64, Lp - 1], dtype=np.int64)
    pj_all = np.unique(np.concatenate([pj, pj_c]))
    gk_sum = np.zeros((len(pj_all), d)); gv_sum = np.zeros((len(pj_all), d))
    for n, i in enumerate(subset):
        sj = sj_of(shape.Ls[i])
        r = oref.sampled_phaseB(inp, i, kv, pj_all, sj)
        gk_sum += r["gk"]; gv_sum += r["gv"]
        check(f"O2[{i}]", g.O2[n][:, heads].permute(1, 0, 2), r["o2"])
        check(f"LSE2[{i}]", g.LSE2[n][heads], r["lse2"], lse=True)
        check(f"dQ2[{i}]", g.dQ2[n][:, heads].permute(1, 0, 2), r["dq2"])
        check(f"dK2[{i}] sampled keys", g.dK2[n][sj, kv], r["dk2"])
        check(f"dV2[{i}] sampled keys", g.dV2[n][sj, kv], r["dv2"])
    check("gK1 (subset), sampled keys", gk_dev[pj_all, kv], gk_sum)
    check("gV1 (subset), sampled keys", gv_dev[pj_all, kv], gv_sum)
    sel = np.searchsorted(pj_all, pj_c)
    _phaseAC_sampled(shape, inp, g, kv, gk_sum[sel], gv_sum[sel], pj_c, ts)


def test_config_ragged_sampled():
    """BASELINE.json configs[2]: 28q/4kv, prefix 16384, ragged suffix lengths (three of the 16);
    Phase A / C at Lp = 16384."""
    shape = inputs.config_ragged()
    order = np.argsort(shape.Ls)
    subset = sorted(int(i) for i in (order[0], order[len(order) // 2], order[-1]))   # shortest, median, longest
    pj = np.array([0, 127, 128, 8191, 8192, 12345, 16255, 16256, 16383], dtype=np.int64)
    sj_of = lambda Ls: np.unique(np.array([0, 1, 63, 64, 127, 128, Ls // 2, Ls - 2, Ls - 1], dtype=np.int64))
    ts = np.array([0, 127, 128, 4095, 8192, 12287, 16256, 16383], dtype=np.int64)
    _phaseABC_subset_sampled(shape, subset, kv=2, pj=pj, sj_of=sj_of, ts=ts)


def test_config_32k_sampled():
    """BASELINE.json configs[4]: 40q/8kv (GQA 5:1), prefix 32768, one of the 8 suffixes of 2048;
    Phase A / C at Lp = 32768."""
    shape = inputs.config_32k()
    pj = np.array([0, 128, 16383, 16384, 32639, 32640, 32767], dtype=np.int64)
    sj_of = lambda Ls: np.array([0, 127, 128, 1024, Ls - 1], dtype=np.int64)
    ts = np.array([0, 128, 16383, 16384, 24575, 32640, 32767], dtype=np.int64)
    _phaseABC_subset_sampled(shape, [3], kv=5, pj=pj, sj_of=sj_of, ts=ts)
