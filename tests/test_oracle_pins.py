"""Pins of the fp64 oracle against what the paper and the mathematics fix (not against itself).

Every test here is CPU-only (-m "not gpu").  A plausible mistake in oracle/pf_oracle.c (dropped
term, wrong sign or index, transposed operand, wrong GQA map, exclusive diagonal, missing sigma)
fails at least one of them.
"""
import math
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2606_01143_b200 import inputs as I

RNG = np.random.default_rng(1234)


def rand_seq(T, Hq, Hkv, d, scale=1.0, rng=RNG):
    q = rng.standard_normal((T, Hq, d)) * scale
    k = rng.standard_normal((T, Hkv, d)) * scale
    v = rng.standard_normal((T, Hkv, d)) * scale
    dO = rng.standard_normal((T, Hq, d)) * scale
    return q, k, v, dO


# ---------------------------------------------------------------------------------------------
# hand-worked example (tests/golden/two_token.txt)
# ---------------------------------------------------------------------------------------------

def _golden():
    path = os.path.join(os.path.dirname(__file__), "golden", "two_token.txt")
    env = {"ln2": math.log(2.0), "ln3": math.log(3.0)}
    out = {}
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        name, expr = line.split(None, 1)
        out[name] = float(eval(expr, {"__builtins__": {}}, env))
    return out


def test_two_token_golden():
    g = _golden()
    q = np.array([1.0, 1.0]).reshape(2, 1, 1)
    k = np.array([0.0, math.log(2.0)]).reshape(2, 1, 1)
    v = np.array([3.0, 6.0]).reshape(2, 1, 1)
    dO = np.array([1.0, 3.0]).reshape(2, 1, 1)
    r = oracle.fullseq(q, k, v, dO, Lp=1, sigma=1.0)
    tol = 1e-14
    assert abs(r["o"][0, 0, 0] - g["o0"]) < tol and abs(r["o"][1, 0, 0] - g["o1"]) < tol
    assert abs(r["lse"][0, 0] - g["lse0"]) < tol and abs(r["lse"][0, 1] - g["lse1"]) < tol
    assert abs(r["dq"][0, 0, 0] - g["dq0"]) < tol and abs(r["dq"][1, 0, 0] - g["dq1"]) < tol
    assert abs(r["dk"][0, 0, 0] - g["dk0_own"]) < tol and abs(r["gk"][0, 0, 0] - g["gk0"]) < tol
    assert abs(r["dv"][0, 0, 0] - g["dv0_own"]) < tol and abs(r["gv"][0, 0, 0] - g["gv0"]) < tol
    assert abs(r["dk"][0, 0, 0] + r["gk"][0, 0, 0] - g["dk0_total"]) < tol
    assert abs(r["dv"][0, 0, 0] + r["gv"][0, 0, 0] - g["dv0_total"]) < tol
    assert abs(r["dk"][1, 0, 0] - g["dk1"]) < tol and abs(r["dv"][1, 0, 0] - g["dv1"]) < tol


# ---------------------------------------------------------------------------------------------
# central finite differences of L = sum <o, dO> (brute force on tiny inputs)
# ---------------------------------------------------------------------------------------------

def _loss(q, k, v, dO, sigma):
    T, Hq, d = q.shape
    hs = np.repeat(np.arange(Hq, dtype=np.int32), T)
    ts = np.tile(np.arange(T, dtype=np.int64), Hq)
    o, _, _, _ = oracle.rows(q, k, v, None, hs, ts, sigma)
    o = o.reshape(Hq, T, d).transpose(1, 0, 2)
    return float((o * dO).sum())


@pytest.mark.parametrize("Hq,Hkv,d,Lp,Ls", [(2, 1, 8, 5, 3), (4, 2, 4, 3, 4), (3, 3, 5, 0, 6)])
def test_finite_differences(Hq, Hkv, d, Lp, Ls):
    T = Lp + Ls
    rng = np.random.default_rng(7)
    q, k, v, dO = rand_seq(T, Hq, Hkv, d, 0.7, rng)
    sigma = 1.0 / math.sqrt(d)
    r = oracle.fullseq(q, k, v, dO, Lp, sigma)
    dk_total = r["dk"].copy(); dk_total[:Lp] += r["gk"]
    dv_total = r["dv"].copy(); dv_total[:Lp] += r["gv"]
    eps = 1e-5
    for name, x, grad in (("q", q, r["dq"]), ("k", k, dk_total), ("v", v, dv_total)):
        num = np.zeros_like(x)
        it = np.nditer(x, flags=["multi_index"])
        for _ in it:
            idx = it.multi_index
            old = x[idx]
            x[idx] = old + eps; lp = _loss(q, k, v, dO, sigma)
            x[idx] = old - eps; lm = _loss(q, k, v, dO, sigma)
            x[idx] = old
            num[idx] = (lp - lm) / (2 * eps)
        err = np.abs(num - grad).max() / max(np.abs(grad).max(), 1e-30)
        assert err < 1e-6, (name, err)


# ---------------------------------------------------------------------------------------------
# the paper's equivalence invariant against an INDEPENDENT matrix-form
# evaluation of the coupling gradients written here with numpy matmuls
# ---------------------------------------------------------------------------------------------

def coupling_matrix_form(Q2, K1, V1, K2, V2, dO2, sigma):
    """gV1 = P21^T dH2, gK1 = sigma dS21^T Q2, summed over the G heads of a kv head."""
    Ls, Hq, d = Q2.shape
    Lp, Hkv, _ = K1.shape
    G = Hq // Hkv
    gK = np.zeros((Lp, Hkv, d)); gV = np.zeros((Lp, Hkv, d))
    causal = np.tril(np.ones((Ls, Ls), dtype=bool))
    for h in range(Hq):
        g = h // G
        S21 = sigma * Q2[:, h] @ K1[:, g].T
        S22 = np.where(causal, sigma * Q2[:, h] @ K2[:, g].T, -np.inf)
        S = np.concatenate([S21, S22], 1)
        P = np.exp(S - S.max(1, keepdims=True)); P /= P.sum(1, keepdims=True)
        P21, P22 = P[:, :Lp], P[:, Lp:]
        O2 = P21 @ V1[:, g] + P22 @ V2[:, g]
        delta = (dO2[:, h] * O2).sum(1, keepdims=True)
        dS21 = P21 * (dO2[:, h] @ V1[:, g].T - delta)
        gV[:, g] += P21.T @ dO2[:, h]
        gK[:, g] += sigma * dS21.T @ Q2[:, h]
    return gK, gV


@pytest.mark.parametrize("Hq,Hkv,d,Lp,Lss", [(4, 2, 16, 24, (7, 12, 5)), (2, 2, 64, 40, (16, 16))])
def test_equivalence_invariant(Hq, Hkv, d, Lp, Lss):
    inp = I.make_group(I.small_case(Hq, Hkv, d, Lp, Lss, seed=11, dist="unit"))
    N = len(Lss)
    sigma = 1.0 / math.sqrt(d)
    w = [1.0 / N] * N
    # LHS: prefix dK/dV of the summed replays, total over ALL rows in one accumulator
    lhs_k = np.zeros((Lp, Hkv, d)); lhs_v = np.zeros((Lp, Hkv, d))
    gs = np.repeat(np.arange(Hkv, dtype=np.int32), Lp)
    js = np.tile(np.arange(Lp, dtype=np.int64), Hkv)
    for i in range(N):
        q, k, v, dO = oracle.reference.concat_replay(inp, i, w[i])
        r = oracle.fullseq(q, k, v, dO, Lp, sigma)
        a, b = oracle.cols(q, k, v, dO, r["lse"], r["delta"], gs, js, 0, q.shape[0], sigma)
        lhs_k += a.reshape(Hkv, Lp, d).transpose(1, 0, 2)
        lhs_v += b.reshape(Hkv, Lp, d).transpose(1, 0, 2)
    # RHS: own-prefix term (prefix-only attention backward with dO1) + sum_i coupling(i)
    own = oracle.fullseq(inp.Q1, inp.K1, inp.V1, inp.dO1, Lp, sigma)
    rhs_k = own["dk"].copy(); rhs_v = own["dv"].copy()
    for i in range(N):
        gK, gV = coupling_matrix_form(oracle.widen(inp.Q2[i]), oracle.widen(inp.K1),
                                      oracle.widen(inp.V1), oracle.widen(inp.K2[i]),
                                      oracle.widen(inp.V2[i]), oracle.widen(inp.dO2[i]), sigma)
        rhs_k += gK; rhs_v += gV
    assert np.abs(lhs_k - rhs_k).max() < 1e-10
    assert np.abs(lhs_v - rhs_v).max() < 1e-10
    # and the group reducer states the same thing
    ref = oracle.group_reference(inp, w, sigma)
    assert np.abs(ref.dK1 - rhs_k).max() < 1e-10 and np.abs(ref.dV1 - rhs_v).max() < 1e-10
    assert np.abs(ref.dK1_own - own["dk"]).max() < 1e-10


def test_pure_coupling_case():
    """dO1 = 0 (suffix-only loss at the top layer): dQ1 = 0, dK1 = gK1, dV1 = gV1."""
    inp = I.make_group(I.small_case(4, 2, 8, 12, (5, 6), seed=3, dist="unit"))
    inp.dO1 = torch.zeros_like(inp.dO1)
    ref = oracle.group_reference(inp)
    assert np.abs(ref.dQ1).max() == 0.0
    assert np.array_equal(ref.dK1, ref.gK1_after[-1]) and np.array_equal(ref.dV1, ref.gV1_after[-1])


# ---------------------------------------------------------------------------------------------
# prefix isolation: prefix rows do not depend on the suffix
# ---------------------------------------------------------------------------------------------

def test_prefix_isolation():
    inp = I.make_group(I.small_case(4, 2, 16, 20, (9, 3, 14), seed=5, dist="unit"))
    ref = oracle.group_reference(inp, weights=[1.0, 1.0, 1.0])
    alone = oracle.fullseq(inp.Q1, inp.K1, inp.V1, inp.dO1, 20)
    for r in ref.replay:
        assert np.abs(r["o"][:20] - alone["o"]).max() <= 1e-15
        assert np.abs(r["lse"][:, :20] - alone["lse"]).max() <= 1e-15
        assert np.abs(r["dq"][:20] - alone["dq"]).max() <= 1e-15  # weight 1 => same prefix-row dq


# ---------------------------------------------------------------------------------------------
# closed forms
# ---------------------------------------------------------------------------------------------

def test_closed_form_row0_and_zero_q():
    T, Hq, Hkv, d = 9, 4, 2, 6
    G = Hq // Hkv
    q, k, v, dO = rand_seq(T, Hq, Hkv, d)
    sigma = 0.37
    r = oracle.fullseq(q, k, v, dO, 0, sigma)
    for h in range(Hq):
        g = h // G
        assert np.abs(r["o"][0, h] - v[0, g]).max() < 1e-13
        assert abs(r["lse"][h, 0] - sigma * q[0, h] @ k[0, g]) < 1e-13
    # Q = 0: p uniform, o_t = mean(v_<=t), LSE_t = log(t+1), dk = 0, dv_j = sum_h sum_{t>=j} do/(t+1)
    r = oracle.fullseq(np.zeros_like(q), k, v, dO, 0, sigma)
    for t in range(T):
        for h in range(Hq):
            assert np.abs(r["o"][t, h] - v[:t + 1, h // G].mean(0)).max() < 1e-13
            assert abs(r["lse"][h, t] - math.log(t + 1)) < 1e-13
    assert np.abs(r["dk"]).max() < 1e-13
    for j in range(T):
        for g in range(Hkv):
            want = sum(dO[t, h] / (t + 1) for h in range(g * G, (g + 1) * G) for t in range(j, T))
            assert np.abs(r["dv"][j, g] - want).max() < 1e-13


def test_closed_form_equal_keys():
    """All key rows equal => scores constant along each row => ds = p (dp - delta) sums against a
    constant key: dq = sigma * k * sum_j ds_tj = 0."""
    T, Hq, Hkv, d = 7, 2, 1, 5
    q, k, v, dO = rand_seq(T, Hq, Hkv, d)
    k[:] = k[0]
    r = oracle.fullseq(q, k, v, dO, 0)
    assert np.abs(r["dq"]).max() < 1e-13


# ---------------------------------------------------------------------------------------------
# invariants
# ---------------------------------------------------------------------------------------------

def test_softmax_normalisation_and_key_shift():
    T, Hq, Hkv, d, Lp = 11, 4, 2, 8, 6
    q, k, v, dO = rand_seq(T, Hq, Hkv, d)
    sigma = 1.0 / math.sqrt(d)
    # sum_j p_tj = 1: with v = 1 every output is 1
    r1 = oracle.fullseq(q, k, np.ones_like(v), dO, Lp, sigma)
    assert np.abs(r1["o"] - 1.0).max() < 1e-13
    # adding c to every key leaves p, o, dq, dk, dv unchanged and shifts LSE_t by sigma <q_t, c>
    c = RNG.standard_normal(d)
    r = oracle.fullseq(q, k, v, dO, Lp, sigma)
    rs = oracle.fullseq(q, k + c, v, dO, Lp, sigma)
    for name in ("o", "dq", "dk", "dv", "gk", "gv"):
        assert np.abs(r[name] - rs[name]).max() < 1e-12, name
    shift = sigma * np.einsum("thd,d->ht", q, c)
    assert np.abs(rs["lse"] - r["lse"] - shift).max() < 1e-12


def test_lse_merge_identity():
    """Two-source KV logic of Phase B: o2 = merge of (attention over prefix keys only) and
    (causal attention over suffix keys only) weighted by their two LSEs."""
    Hq, Hkv, d, Lp, Ls = 4, 2, 8, 10, 7
    inp = I.make_group(I.small_case(Hq, Hkv, d, Lp, (Ls,), seed=21, dist="unit"))
    q, k, v, dO = oracle.reference.concat_replay(inp, 0, 1.0)
    full = oracle.fullseq(q, k, v, dO, Lp)
    G = Hq // Hkv
    Q2 = oracle.widen(inp.Q2[0]); K1 = oracle.widen(inp.K1); V1 = oracle.widen(inp.V1)
    sigma = 1.0 / math.sqrt(d)
    # suffix-only causal part through the oracle, prefix-only part written out with numpy
    suf = oracle.fullseq(Q2, oracle.widen(inp.K2[0]), oracle.widen(inp.V2[0]),
                         oracle.widen(inp.dO2[0]), 0)
    for h in range(Hq):
        g = h // G
        S21 = sigma * Q2[:, h] @ K1[:, g].T
        lse_p = np.log(np.exp(S21).sum(1))
        o_p = (np.exp(S21 - lse_p[:, None])) @ V1[:, g]
        lse_s = suf["lse"][h]
        lse = np.logaddexp(lse_p, lse_s)
        o = np.exp(lse_p - lse)[:, None] * o_p + np.exp(lse_s - lse)[:, None] * suf["o"][:, h]
        assert np.abs(full["lse"][h, Lp:] - lse).max() < 1e-12
        assert np.abs(full["o"][Lp:, h] - o).max() < 1e-12


# ---------------------------------------------------------------------------------------------
# library special case: torch float64 CPU SDPA + autograd on BASELINE.json config 1
# ---------------------------------------------------------------------------------------------

def _torch_sdpa(q, k, v, dO, sigma):
    T, Hq, d = q.shape
    Hkv = k.shape[1]
    G = Hq // Hkv
    tq = torch.tensor(q).permute(1, 0, 2).contiguous().requires_grad_(True)      # [Hq,T,d]
    tk = torch.tensor(k).permute(1, 0, 2).contiguous().requires_grad_(True)      # [Hkv,T,d]
    tv = torch.tensor(v).permute(1, 0, 2).contiguous().requires_grad_(True)
    ke = tk.repeat_interleave(G, dim=0); ve = tv.repeat_interleave(G, dim=0)
    mask = torch.tril(torch.ones(T, T, dtype=torch.bool))
    o = torch.nn.functional.scaled_dot_product_attention(
        tq[None], ke[None], ve[None], attn_mask=mask, scale=sigma)[0]
    o.backward(torch.tensor(dO).permute(1, 0, 2))
    s = (tq.detach() @ ke.detach().transpose(1, 2)) * sigma
    lse = torch.logsumexp(s.masked_fill(~mask, float("-inf")), dim=-1)
    return (o.detach().permute(1, 0, 2).numpy(), lse.numpy(), tq.grad.permute(1, 0, 2).numpy(),
            tk.grad.permute(1, 0, 2).numpy(), tv.grad.permute(1, 0, 2).numpy())


@pytest.mark.parametrize("case", ["config1", "gqa"])
def test_against_torch_sdpa_float64(case):
    if case == "config1":
        inp = I.make_group(I.config_tiny())
    else:
        inp = I.make_group(I.small_case(6, 2, 16, 50, (13, 9), seed=2, dist="unit"))
    Lp = inp.Q1.shape[0]
    for i in range(len(inp.Q2)):
        q, k, v, dO = oracle.reference.concat_replay(inp, i, 0.25)
        sigma = 1.0 / math.sqrt(q.shape[2])
        r = oracle.fullseq(q, k, v, dO, Lp, sigma)
        o, lse, dq, dk, dv = _torch_sdpa(q, k, v, dO, sigma)
        dk_total = r["dk"].copy(); dk_total[:Lp] += r["gk"]
        dv_total = r["dv"].copy(); dv_total[:Lp] += r["gv"]
        assert np.abs(r["o"] - o).max() < 1e-10
        assert np.abs(r["lse"] - lse).max() < 1e-10
        assert np.abs(r["dq"] - dq).max() < 1e-10
        assert np.abs(dk_total - dk).max() < 1e-10
        assert np.abs(dv_total - dv).max() < 1e-10


# ---------------------------------------------------------------------------------------------
# organisation independence
# ---------------------------------------------------------------------------------------------

def test_organisation_independence():
    inp = I.make_group(I.small_case(4, 2, 8, 14, (5, 9, 7), seed=9, dist="unit"))
    a = oracle.group_reference(inp)
    b = oracle.group_reference(inp, order=[2, 0, 1])
    for name in ("dQ1", "dK1", "dV1"):
        assert np.abs(getattr(a, name) - getattr(b, name)).max() < 1e-12
    assert np.abs(a.gK1_after[2] - b.gK1_after[1]).max() < 1e-12  # both = total over 3 suffixes
    # N = 1: PrefixFlow == one full-sequence pass
    one = I.make_group(I.small_case(4, 2, 8, 14, (6,), seed=9, dist="unit"))
    ref = oracle.group_reference(one)
    q, k, v, dO = oracle.reference.concat_replay(one, 0, 1.0)
    o, lse, dq, dk, dv = _torch_sdpa(q, k, v, dO, 1.0 / math.sqrt(8))
    assert np.abs(np.concatenate([ref.dK1, ref.dK2[0]]) - dk).max() < 1e-12
    assert np.abs(np.concatenate([ref.dV1, ref.dV2[0]]) - dv).max() < 1e-12
    assert np.abs(np.concatenate([ref.dQ1, ref.dQ2[0]]) - dq).max() < 1e-12
    assert np.abs(np.concatenate([ref.O1, ref.O2[0]]) - o).max() < 1e-12


def test_sampled_helpers_agree_with_full():
    inp = I.make_group(I.small_case(4, 2, 8, 20, (9, 6), seed=13, dist="unit"))
    ref = oracle.group_reference(inp)
    s = oracle.sampled_phaseB(inp, 1, 1, [0, 7, 19], [0, 5])
    assert np.abs(s["gk"] - ref.gK1_each[1][[0, 7, 19], 1]).max() < 1e-13
    assert np.abs(s["gv"] - ref.gV1_each[1][[0, 7, 19], 1]).max() < 1e-13
    assert np.abs(s["dk2"] - ref.dK2[1][[0, 5], 1]).max() < 1e-13
    assert np.abs(s["o2"] - ref.O2[1][:, 2:4].transpose(1, 0, 2)).max() < 1e-13
    assert np.abs(s["dq2"] - ref.dQ2[1][:, 2:4].transpose(1, 0, 2)).max() < 1e-13


# ---------------------------------------------------------------------------------------------
# companions: RoPE with continuing positions and the dW_K split
# ---------------------------------------------------------------------------------------------

def test_rope_pins():
    rng = np.random.default_rng(5)
    L, H, d, base = 9, 3, 16, 10000.0
    x = rng.standard_normal((L, H, d))
    pos = np.arange(100, 100 + L)
    y = oracle.rope(x, pos, base)
    # (a) a worked value (tests/golden/rope_worked.txt): d = 2, position 1: the pair is rotated by 1 rad
    g = oracle.rope(np.array([[[1.0, 0.0]]]), [1], base)
    assert abs(g[0, 0, 0] - 0.5403023058681398) < 1e-15 and abs(g[0, 0, 1] - 0.8414709848078965) < 1e-15
    g = oracle.rope(np.array([[[0.0, 1.0]]]), [1], base)      # sign of the cross terms
    assert abs(g[0, 0, 0] + 0.8414709848078965) < 1e-15 and abs(g[0, 0, 1] - 0.5403023058681398) < 1e-15
    # (b) position 0 is the identity; rotations preserve the norm of every (token, head) row
    assert np.abs(oracle.rope(x, np.zeros(L, dtype=int), base) - x).max() == 0.0
    assert np.abs(np.linalg.norm(y, axis=-1) - np.linalg.norm(x, axis=-1)).max() < 1e-13
    # (c) independent route: pair (x_j, x_{j+d/2}) as a complex number times e^{i a}; the frequency of
    # pair j is base^(-2j/d): pair 0 turns by `position` radians, the last pair slowest
    z = (x[..., : d // 2] + 1j * x[..., d // 2:]) * np.exp(
        1j * pos[:, None, None] * base ** (-np.arange(d // 2) / (d // 2)))
    assert np.abs(np.concatenate([z.real, z.imag], -1) - y).max() < 1e-12
    # (d) the relative-position property that makes continuing positions matter:
    # <R_m q, R_n k> depends on m - n only, and differs if the suffix restarted at 0
    q, k = rng.standard_normal((1, 1, d)), rng.standard_normal((1, 1, d))
    dot = lambda m, n: float((oracle.rope(q, [m], base) * oracle.rope(k, [n], base)).sum())
    assert abs(dot(1000, 993) - dot(7, 0)) < 1e-11 and abs(dot(1000, 993) - dot(0, 993)) > 1e-3
    # (e) inverse is the transpose: R^T R = I and <R x, g> = <x, R^T g> (the backward of a linear map)
    gy = rng.standard_normal((L, H, d))
    assert np.abs(oracle.rope(y, pos, base, inverse=True) - x).max() < 1e-13
    assert abs((y * gy).sum() - (x * oracle.rope(gy, pos, base, inverse=True)).sum()) < 1e-11
    # (f) torch, rotate-half formulation in fp64 (how the HF Llama / Qwen code applies it)
    xt = torch.tensor(x)
    inv = base ** (-torch.arange(0, d, 2, dtype=torch.float64) / d)
    ang = torch.tensor(pos, dtype=torch.float64)[:, None] * inv[None]
    cos, sin = torch.cat([ang.cos(), ang.cos()], -1)[:, None], torch.cat([ang.sin(), ang.sin()], -1)[:, None]
    rot = torch.cat([-xt[..., d // 2:], xt[..., : d // 2]], -1)
    assert np.abs((xt * cos + rot * sin).numpy() - y).max() < 1e-13


def test_kv_proj_grad_split_equals_full_sequence_replays():
    """dW_K = X1^T dK1 + sum_i X2(i)^T dK2(i) with the Phase-C dK1 (which already holds
    every gK1(i)) equals the baseline's sum over the N full-sequence replays of [X1; X2(i)]^T dK(i)."""
    inp = I.make_group(I.small_case(4, 2, 8, 11, (5, 7, 3), seed=21, dist="unit"))
    ref = oracle.group_reference(inp)
    rng = np.random.default_rng(3)
    dm, N = 6, 3
    X1 = rng.standard_normal((11, dm))
    X2 = [rng.standard_normal((L, dm)) for L in (5, 7, 3)]
    split = oracle.kv_proj_grad(X1, ref.dK1, X2, ref.dK2)
    full = np.zeros_like(split)
    for i in range(N):
        q, k, v, dO = oracle.reference.concat_replay(inp, i, 1.0 / N)
        r = oracle.fullseq(q, k, v, dO)
        full += np.concatenate([X1, X2[i]]).T @ r["dk"].reshape(11 + X2[i].shape[0], -1)
    assert np.abs(split - full).max() < 1e-10 * max(1.0, np.abs(full).max())
    # closed form: one token, one head: dW = outer(x, dk)
    one = oracle.kv_proj_grad(np.array([[2.0, 3.0]]), np.array([[[1.0, -1.0]]]), [], [])
    assert np.array_equal(one, np.array([[2.0, -2.0], [3.0, -3.0]]))
