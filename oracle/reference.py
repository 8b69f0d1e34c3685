"""Python face of the fp64 oracle (oracle/pf_oracle.c).  TEST INFRASTRUCTURE, not product.

`fullseq` evaluates the definition on one concatenated
trajectory [P || S(i)]; `group_reference` runs the N replays of a rollout group and reduces them
into the values each C-ABI call must produce (table in DESIGN.md "Oracle"):

    O1, LSE1            rows t <  Lp of any replay (identical for all i)
    O2(i), LSE2(i)      rows t >= Lp of replay i
    dQ2(i), dK2(i), dV2(i)   rows / keys >= Lp of replay i
    gK1, gV1 after k suffixes   sum_{i<=k} coupling accumulators (keys < Lp, rows >= Lp)
    dQ1, dK1, dV1       sum_i of prefix rows / keys over the N replays, where replay i uses the
                        prefix-row adjoint w_i * dO1, sum_i w_i = 1 (reading 1)

All arithmetic happens in pf_oracle.c in fp64; this file only marshals arrays, slices and adds.
"""
from __future__ import annotations

import ctypes
import dataclasses
import math
import os
import subprocess
from typing import Dict, List, Optional, Sequence

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pf_oracle.c")
_SO = os.path.join(_HERE, "libpf_oracle.so")
_lib = None


class _Shape(ctypes.Structure):
    _fields_ = [("T", ctypes.c_int64), ("Hq", ctypes.c_int32), ("Hkv", ctypes.c_int32),
                ("d", ctypes.c_int32), ("sigma", ctypes.c_double)]


def build(force: bool = False) -> str:
    """Compile pf_oracle.c with gcc (plain -O2, OpenMP). Building the checker is not using it."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", _SO, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        L.pfo_rows.restype = ctypes.c_int
        L.pfo_rows.argtypes = [ctypes.POINTER(_Shape), dp, dp, dp, dp, ctypes.c_int64,
                               ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int64),
                               dp, dp, dp, dp]
        L.pfo_cols.restype = ctypes.c_int
        L.pfo_cols.argtypes = [ctypes.POINTER(_Shape), dp, dp, dp, dp, dp, dp, ctypes.c_int64,
                               ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int64),
                               ctypes.c_int64, ctypes.c_int64, dp, dp]
        L.pfo_max_threads.restype = ctypes.c_int
        _lib = L
    return _lib


def max_threads() -> int:
    return int(lib().pfo_max_threads())


def widen(x) -> np.ndarray:
    """bf16 / fp32 torch tensor (or array) -> contiguous float64 numpy array, exactly."""
    if isinstance(x, torch.Tensor):
        x = x.detach().cpu().to(torch.float64).numpy()
    return np.ascontiguousarray(x, dtype=np.float64)


def _p(a: Optional[np.ndarray]):
    if a is None:
        return None
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _shape(T, Hq, Hkv, d, sigma):
    return _Shape(int(T), int(Hq), int(Hkv), int(d), float(sigma))


def rows(q, k, v, dO, hs, ts, sigma=None):
    """o, lse, delta, dq for the listed (h, t) rows of one sequence. q,dO [T,Hq,d]; k,v [T,Hkv,d]."""
    T, Hq, d = q.shape
    Hkv = k.shape[1]
    sigma = 1.0 / math.sqrt(d) if sigma is None else sigma
    hs = np.ascontiguousarray(hs, dtype=np.int32)
    ts = np.ascontiguousarray(ts, dtype=np.int64)
    n = len(hs)
    o = np.empty((n, d)); lse = np.empty(n); delta = np.empty(n); dq = np.empty((n, d))
    sh = _shape(T, Hq, Hkv, d, sigma)
    rc = lib().pfo_rows(ctypes.byref(sh), _p(q), _p(k), _p(v), _p(dO), n,
                        hs.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)),
                        ts.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)),
                        _p(o), _p(lse), _p(delta), _p(dq))
    if rc != 0:
        raise ValueError("pfo_rows: bad argument")
    if dO is None:
        return o, lse, None, None
    return o, lse, delta, dq


def cols(q, k, v, dO, lse, delta, gs, js, r0, r1, sigma=None):
    """dk, dv of the listed (g, j) key columns from rows max(j, r0) <= t < r1. lse, delta [Hq,T]."""
    T, Hq, d = q.shape
    Hkv = k.shape[1]
    sigma = 1.0 / math.sqrt(d) if sigma is None else sigma
    gs = np.ascontiguousarray(gs, dtype=np.int32)
    js = np.ascontiguousarray(js, dtype=np.int64)
    n = len(gs)
    dk = np.empty((n, d)); dv = np.empty((n, d))
    sh = _shape(T, Hq, Hkv, d, sigma)
    lse = np.ascontiguousarray(lse, dtype=np.float64)
    delta = np.ascontiguousarray(delta, dtype=np.float64)
    assert lse.shape == (Hq, T) and delta.shape == (Hq, T)
    rc = lib().pfo_cols(ctypes.byref(sh), _p(q), _p(k), _p(v), _p(dO), _p(lse), _p(delta), n,
                        gs.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)),
                        js.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)),
                        int(r0), int(r1), _p(dk), _p(dv))
    if rc != 0:
        raise ValueError("pfo_cols: bad argument")
    return dk, dv


def fullseq(q, k, v, dO, Lp: int = 0, sigma=None) -> Dict[str, np.ndarray]:
    """Full-sequence causal attention forward + backward on one [P || S] of T tokens.

    Returns o [T,Hq,d], lse [Hq,T], delta [Hq,T], dq [T,Hq,d], and for the keys two accumulators
    kept apart: dk/dv [T,Hkv,d] = contributions of rows t < Lp to keys j < Lp
    ("own-prefix term") and of rows t >= Lp to keys j >= Lp (suffix keys); gk/gv [Lp,Hkv,d] =
    contributions of rows t >= Lp to keys j < Lp (the coupling gradients of PAPER.md:196).
    The textbook full-sequence gradient of a prefix key is dk[:Lp] + gk.
    """
    q, k, v, dO = widen(q), widen(k), widen(v), widen(dO)
    T, Hq, d = q.shape
    Hkv = k.shape[1]
    hs = np.repeat(np.arange(Hq, dtype=np.int32), T)
    ts = np.tile(np.arange(T, dtype=np.int64), Hq)
    o, lse, delta, dq = rows(q, k, v, dO, hs, ts, sigma)
    o = np.ascontiguousarray(o.reshape(Hq, T, d).transpose(1, 0, 2))
    dq = np.ascontiguousarray(dq.reshape(Hq, T, d).transpose(1, 0, 2))
    lse = lse.reshape(Hq, T)
    delta = delta.reshape(Hq, T)
    dk = np.zeros((T, Hkv, d)); dv = np.zeros((T, Hkv, d))
    gk = np.zeros((Lp, Hkv, d)); gv = np.zeros((Lp, Hkv, d))
    # own-prefix term: keys < Lp, rows < Lp
    if Lp > 0:
        gs = np.repeat(np.arange(Hkv, dtype=np.int32), Lp)
        js = np.tile(np.arange(Lp, dtype=np.int64), Hkv)
        a, b = cols(q, k, v, dO, lse, delta, gs, js, 0, Lp, sigma)
        dk[:Lp] = a.reshape(Hkv, Lp, d).transpose(1, 0, 2)
        dv[:Lp] = b.reshape(Hkv, Lp, d).transpose(1, 0, 2)
        if T > Lp:  # coupling: keys < Lp, rows >= Lp
            a, b = cols(q, k, v, dO, lse, delta, gs, js, Lp, T, sigma)
            gk[:] = a.reshape(Hkv, Lp, d).transpose(1, 0, 2)
            gv[:] = b.reshape(Hkv, Lp, d).transpose(1, 0, 2)
    if T > Lp:  # suffix keys
        Ls = T - Lp
        gs = np.repeat(np.arange(Hkv, dtype=np.int32), Ls)
        js = np.tile(np.arange(Lp, T, dtype=np.int64), Hkv)
        a, b = cols(q, k, v, dO, lse, delta, gs, js, Lp, T, sigma)
        dk[Lp:] = a.reshape(Hkv, Ls, d).transpose(1, 0, 2)
        dv[Lp:] = b.reshape(Hkv, Ls, d).transpose(1, 0, 2)
    return dict(o=o, lse=lse, delta=delta, dq=dq, dk=dk, dv=dv, gk=gk, gv=gv)


@dataclasses.dataclass
class GroupReference:
    O1: np.ndarray; LSE1: np.ndarray
    O2: List[np.ndarray]; LSE2: List[np.ndarray]
    dQ2: List[np.ndarray]; dK2: List[np.ndarray]; dV2: List[np.ndarray]
    gK1_after: List[np.ndarray]; gV1_after: List[np.ndarray]   # cumulative, after suffix i
    gK1_each: List[np.ndarray]; gV1_each: List[np.ndarray]     # coupling of suffix i alone
    dQ1: np.ndarray; dK1: np.ndarray; dV1: np.ndarray
    dK1_own: np.ndarray; dV1_own: np.ndarray
    replay: List[Dict[str, np.ndarray]]


def concat_replay(inp, i: int, w: float):
    """[P || S(i)] inputs of replay i; prefix-row adjoint = w * dO1 (reading 1)."""
    q = np.concatenate([widen(inp.Q1), widen(inp.Q2[i])], 0)
    k = np.concatenate([widen(inp.K1), widen(inp.K2[i])], 0)
    v = np.concatenate([widen(inp.V1), widen(inp.V2[i])], 0)
    dO = np.concatenate([w * widen(inp.dO1), widen(inp.dO2[i])], 0)
    return q, k, v, dO


def group_reference(inp, weights: Optional[Sequence[float]] = None, sigma=None,
                    order: Optional[Sequence[int]] = None) -> GroupReference:
    """N full-sequence replays of a rollout group, reduced to what each C-ABI call must produce."""
    N = len(inp.Q2)
    Lp = inp.Q1.shape[0]
    if weights is None:
        weights = [1.0 / N] * N if N > 0 else []
    order = list(range(N)) if order is None else list(order)
    rep = [None] * N
    for i in order:
        q, k, v, dO = concat_replay(inp, i, weights[i])
        rep[i] = fullseq(q, k, v, dO, Lp, sigma)
    Hq, d = inp.Q1.shape[1], inp.Q1.shape[2]
    Hkv = inp.K1.shape[1]
    if N == 0:
        r = fullseq(widen(inp.Q1), widen(inp.K1), widen(inp.V1), widen(inp.dO1), Lp, sigma)
        return GroupReference(r["o"], r["lse"], [], [], [], [], [], [], [], [], [],
                              r["dq"], r["dk"], r["dv"], r["dk"], r["dv"], [])
    O1 = rep[order[0]]["o"][:Lp]; LSE1 = rep[order[0]]["lse"][:, :Lp]
    gk_acc = np.zeros((Lp, Hkv, d)); gv_acc = np.zeros((Lp, Hkv, d))
    gK_after = [None] * N; gV_after = [None] * N
    dQ1 = np.zeros((Lp, Hq, d)); dK_own = np.zeros((Lp, Hkv, d)); dV_own = np.zeros((Lp, Hkv, d))
    for i in order:
        gk_acc = gk_acc + rep[i]["gk"]; gv_acc = gv_acc + rep[i]["gv"]
        gK_after[i] = gk_acc.copy(); gV_after[i] = gv_acc.copy()
        dQ1 += rep[i]["dq"][:Lp]; dK_own += rep[i]["dk"][:Lp]; dV_own += rep[i]["dv"][:Lp]
    return GroupReference(
        O1=O1, LSE1=LSE1,
        O2=[r["o"][Lp:] for r in rep], LSE2=[r["lse"][:, Lp:] for r in rep],
        dQ2=[r["dq"][Lp:] for r in rep], dK2=[r["dk"][Lp:] for r in rep],
        dV2=[r["dv"][Lp:] for r in rep],
        gK1_after=gK_after, gV1_after=gV_after,
        gK1_each=[r["gk"] for r in rep], gV1_each=[r["gv"] for r in rep],
        dQ1=dQ1, dK1=dK_own + gk_acc, dV1=dV_own + gv_acc, dK1_own=dK_own, dV1_own=dV_own,
        replay=rep)


# ----------------------------------------------------------------------------------------------
# Sampled evaluation for full-size configs (the oracle computes the sampled outputs one by one)
# ----------------------------------------------------------------------------------------------

def sampled_rows(q, k, v, dO, hs, ts, sigma=None):
    """o, lse, delta, dq of sampled (h, t) rows of one sequence (inputs any dtype; widened)."""
    return rows(widen(q), widen(k), widen(v), None if dO is None else widen(dO), hs, ts, sigma)


def sampled_phaseB(inp, i: int, g: int, prefix_js: Sequence[int], suffix_js: Sequence[int],
                   sigma=None):
    """For suffix i and ONE kv head g: coupling gK1/gV1 at sampled prefix keys and dK2/dV2 at
    sampled suffix keys (suffix-local indices). Needs the row statistics of every suffix row of the
    G heads of group g; returns those rows too (O2, LSE2, dQ2 of heads g*G..g*G+G-1)."""
    q, k, v, dO = concat_replay(inp, i, 0.0)
    T, Hq, d = q.shape
    Hkv = k.shape[1]
    G = Hq // Hkv
    Lp = inp.Q1.shape[0]
    Ls = T - Lp
    heads = np.arange(g * G, (g + 1) * G, dtype=np.int32)
    hs = np.repeat(heads, Ls)
    ts = np.tile(np.arange(Lp, T, dtype=np.int64), G)
    o, lse, delta, dq = rows(q, k, v, dO, hs, ts, sigma)
    lse_full = np.full((Hq, T), np.nan); delta_full = np.full((Hq, T), np.nan)
    lse_full[g * G:(g + 1) * G, Lp:] = lse.reshape(G, Ls)
    delta_full[g * G:(g + 1) * G, Lp:] = delta.reshape(G, Ls)
    pj = np.asarray(prefix_js, dtype=np.int64)
    sj = np.asarray(suffix_js, dtype=np.int64) + Lp
    gk, gv = cols(q, k, v, dO, lse_full, delta_full, np.full(len(pj), g, np.int32), pj, Lp, T, sigma)
    dk2, dv2 = cols(q, k, v, dO, lse_full, delta_full, np.full(len(sj), g, np.int32), sj, Lp, T, sigma)
    return dict(gk=gk, gv=gv, dk2=dk2, dv2=dv2,
                o2=o.reshape(G, Ls, d), lse2=lse.reshape(G, Ls), dq2=dq.reshape(G, Ls, d),
                heads=heads)
