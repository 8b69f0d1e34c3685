"""Shared helpers of the GPU parity tests: tolerance gates and group-level comparison.

Gates (SURVEY.md §8c readings 15-16):
  official  max|err| <= 1e-2 * max|ref| + 1e-3                      (BASELINE.json north_star)
  strict    max|err| <= 1e-2 * max|ref|   and   ||err||_2 <= 5e-3 * ||ref||_2   (build-owned)
  LSE       max|err| <= 1e-3 absolute
"""
from __future__ import annotations

import numpy as np
import torch

OFFICIAL_REL, OFFICIAL_ABS = 1e-2, 1e-3
STRICT_MAX_REL, STRICT_RMS_REL = 1e-2, 5e-3
LSE_ABS = 1e-3


def to_np(x) -> np.ndarray:
    if isinstance(x, torch.Tensor):
        return x.detach().to("cpu").to(torch.float64).numpy()
    return np.asarray(x, dtype=np.float64)


def check(name: str, got, ref, lse: bool = False, strict: bool = True) -> dict:
    """Assert the gates for one tensor; return the measured errors."""
    got, ref = to_np(got), to_np(ref)
    assert got.shape == ref.shape, f"{name}: shape {got.shape} vs {ref.shape}"
    assert np.isfinite(got).all(), f"{name}: non-finite values in GPU output"
    if ref.size == 0:
        return dict(name=name, max_err=0.0, max_ref=0.0, rms_rel=0.0)
    err = np.abs(got - ref)
    max_err, max_ref = float(err.max()), float(np.abs(ref).max())
    rms_ref = float(np.sqrt((ref ** 2).sum()))
    rms_rel = float(np.sqrt((err ** 2).sum())) / rms_ref if rms_ref > 0 else 0.0
    res = dict(name=name, max_err=max_err, max_ref=max_ref, rms_rel=rms_rel)
    assert max_err <= OFFICIAL_REL * max_ref + OFFICIAL_ABS, f"official gate failed: {res}"
    if lse:
        assert max_err <= LSE_ABS, f"LSE gate failed: {res}"
    elif strict:
        if max_ref > 0:
            assert max_err <= STRICT_MAX_REL * max_ref, f"strict max gate failed: {res}"
            assert rms_rel <= STRICT_RMS_REL, f"strict rms gate failed: {res}"
        else:
            assert max_err == 0.0, f"reference is exactly zero but GPU is not: {res}"
    return res


def compare_group(g, ref, gk_snapshots=None, order=None) -> list:
    """DeviceGroup outputs (after run_prefixflow_step) vs oracle GroupReference."""
    out = []
    out.append(check("O1", g.O1, ref.O1))
    out.append(check("LSE1", g.LSE1, ref.LSE1, lse=True))
    for i in range(len(g.Ls)):
        out.append(check(f"O2[{i}]", g.O2[i], ref.O2[i]))
        out.append(check(f"LSE2[{i}]", g.LSE2[i], ref.LSE2[i], lse=True))
        out.append(check(f"dQ2[{i}]", g.dQ2[i], ref.dQ2[i]))
        out.append(check(f"dK2[{i}]", g.dK2[i], ref.dK2[i]))
        out.append(check(f"dV2[{i}]", g.dV2[i], ref.dV2[i]))
    if gk_snapshots is not None:
        for i, (gk, gv) in gk_snapshots.items():
            out.append(check(f"gK1 after suffix {i}", gk, ref.gK1_after[i]))
            out.append(check(f"gV1 after suffix {i}", gv, ref.gV1_after[i]))
    out.append(check("dQ1", g.dQ1, ref.dQ1))
    out.append(check("dK1", g.dK1, ref.dK1))
    out.append(check("dV1", g.dV1, ref.dV1))
    return out
