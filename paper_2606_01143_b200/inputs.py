"""Seeded synthetic rollout groups [P||S(1)] ... [P||S(N)] (shapes from BASELINE.json configs).

This module is the ONLY code shared by the CUDA path and the oracle. It holds no arithmetic of
the method: it draws Gaussian tensors, scales them, rounds to bf16 and names the shapes.

Recipe: torch CPU generator; prefix tensors
Q1, K1, V1, dO1 are drawn from seed `base`; suffix i draws its length (ragged configs only:
randint(lo, hi+1)) and then Q2, K2, V2, dO2 from seed `base + 1 + i`; every tensor is
fp32 randn * scale -> bf16 (round to nearest even). scale = 1/sqrt(d) ("std", the BASELINE.json
distribution) or 1 ("unit", the unit-logit distribution of SURVEY.md §8c reading 16).
"spike" is the adversarial-logit variant of "unit" (real attention has sinks and retrieval hits):
a fixed +-1 direction u per KV head is added to every query row and, with growing multipliers,
to a few key rows late in the prefix and late in every suffix, so that the scaled score of those
keys exceeds everything before them by ~0.75 sqrt(d) nats (> 8 in log2 units) for EVERY row --
an online softmax must re-reference its running maximum there, several tiles into the sequence.
"ramp" adds a * u to every query row and a * (position / T) * u to key row `position` (prefix
positions 0..Lp-1, suffix positions continue at Lp; T = Lp + longest suffix; a = sqrt(RAMP_NATS /
sqrt(d)) ~ 1.5): the scaled scores of every row grow linearly by RAMP_NATS = 24 nats (35 log2 units)
over the sequence, so the running maximum is re-referenced ~4 times per row, spread over the whole
KV loop, while the softmax mass stays on many recent keys and the gradients keep a healthy
magnitude.  The planted component is kept at ~1.5x the noise on purpose: a key (query) component of
norm a multiplies the bf16 rounding of dS into dQ (dK) by a, which is rounding of the bf16
contract, not of a kernel.
Layout is token-major [L, H, d] with d contiguous (SURVEY.md §8c reading 7).

The paper measures on Llama3-8B / Qwen3-8B with MuSiQue RAG prompts and synthetic length sweeps
(PAPER.md:335, 365); these tensors stand in for those workloads: attention cost depends on shapes
only.
"""
from __future__ import annotations

import dataclasses
import math
from typing import List, Optional, Sequence

import torch


@dataclasses.dataclass
class GroupShape:
    """One rollout group: a shared prefix of Lp tokens and N suffixes."""

    name: str
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    Lp: int
    Ls: List[int]
    seed: int = 0
    dist: str = "std"  # "std": N(0,1)/sqrt(d);  "unit": N(0,1);  "spike" / "ramp": unit + planted keys

    @property
    def N(self) -> int:
        return len(self.Ls)

    @property
    def G(self) -> int:
        return self.n_q_heads // self.n_kv_heads


@dataclasses.dataclass
class GroupInputs:
    shape: GroupShape
    Q1: torch.Tensor  # [Lp, Hq, d] bf16
    K1: torch.Tensor  # [Lp, Hkv, d]
    V1: torch.Tensor
    dO1: torch.Tensor  # [Lp, Hq, d]
    Q2: List[torch.Tensor]  # each [Ls_i, Hq, d]
    K2: List[torch.Tensor]
    V2: List[torch.Tensor]
    dO2: List[torch.Tensor]


def _draw(gen: torch.Generator, L: int, H: int, d: int, scale: float,
          add: Optional[torch.Tensor] = None) -> torch.Tensor:
    x = torch.randn((L, H, d), generator=gen, dtype=torch.float32) * scale
    if add is not None:
        x = x + add
    return x.to(torch.bfloat16)


# "spike": planted key rows as (fraction of the sequence length, multiplier of u); multipliers
# grow by 0.75 so that each planted key beats the previous one by 0.75 sqrt(d) nats in every row
SPIKE_PREFIX = ((0.30, 1.00), (0.62, 1.75), (0.97, 2.50))
SPIKE_SUFFIX = ((0.45, 3.25), (0.93, 4.00))


def spike_rows(L: int, plan) -> List[tuple]:
    """(row, multiplier) of the planted keys of a sequence of L tokens."""
    return [(min(L - 1, int(f * L)), m) for f, m in plan] if L > 0 else []


def _spike_direction(seed: int, Hkv: int, d: int) -> torch.Tensor:
    g = torch.Generator(device="cpu")
    g.manual_seed(seed + 999983)
    return (torch.randint(0, 2, (Hkv, d), generator=g).to(torch.float32) * 2.0 - 1.0)


RAMP_NATS = 24.0


def ramp_amplitude(d: int) -> float:
    return math.sqrt(RAMP_NATS / math.sqrt(d))


def _key_ramp(u: torch.Tensor, L: int, pos0: int, T: int, d: int) -> torch.Tensor:
    a = torch.arange(pos0, pos0 + L, dtype=torch.float32) * (ramp_amplitude(d) / max(1, T))
    return a.view(L, 1, 1) * u.view(1, *u.shape)


def _key_spikes(u: torch.Tensor, L: int, plan) -> torch.Tensor:
    add = torch.zeros((L,) + tuple(u.shape), dtype=torch.float32)
    for row, m in spike_rows(L, plan):
        add[row] = m * u
    return add


RAGGED_LO, RAGGED_HI = 256, 2048  # BASELINE.json configs[2]: lengths uniform in [256, 2048]


def ragged_lengths(seed: int, n: int) -> List[int]:
    """Suffix i draws its length as the first value of its own stream, seed `seed + 1 + i`."""
    out = []
    for i in range(n):
        g = torch.Generator(device="cpu")
        g.manual_seed(seed + 1 + i)
        out.append(int(torch.randint(RAGGED_LO, RAGGED_HI + 1, (1,), generator=g).item()))
    return out


def make_group(shape: GroupShape, only_suffixes: Optional[Sequence[int]] = None) -> GroupInputs:
    """Draw the tensors of one group. `only_suffixes` limits which suffixes are materialised
    (the others are left as empty placeholders) without changing any drawn value."""
    Hq, Hkv, d = shape.n_q_heads, shape.n_kv_heads, shape.head_dim
    if shape.dist not in ("std", "unit", "spike", "ramp"):
        raise ValueError(f"unknown dist {shape.dist!r}")
    scale = 1.0 / math.sqrt(d) if shape.dist == "std" else 1.0
    uq = k1_add = None
    if shape.dist in ("spike", "ramp"):
        u = _spike_direction(shape.seed, Hkv, d)                     # [Hkv, d]
        uq = u.repeat_interleave(Hq // Hkv, 0)                       # query head h -> u[h // G]
        T = shape.Lp + max(shape.Ls, default=0)
        if shape.dist == "ramp":
            uq = uq * ramp_amplitude(d)
        k1_add = (_key_spikes(u, shape.Lp, SPIKE_PREFIX) if shape.dist == "spike"
                  else _key_ramp(u, shape.Lp, 0, T, d))
    g = torch.Generator(device="cpu")
    g.manual_seed(shape.seed)
    Q1 = _draw(g, shape.Lp, Hq, d, scale, uq)
    K1 = _draw(g, shape.Lp, Hkv, d, scale, k1_add)
    V1 = _draw(g, shape.Lp, Hkv, d, scale)
    dO1 = _draw(g, shape.Lp, Hq, d, scale)
    Q2, K2, V2, dO2 = [], [], [], []
    for i, Ls in enumerate(shape.Ls):
        if only_suffixes is not None and i not in only_suffixes:
            e = torch.empty((0, Hq, d), dtype=torch.bfloat16)
            ek = torch.empty((0, Hkv, d), dtype=torch.bfloat16)
            Q2.append(e), K2.append(ek), V2.append(ek), dO2.append(e)
            continue
        gi = torch.Generator(device="cpu")
        gi.manual_seed(shape.seed + 1 + i)
        # every suffix stream starts with its length draw (used by the ragged config only)
        torch.randint(RAGGED_LO, RAGGED_HI + 1, (1,), generator=gi)
        Q2.append(_draw(gi, Ls, Hq, d, scale, uq))
        k2_add = None
        if shape.dist == "spike":
            k2_add = _key_spikes(u, Ls, SPIKE_SUFFIX)
        elif shape.dist == "ramp":
            k2_add = _key_ramp(u, Ls, shape.Lp, T, d)
        K2.append(_draw(gi, Ls, Hkv, d, scale, k2_add))
        V2.append(_draw(gi, Ls, Hkv, d, scale))
        dO2.append(_draw(gi, Ls, Hq, d, scale))
    return GroupInputs(shape, Q1, K1, V1, dO1, Q2, K2, V2, dO2)


# ----------------------------------------------------------------------------------------------
# BASELINE.json configs (index = position in BASELINE.json "configs")
# ----------------------------------------------------------------------------------------------

def config_tiny(dist: str = "std") -> GroupShape:
    """configs[0]: 2q/2kv heads, d=64, prefix 256, N=4 suffixes of 64 tokens, seed 0."""
    return GroupShape("tiny", 2, 2, 64, 256, [64] * 4, seed=0, dist=dist)


def config_7b(dist: str = "std") -> GroupShape:
    """configs[1]: 28q/4kv (GQA 7:1), d=128, prefix 5120, N=8 suffixes of 1024 (83% prefix)."""
    return GroupShape("7b-83pct", 28, 4, 128, 5120, [1024] * 8, seed=1000, dist=dist)


def config_ragged(dist: str = "std") -> GroupShape:
    """configs[2]: 28q/4kv, d=128, prefix 16384, N=16, suffix lengths uniform in [256, 2048]."""
    seed = 2000
    return GroupShape("ragged-rag", 28, 4, 128, 16384, ragged_lengths(seed, 16),
                      seed=seed, dist=dist)


SWEEP_RATIOS = {20: 1664, 50: 4096, 83: 6784, 95: 7808}  # prefix length at total 8192 (x128)
SWEEP_N = (2, 4, 8, 16)


def config_sweep(ratio_pct: int, n: int, dist: str = "std", total: int = 8192) -> GroupShape:
    """configs[3]: 32q/8kv, d=128, total length 8192 per trajectory, prefix ratio x group size."""
    Lp = SWEEP_RATIOS[ratio_pct] if total == 8192 else (total * ratio_pct // 100) // 128 * 128
    return GroupShape(f"sweep-r{ratio_pct}-n{n}", 32, 8, 128, Lp, [total - Lp] * n,
                      seed=3000 + 10 * ratio_pct + n, dist=dist)


def config_32k(dist: str = "std") -> GroupShape:
    """configs[4]: 40q/8kv, d=128, prefix 32768, N=8 suffixes of 2048 (memory stress)."""
    return GroupShape("32k-stress", 40, 8, 128, 32768, [2048] * 8, seed=4000, dist=dist)


def small_case(Hq: int, Hkv: int, d: int, Lp: int, Ls: Sequence[int], seed: int = 7,
               dist: str = "std") -> GroupShape:
    return GroupShape("case", Hq, Hkv, d, Lp, list(Ls), seed=seed, dist=dist)
