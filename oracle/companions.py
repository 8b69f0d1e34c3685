"""fp64 oracle of the two companions of the attention path.  TEST INFRASTRUCTURE, not product.

rope           rotary position embedding with the position continuing after the prefix
               ("RoPE positions for suffix tokens continue after the prefix length
               rather than restarting from zero"); the definition of the rotate-half convention
               used by the models the paper trains (Llama 3 / Qwen 3):
                   theta_j = base^(-2 j / d),  j = 0 .. d/2 - 1,   a = position * theta_j
                   y[j]       = x[j] cos a - x[j + d/2] sin a
                   y[j + d/2] = x[j + d/2] cos a + x[j] sin a
               inverse = the transpose rotation (a -> -a): the backward of the map, dX = R^T dY.
kv_proj_grad   the parameter-gradient split of PAPER.md:212:
                   dW_K = X1^T dK1 + sum_i X2(i)^T dK2(i)
               written out as plain matrix products.

Plain numpy, one formula per line, no blocking.  Pins in tests/test_oracle_pins.py.
"""
from __future__ import annotations

from typing import Sequence

import numpy as np


def rope(x: np.ndarray, positions: Sequence[int], base: float = 10000.0, inverse: bool = False) -> np.ndarray:
    """x [L, H, d] (any float dtype, widened to fp64), positions [L] -> rotated copy, fp64."""
    x = np.asarray(x, dtype=np.float64)
    L, H, d = x.shape
    half = d // 2
    y = np.empty_like(x)
    for t in range(L):
        for j in range(half):
            a = float(positions[t]) * base ** (-2.0 * j / d)
            if inverse:
                a = -a
            c, s = np.cos(a), np.sin(a)
            y[t, :, j] = x[t, :, j] * c - x[t, :, j + half] * s
            y[t, :, j + half] = x[t, :, j + half] * c + x[t, :, j] * s
    return y


def kv_proj_grad(X1: np.ndarray, dK1: np.ndarray, X2: Sequence[np.ndarray], dK2: Sequence[np.ndarray],
                 alpha: Sequence[float] = None) -> np.ndarray:
    """dW [dm, Hkv*d] = X1^T dK1 + sum_i alpha_i X2(i)^T dK2(i); dK* are [L, Hkv, d]."""
    X1 = np.asarray(X1, dtype=np.float64)
    dW = X1.T @ np.asarray(dK1, dtype=np.float64).reshape(X1.shape[0], -1)
    for i, (x, g) in enumerate(zip(X2, dK2)):
        x = np.asarray(x, dtype=np.float64)
        a = 1.0 if alpha is None else float(alpha[i])
        dW = dW + a * (x.T @ np.asarray(g, dtype=np.float64).reshape(x.shape[0], -1))
    return dW
