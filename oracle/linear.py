"""ORACLE (test infrastructure) — S7 reference: the UNSHARDED linear layer Y = X W^T in fp64.

PAPER.md:45, :92-94 — ETP shards "attention and linear layers" with unequal widths; a correct resharded
state must compute the same layer output as the unsharded weight.  This is the textbook definition
(no sharding, no blocking); numpy's matmul is the library routine, pinned against an explicit triple loop
in tests/test_oracle_linear.py.
"""
from __future__ import annotations

import numpy as np


def decode16(u8: np.ndarray, dtype: str) -> np.ndarray:
    """Exact upcast of little-endian 16-bit floats (given as bytes) to fp64."""
    u16 = np.ascontiguousarray(u8).view(np.uint16)
    if dtype == "fp16":
        return u16.view(np.float16).astype(np.float64)
    if dtype == "bf16":
        return (u16.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    raise ValueError(dtype)


def linear_ref(x: np.ndarray, w: np.ndarray) -> np.ndarray:
    """x [T][K], w [N][K] (fp64) -> y [T][N] = x @ w.T"""
    return np.asarray(x, dtype=np.float64) @ np.asarray(w, dtype=np.float64).T


def linear_triple_loop(x: np.ndarray, w: np.ndarray) -> np.ndarray:
    T, K = x.shape
    N = w.shape[0]
    y = np.zeros((T, N), dtype=np.float64)
    for t in range(T):
        for n in range(N):
            acc = 0.0
            for k in range(K):
                acc += float(x[t, k]) * float(w[n, k])
            y[t, n] = acc
    return y


def max_rel_err(y: np.ndarray, ref: np.ndarray) -> float:
    """north_star "max relative error 5e-3", reading G1: max|y - ref| / max|ref| over the whole output."""
    d = float(np.max(np.abs(np.asarray(y, dtype=np.float64) - ref)))
    m = float(np.max(np.abs(ref)))
    return d / m if m > 0 else d
