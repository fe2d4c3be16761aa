"""ORACLE (test infrastructure) — S7 reference: the UNSHARDED linear layer Y = X W^T in fp64.

PAPER.md:45, :92-94 — ETP shards "attention and linear layers" with unequal widths; a correct resharded
state must compute the same layer output as the unsharded weight.  This is the textbook definition
(no sharding, no blocking); numpy's matmul is the library routine, pinned against an explicit triple loop
in tests/test_oracle_state.py::test_linear_ref_is_the_textbook_definition (decode16 against torch in
::test_decode16_exact, the MoE layer in ::test_moe_route_hand_worked / ::test_moe_ref_special_cases).
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


# ---------------------------------------------------------------------------------------------- MoE layer (config 4)
# SURVEY.md 8(c) reading G5 / DESIGN.md G5; PAPER.md:172-174 (MoE experts are the unit of the expert-granularity plan).
# Router logits -> softmax over all experts -> top-k (tie -> lower expert index) -> weights renormalised to sum 1;
# y[t] = sum over the k chosen experts e of w[t,e] * down_e( silu(gate_e x[t]) * (up_e x[t]) ).  Plain loops, fp64.
def moe_route(logits: np.ndarray, top_k: int):
    """logits [T][E] -> (experts [T][top_k] int64 in descending probability, weights [T][top_k] fp64 summing to 1)."""
    logits = np.asarray(logits, dtype=np.float64)
    T, E = logits.shape
    idx = np.zeros((T, top_k), dtype=np.int64)
    wts = np.zeros((T, top_k), dtype=np.float64)
    for t in range(T):
        z = np.exp(logits[t] - logits[t].max())
        p = z / z.sum()
        order = sorted(range(E), key=lambda e: (-p[e], e))[:top_k]
        s = sum(p[e] for e in order)
        for j, e in enumerate(order):
            idx[t, j] = e
            wts[t, j] = p[e] / s
    return idx, wts


def silu(v: np.ndarray) -> np.ndarray:
    return v / (1.0 + np.exp(-v))


def swiglu_ref(x: np.ndarray, gate_e: np.ndarray, up_e: np.ndarray) -> np.ndarray:
    """The intermediate of one expert, row by row: h[r] = silu(gate_e x[r]) * (up_e x[r]) in fp64 (x [R][hidden]; gate_e, up_e
    [ffn][hidden]).  It is the inner term of moe_ref written for a block of rows; pins the fused gate|up kernel."""
    x = np.asarray(x, dtype=np.float64)
    out = np.zeros((x.shape[0], gate_e.shape[0]), dtype=np.float64)
    for r in range(x.shape[0]):
        out[r] = silu(np.asarray(gate_e, dtype=np.float64) @ x[r]) * (np.asarray(up_e, dtype=np.float64) @ x[r])
    return out


def moe_ref(x: np.ndarray, logits: np.ndarray, gate: np.ndarray, up: np.ndarray, down_t: np.ndarray, top_k: int) -> np.ndarray:
    """x [T][hidden]; gate, up [E][ffn][hidden]; down_t [E][ffn][hidden] (row-parallel weights are stored transposed,
    reading L1: down_e(h) = h @ down_t[e]); gate / up / down_t may be arrays or mappings expert -> matrix (only the routed
    experts are touched); returns y [T][hidden] in fp64."""
    x = np.asarray(x, dtype=np.float64)
    idx, wts = moe_route(logits, top_k)
    y = np.zeros((x.shape[0], x.shape[1]), dtype=np.float64)
    for t in range(x.shape[0]):
        for j in range(top_k):
            e = int(idx[t, j])
            h = silu(np.asarray(gate[e], dtype=np.float64) @ x[t]) * (np.asarray(up[e], dtype=np.float64) @ x[t])
            y[t] += wts[t, j] * (h @ np.asarray(down_t[e], dtype=np.float64))
    return y
