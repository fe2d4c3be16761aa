"""Test-side MoE layer on the resharded expert slabs (SURVEY.md 8(c) reading G5): the router (softmax, top-k, renormalised
weights), the SwiGLU activation and the weighted combine are harness glue in torch; every matrix product is a per-expert call
to etp_shard_linear (C ABI) on the expert's bytes exactly where the reshard left them.  The expected output comes from
oracle/linear.py::moe_ref on the UNSHARDED expert matrices."""
from __future__ import annotations

import numpy as np
import torch

import paper_2511_11617_b200 as etp


def expert_view(slab_ptr: int, anchor: int, cap: int, unit_bytes: int, e: int, rows: int, row_bytes: int):
    """One expert (= one unit of the expert-granularity plan) as a single-rank tensor of `rows` one-row units."""
    assert rows * row_bytes == unit_bytes
    base = slab_ptr + ((e - anchor) % cap) * unit_bytes
    return etp.TensorDesc(rows, row_bytes, {0: (base, rows, 0)}, 1, 0), [(0, 0, rows, 1)]


def route(logits: torch.Tensor, top_k: int):
    """fp64 softmax, top-k with ties to the lower expert index (stable sort), weights renormalised to sum 1."""
    p = torch.softmax(logits.double(), dim=1)
    order = torch.argsort(-p, dim=1, stable=True)[:, :top_k]
    w = torch.gather(p, 1, order)
    return order, w / w.sum(dim=1, keepdim=True)


def moe_layer_per_expert(ctx, dtype: str, x: torch.Tensor, logits: torch.Tensor, top_k: int, ffn: int, locate):
    """x [T][hidden] (16-bit, device), logits [T][E].  locate(kind, e) -> (slab_ptr, anchor, cap, unit_bytes) of the slab that
    holds expert e of kind in {"gate", "up", "down_t"}.  Returns (y fp32 [T][hidden], order, weights, calls)."""
    T, hidden = x.shape
    dt = x.dtype
    order, wts = route(logits, top_k)
    y = torch.zeros(T, hidden, dtype=torch.float32, device=x.device)
    calls = 0
    for e in torch.unique(order).tolist():
        tok, j = (order == e).nonzero(as_tuple=True)
        ne = int(tok.numel())
        xe = x[tok].contiguous()
        outs = {}
        for kind in ("gate", "up"):
            desc, lay = expert_view(*locate(kind, e), e, ffn, hidden * 2)
            o = torch.full((ne, ffn), float("nan"), dtype=dt, device=x.device)
            etp.etp_shard_linear(ctx, etp.COL_PARALLEL, dtype, xe.data_ptr(), ne, hidden, ffn, desc, lay, 1, o.data_ptr())
            outs[kind] = o
        h = (torch.nn.functional.silu(outs["gate"].float()) * outs["up"].float()).to(dt).contiguous()
        desc, lay = expert_view(*locate("down_t", e), e, ffn, hidden * 2)
        ye = torch.full((ne, hidden), float("nan"), dtype=dt, device=x.device)
        etp.etp_shard_linear(ctx, etp.ROW_PARALLEL, dtype, h.data_ptr(), ne, ffn, hidden, desc, lay, 1, ye.data_ptr())
        calls += 3
        y.index_add_(0, tok, wts[tok, j].float()[:, None] * ye.float())
    torch.cuda.synchronize()
    return y, order.cpu().numpy(), wts.cpu().numpy(), calls


def check_against_oracle(y, order, wts, x_f64, logits_f64, gate, up, down_t, top_k, tol=5e-3):
    from oracle import linear as OL
    idx, w = OL.moe_route(logits_f64, top_k)
    assert np.array_equal(order, idx), "routing decision differs from the oracle's"
    np.testing.assert_allclose(wts, w, rtol=1e-9)
    ref = OL.moe_ref(x_f64, logits_f64, gate, up, down_t, top_k)
    got = y.double().cpu().numpy()
    assert np.isfinite(got).all()
    err = OL.max_rel_err(got, ref)
    assert err <= tol, f"MoE layer output: max relative error {err:.3e} > {tol}"
    return err
