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


def moe_layer_grouped(ctx, dtype: str, x: torch.Tensor, logits: torch.Tensor, top_k: int, ffn: int, descs, layout):
    """Same layer through etp_moe_linear: the (token, expert) pairs are sorted by expert, then ONE grouped
    launch each for gate, up and down on the whole expert tensors.  descs = {"gate"|"up"|"down_t": TensorDesc of the expert
    tensor (one unit = one expert)}, layout = the expert class's shards.  Returns (y fp32, order, weights, per-expert rows)."""
    T, hidden = x.shape
    dt = x.dtype
    E = logits.shape[1]
    order, wts = route(logits, top_k)
    flat_e = order.reshape(-1)
    perm = torch.argsort(flat_e, stable=True)                     # grouped by expert, token order kept inside a group
    tok = (perm // top_k)
    counts = torch.bincount(flat_e, minlength=E).cpu().numpy()
    offs = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    R = int(offs[-1])
    xp = x[tok].contiguous()
    g = torch.full((R, ffn), float("nan"), dtype=dt, device=x.device)
    u = torch.full((R, ffn), float("nan"), dtype=dt, device=x.device)
    etp.etp_moe_linear(ctx, etp.COL_PARALLEL, dtype, xp.data_ptr(), offs, hidden, ffn, descs["gate"], layout, g.data_ptr())
    etp.etp_moe_linear(ctx, etp.COL_PARALLEL, dtype, xp.data_ptr(), offs, hidden, ffn, descs["up"], layout, u.data_ptr())
    h = (torch.nn.functional.silu(g.float()) * u.float()).to(dt).contiguous()
    yp = torch.full((R, hidden), float("nan"), dtype=dt, device=x.device)
    etp.etp_moe_linear(ctx, etp.ROW_PARALLEL, dtype, h.data_ptr(), offs, ffn, hidden, descs["down_t"], layout, yp.data_ptr())
    torch.cuda.synchronize()
    w_flat = wts.reshape(-1)[perm].float()
    y = torch.zeros(T, hidden, dtype=torch.float32, device=x.device)
    y.index_add_(0, tok, w_flat[:, None] * yp.float())
    return y, order.cpu().numpy(), wts.cpu().numpy(), counts, (g, u, yp, tok, flat_e[perm])
