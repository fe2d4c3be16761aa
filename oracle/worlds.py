"""ORACLE (test infrastructure) — builds the seeded synthetic state of a config ("world") as host arrays.
Used by the tests (through ``tests/harness.py``) and by ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs.

This module itself does no method arithmetic: partition / plan come from the ``side`` object it is given
(``OracleSide`` here; the GPU tests pass a side that calls the C-ABI), and slot placement of the INITIAL
state is done by the oracle's ``place_units`` (test infrastructure producing inputs; inputs never come
from the CUDA path).  Slab capacities follow DESIGN.md "Input recipe": ``span`` = union span of every
interval the rank holds over the scenario (single-phase), ``tight`` = widest shard (wrap + multi-phase).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Tuple

import numpy as np
import torch

from oracle import planning as OP
from oracle import state as OS
from workloads import SEED0, Config, TensorSpec, fill_bytes, fill_normal16, tensor_inventory
from workloads.configs import class_units
from workloads.gen import as_u8, make_page_table, torch_dtype

GUARD = 256  # guard-band bytes either side of every GPU buffer


def seed_for(cfg: Config) -> int:
    return SEED0 + 1000 * cfg.index


class OracleSide:
    name = "oracle"

    @staticmethod
    def partition(H, M, policy="floor", align=1):
        return OP.partition(H, M, policy, align)

    @staticmethod
    def plan(old_layout, M, target_bounds=None):
        return OP.cmm_plan(old_layout, M, target_bounds)


@dataclass
class Step:
    dead: int
    old: Dict[str, list]        # klass -> layout with alive mask applied
    tasks: Dict[str, list]
    new: Dict[str, list]


def plan_scenario(cfg: Config, side, new_policy: Optional[str] = None, failed=None) -> List[Step]:
    sc = cfg.scenario
    new_policy = new_policy or sc.new_policy
    failed = sc.failed if failed is None else failed
    cur = {}
    for klass, H in class_units(cfg).items():
        if klass in sc.old_widths:
            cur[klass] = OP.layout_from_widths(sc.old_widths[klass])
        else:
            cur[klass] = OP.layout_from_bounds(side.partition(H, sc.n_old, sc.old_policy))
    steps = []
    for dead in failed:
        st = Step(dead, {}, {}, {})
        for klass, H in class_units(cfg).items():
            old = [(r, s, e, 0 if r == dead else 1) for (r, s, e, _) in cur[klass]]
            M = len(old) - 1
            tb = side.partition(H, M, new_policy)
            tasks, new = side.plan(old, M, tb)
            st.old[klass], st.tasks[klass], st.new[klass] = old, tasks, new
            cur[klass] = new
        steps.append(st)
    return steps


def slab_geometry(steps: List[Step], klass: str, mode: str) -> Dict[int, Tuple[int, int]]:
    """rank -> (anchor, cap).  anchor = the rank's first unit at allocation (reading L3)."""
    first = {r: (s, e) for (r, s, e, _) in steps[0].old[klass]}
    held: Dict[int, List[Tuple[int, int]]] = {r: [iv] for r, iv in first.items()}
    for st in steps:
        for (r, s, e, _) in st.new[klass]:
            held[r].append((s, e))
    geom = {}
    for r, ivs in held.items():
        anchor = first[r][0]
        if mode == "span":
            cap = max(e for (_, e) in ivs) - min(s for (s, _) in ivs)
        elif mode == "tight":
            cap = max(e - s for (s, e) in ivs)
        elif mode == "full":      # the paper's "unified address view": cap = H, anchor = 0
            cap, anchor = max(e for (_, _, e, _) in steps[0].old[klass]), 0
        else:
            raise ValueError(mode)
        geom[r] = (anchor, max(cap, 1))
    return geom


@dataclass
class ParamWorld:
    cfg: Config
    specs: List[TensorSpec]
    steps: List[Step]
    geom: Dict[str, Dict[int, Tuple[int, int]]]          # tensor name -> rank -> (anchor, cap)
    unsharded: Dict[str, np.ndarray]                     # tensor name -> uint8 [H*unit_bytes]
    slabs: Dict[str, Dict[int, np.ndarray]]              # tensor name -> rank -> uint8 [cap*unit_bytes]


def build_param_world(cfg: Config, side=OracleSide, mode="span", new_policy=None, failed=None, device="cpu") -> ParamWorld:
    """Unsharded tensors ~N(0, std) in the config dtype, slabs pre-filled with seeded garbage, then the old shard
    placed unit by unit.  ``device`` only says where the seeded generator runs (same bytes on CPU and CUDA)."""
    seed = seed_for(cfg)
    specs = tensor_inventory(cfg)
    steps = plan_scenario(cfg, side, new_policy, failed)
    dt = torch_dtype(cfg.model.dtype)
    geom, unsharded, slabs = {}, {}, {}
    for sp in specs:
        g = slab_geometry(steps, sp.klass, mode)
        geom[sp.name] = g
        n_el = sp.total_units * sp.unit_bytes // cfg.model.elem_bytes
        w = as_u8(fill_normal16(seed, sp.stream, 0, n_el, cfg.model.init_std, dt, device=device)).copy()
        unsharded[sp.name] = w
        slabs[sp.name] = {}
        for (r, s, e, _) in steps[0].old[sp.klass]:
            anchor, cap = g[r]
            nb = cap * sp.unit_bytes
            nb8 = (nb + 7) // 8 * 8
            slab = as_u8(fill_bytes(seed, 10_000 + sp.stream * 16 + r, 0, nb8, device=device))[:nb].copy()
            OS.place_units(slab, anchor, cap, sp.unit_bytes, s, e, w)
            slabs[sp.name][r] = slab
    return ParamWorld(cfg, specs, steps, geom, unsharded, slabs)


def oracle_reshard_params(world: ParamWorld, step_idx: int, slabs=None):
    """Apply step ``step_idx``'s plans to every tensor with the oracle.  Returns (out slabs, byte stats)."""
    st = world.steps[step_idx]
    slabs = world.slabs if slabs is None else slabs
    out, tot = {}, {"d2d_bytes": 0, "h2d_bytes": 0, "kept_bytes": 0}
    for sp in world.specs:
        snap = {r: a for r, a in slabs[sp.name].items() if r != st.dead}
        o, s = OS.apply_params(st.tasks[sp.klass], snap, world.geom[sp.name], sp.unit_bytes,
                               world.unsharded[sp.name], 0)
        out[sp.name] = o
        for k in tot:
            tot[k] += s[k]
    return out, tot


# ------------------------------------------------------------------------------------------ KV
@dataclass
class KVWorld:
    cfg: Config
    g: OS.KVGeom
    steps: List[Step]
    anchors: Dict[int, int]
    table: np.ndarray
    seq_lens: np.ndarray
    last_use: np.ndarray
    kv_ref: np.ndarray            # uint8 [seq][token][layer][2][head][frag]   (the plain definition's reference)
    pools: Dict[int, np.ndarray]  # rank -> uint8 pool image
    host_backup: Optional[np.ndarray]
    host_head0: int
    host_heads: int


def build_kv_world(cfg: Config, side=OracleSide, head_cap: Optional[int] = None, layout: int = 0,
                   new_policy=None, failed=None, seq_lens=None, device="cpu") -> KVWorld:
    """KV_ref values ~N(0,1); every rank's pool is seeded garbage with the rank's old heads of every live block
    written in (through numpy N-d indexing, not the oracle's offset arithmetic).  ``device`` only says where the
    seeded generator runs."""
    seed = seed_for(cfg) + 500
    m, kv = cfg.model, cfg.kv
    steps = plan_scenario(cfg, side, new_policy, failed)
    if seq_lens is None:
        seq_lens = [kv.seq_len] * kv.n_seqs
    table, seq_lens, last_use, n_blocks = make_page_table(kv.n_seqs, seq_lens, kv.block_size, kv.pool_slack, seed)
    widths = [e - s for st in steps for (_, s, e, _) in st.new["head"]] + [e - s for (_, s, e, _) in steps[0].old["head"]]
    head_cap = head_cap or max(widths)
    g = OS.KVGeom(m.n_layers, n_blocks, kv.block_size, head_cap, m.head_dim, m.elem_bytes, layout)
    dt = torch_dtype(m.dtype)
    max_len = int(max(seq_lens)) if len(seq_lens) else 0
    n_ref = kv.n_seqs * max_len * m.n_layers * 2 * m.n_kv_heads * m.head_dim
    kv_ref = as_u8(fill_normal16(seed, 1, 0, n_ref, 1.0, dt, device=device)).copy().reshape(
        kv.n_seqs, max_len, m.n_layers, 2, m.n_kv_heads, g.frag_bytes)
    anchors = {r: s for (r, s, e, _) in steps[0].old["head"]}
    pools = {}

    def view(pool, heads):
        if layout == 0:
            return pool.reshape(m.n_layers, 2, n_blocks, kv.block_size, heads, g.frag_bytes)
        return pool.reshape(m.n_layers, 2, n_blocks, heads, kv.block_size, g.frag_bytes)

    def put(v, b, t, slot_, frags):          # frags: [layer][K|V][frag_bytes] of one (token, head)
        if layout == 0:
            v[:, :, b, t, slot_] = frags
        else:
            v[:, :, b, slot_, t] = frags

    dead0 = steps[0].dead
    for (r, s, e, _) in steps[0].old["head"]:
        nb = g.pool_bytes()
        pool = as_u8(fill_bytes(seed, 100 + r, 0, (nb + 7) // 8 * 8, device=device))[:nb].copy()
        v = view(pool, head_cap)
        for sq in range(kv.n_seqs):
            for t in range(int(seq_lens[sq])):
                b = int(table[sq, t // kv.block_size])
                for h in range(s, e):
                    put(v, b, t % kv.block_size, (h - anchors[r]) % head_cap, kv_ref[sq, t, :, :, h])
        pools[r] = pool
    # host backup = the first dead rank's pool, compacted to its own heads (reading K4)
    ds, de = [(s, e) for (r, s, e, _) in steps[0].old["head"] if r == dead0][0]
    hh = de - ds
    host = None
    if hh > 0:
        nb = g.pool_bytes(hh)
        host = as_u8(fill_bytes(seed, 99, 0, (nb + 7) // 8 * 8, device=device))[:nb].copy()
        hv = view(host, hh)
        dv = view(pools[dead0], head_cap)
        for h in range(ds, de):
            if layout == 0:
                hv[:, :, :, :, h - ds] = dv[:, :, :, :, (h - anchors[dead0]) % head_cap]
            else:
                hv[:, :, :, h - ds] = dv[:, :, :, (h - anchors[dead0]) % head_cap]
    return KVWorld(cfg, g, steps, anchors, table, seq_lens, last_use, kv_ref, pools, host, ds, hh)


def kv_view(world: KVWorld, pool: np.ndarray, heads: Optional[int] = None):
    g, h = world.g, (heads or world.g.head_cap)
    if g.layout == 0:
        return pool.reshape(g.n_layers, 2, g.n_blocks, g.block_size, h, g.frag_bytes)
    return pool.reshape(g.n_layers, 2, g.n_blocks, h, g.block_size, g.frag_bytes)


def kv_get(world: KVWorld, pool, l, c, b, t, slot_):
    v = kv_view(world, pool)
    return v[l, c, b, t, slot_] if world.g.layout == 0 else v[l, c, b, slot_, t]
