"""Device-resident Elastic-TP model state for a ``workloads.Config``: every simulated TP rank is its own HBM allocation
(one parameter arena + one paged-KV pool per rank), filled from the seeded position-addressable generators of
``workloads.gen``, plus the reload sources (pinned-host or device-resident images of the failed rank's bytes).

This is allocation + argument marshalling for ``bench.py``, ``__graft_entry__.smoke()`` and the full-size GPU tests.
Every step of the path (partition, CMM plan, lowering, copies, page-table rewrite) runs inside libetp.so; slab sizes come
from ``etp_plan_slab_span`` ("a single pass pre-allocates all destination buffers").  Nothing here imports
``oracle/`` and nothing here falls back to the CPU.
"""
from __future__ import annotations

import math
from dataclasses import dataclass
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np
import torch

from workloads import SEED0, Config, TensorSpec, fill_bytes, fill_normal16, tensor_inventory
from workloads.configs import class_units
from workloads.gen import fill_kv_pool, make_page_table, torch_dtype

from . import binding as B

ALIGN = 256


def _round_up(n: int, a: int = ALIGN) -> int:
    return (n + a - 1) // a * a


class Arena:
    """One contiguous uint8 allocation carved into 256-B aligned views (one per simulated rank / per image)."""

    def __init__(self, n_bytes: int, device, pinned: bool = False, zero: bool = True):
        n = max(int(n_bytes), ALIGN)
        if pinned:
            self.t = torch.empty(n, dtype=torch.uint8, pin_memory=True)
        elif zero:
            self.t = torch.zeros(n, dtype=torch.uint8, device=device)
        else:
            self.t = torch.empty(n, dtype=torch.uint8, device=device)
        assert self.t.data_ptr() % ALIGN == 0
        self.off = 0

    @classmethod
    def wrap(cls, t: torch.Tensor) -> "Arena":
        """An arena over memory somebody else allocated (a CUDA-IPC mapping of a peer process' arena)."""
        a = cls.__new__(cls)
        a.t, a.off = t, 0
        return a

    def take(self, n_bytes: int) -> torch.Tensor:
        a = self.off
        self.off = a + _round_up(n_bytes)
        assert self.off <= self.t.numel(), "arena overflow"
        return self.t[a:a + n_bytes]


@dataclass
class StepPlan:
    dead: int
    old: Dict[str, List[B.Shard]]      # per class, alive mask applied
    new: Dict[str, List[B.Shard]]
    bounds: Dict[str, List[int]]
    plans: Dict[str, B.Plan]


class ModelState:
    """Slabs, pools, images and page table of one config.  ``image`` in {"pinned", "device", "both"}."""

    def __init__(self, cfg: Config, device="cuda:0", image: str = "both", with_kv: bool = True,
                 with_params: bool = True, slack_garbage: bool = False, seq_lens: Optional[Sequence[int]] = None,
                 plan_mode: int = B.PLAN_CMM, cap_mode: str = "span", kv_layout: int = B.KV_TOKEN_MAJOR,
                 shard: Optional[Tuple[int, int]] = None, exchange=None):
        self.cfg, self.device = cfg, torch.device(device)
        self.cap_mode = cap_mode          # "span": union span of the rank's intervals (one hazard phase, L5);
                                          # "tight": the widest shard the rank ever holds (shards wrap, plans need phases)
        self.plan_mode = plan_mode        # B.PLAN_CMM (the paper's planner) | PLAN_GREEDY | PLAN_FULL_RELOAD
        self.kv_layout = kv_layout        # B.KV_TOKEN_MAJOR (reading K1) | B.KV_HEAD_MAJOR (its optional second layout)
        # One process per GPU: shard = (this process, number of processes); simulated rank r lives in the
        # memory of process r mod n.  This process allocates and fills only ITS ranks; the others' arenas / pools are opened as
        # CUDA-IPC mappings (`exchange`: an all-gather of picklable handles, e.g. torch.distributed.all_gather_object).
        self.shard, self.exchange = shard, exchange
        self.seed = SEED0 + 1000 * cfg.index
        self.image_kinds = ("pinned", "device") if image == "both" else (image,)
        self.specs: List[TensorSpec] = tensor_inventory(cfg) if with_params else []
        self.klasses = sorted(class_units(cfg))
        self.class_index = {k: i for i, k in enumerate(self.klasses)}
        self.n_ranks = cfg.scenario.n_old
        self.dt = torch_dtype(cfg.model.dtype)
        self.steps = self.plan_steps()
        self._geometry()
        if with_params:
            self._alloc_params(slack_garbage)
        self.kv = None
        if with_kv:
            self._alloc_kv(slack_garbage, seq_lens)
        self._prepared: Dict[Tuple[int, str], object] = {}

    def is_local(self, rank: int) -> bool:
        return self.shard is None or rank % self.shard[1] == self.shard[0]

    def rank_devices(self) -> List[int]:
        """etp_ctx_set_rank_devices map of this process: its own ranks on logical device 0, everybody else's -1."""
        return [0 if self.is_local(r) else -1 for r in range(self.n_ranks)]

    def _open_remote(self, local: Dict[int, torch.Tensor]) -> Dict[int, torch.Tensor]:
        """rank -> uint8 tensor for EVERY rank: the local ones as they are, the others through CUDA IPC."""
        if self.shard is None:
            return dict(local)
        mine = {r: t.untyped_storage()._share_cuda_() + (t.storage_offset(), t.numel()) for r, t in local.items()}
        out = dict(local)
        for handles in self.exchange(mine):
            for r, h in handles.items():
                if r in out:
                    continue
                st = torch.UntypedStorage._new_shared_cuda(*h[:-2])
                out[r] = torch.empty(0, dtype=torch.uint8, device=st.device).set_(st, h[-2], (h[-1],))
        return out

    # ------------------------------------------------------------------ S1 + S2 through the C ABI
    def initial_layouts(self) -> Dict[str, List[B.Shard]]:
        sc = self.cfg.scenario
        cur = {}
        for klass, H in class_units(self.cfg).items():
            if klass in sc.old_widths:
                b = [0]
                for w in sc.old_widths[klass]:
                    b.append(b[-1] + int(w))
            else:
                b = B.etp_partition(H, sc.n_old, sc.old_policy, granularity=klass)
            cur[klass] = [(r, b[r], b[r + 1], 1) for r in range(sc.n_old)]
        return cur

    def plan_step(self, cur: Dict[str, List[B.Shard]], dead: int) -> StepPlan:
        sc = self.cfg.scenario
        st = StepPlan(dead, {}, {}, {}, {})
        for klass, H in class_units(self.cfg).items():
            old = [(r, s, e, 0 if r == dead else 1) for (r, s, e, _) in cur[klass]]
            M = len(old) - 1
            tb = B.etp_partition(H, M, sc.new_policy, granularity=klass)
            # migration-aware (reading M1): the planner also places the wide shards, so no bounds are imposed
            plan = B.etp_plan_create(self.plan_mode, old, M, None if self.plan_mode == B.PLAN_MIGRATION_AWARE else tb)
            st.new[klass] = plan.new_layout()
            if self.plan_mode == B.PLAN_MIGRATION_AWARE:
                tb = [b for (_, b, _, _) in st.new[klass]] + [st.new[klass][-1][2]]
            st.old[klass], st.bounds[klass], st.plans[klass] = old, tb, plan
        return st

    def plan_steps(self) -> List[StepPlan]:
        cur = self.initial_layouts()
        out = []
        for dead in self.cfg.scenario.failed:
            st = self.plan_step(cur, dead)
            out.append(st)
            cur = st.new
        return out

    # ------------------------------------------------------------------ pre-allocation pass
    def _geometry(self) -> None:
        """rank -> (anchor, cap) per class: anchor = the rank's first unit at allocation, cap = union span over the
        scenario (single hazard phase, L5).  reload_range per class = units any RELOAD task reads."""
        self.geom: Dict[str, Dict[int, Tuple[int, int]]] = {}
        self.reload_range: Dict[str, Tuple[int, int]] = {}
        first = self.initial_layouts()
        for klass in self.klasses:
            g = {}
            for (r, s, e, _) in first[klass]:
                lo, hi = s, e
                for st in self.steps:
                    if any(rr == r for (rr, _, _, _) in st.old[klass]):
                        a, n = st.plans[klass].slab_span(r)
                        if n > 0:
                            lo, hi = min(lo, a), max(hi, a + n)
                if self.cap_mode == "tight":
                    widest = max([e - s] + [e2 - s2 for st in self.steps for (rr, s2, e2, _) in st.new[klass] if rr == r])
                    g[r] = (s, max(widest, 1))
                else:
                    g[r] = (s, max(hi - lo, 1))
            self.geom[klass] = g
            rl = [(b, e) for st in self.steps for (k, _, _, b, e) in st.plans[klass].tasks() if k == B.RELOAD]
            self.reload_range[klass] = (min(b for b, _ in rl), max(e for _, e in rl)) if rl else (0, 0)

    def _alloc_params(self, slack_garbage: bool) -> None:
        first = self.initial_layouts()
        need = {r: 0 for r in range(self.n_ranks)}
        img_bytes = 0
        for sp in self.specs:
            for r, (_, cap) in self.geom[sp.klass].items():
                need[r] += _round_up(cap * sp.unit_bytes)
            lo, hi = self.reload_range[sp.klass]
            img_bytes += _round_up((hi - lo) * sp.unit_bytes)
        local = {r: Arena(need[r], self.device) for r in range(self.n_ranks) if self.is_local(r)}
        opened = self._open_remote({r: a.t for r, a in local.items()})
        self.rank_arena = {r: local[r] if r in local else Arena.wrap(opened[r]) for r in range(self.n_ranks)}
        self.image_arena = {k: Arena(img_bytes, self.device, pinned=(k == "pinned"), zero=False) for k in self.image_kinds}
        self.slabs: Dict[str, Dict[int, torch.Tensor]] = {}
        self.images: Dict[str, Dict[str, torch.Tensor]] = {k: {} for k in self.image_kinds}
        eb = self.cfg.model.elem_bytes
        for sp in self.specs:
            epu = sp.unit_bytes // eb
            self.slabs[sp.name] = {}
            for (r, s, e, _) in first[sp.klass]:
                _, cap = self.geom[sp.klass][r]
                slab = self.rank_arena[r].take(cap * sp.unit_bytes)
                self.slabs[sp.name][r] = slab
                if not self.is_local(r):
                    continue                   # its owner fills it
                if slack_garbage:
                    nb8 = (slab.numel() + 7) // 8 * 8
                    slab.copy_(fill_bytes(self.seed, 10_000 + sp.stream * 16 + r, 0, nb8, device=self.device)[: slab.numel()])
                if e > s:   # anchor = s, so the old shard sits at slots [0, e - s)
                    fill_normal16(self.seed, sp.stream, s * epu, (e - s) * epu, self.cfg.model.init_std, self.dt,
                                  out=slab[: (e - s) * sp.unit_bytes].view(self.dt))
            lo, hi = self.reload_range[sp.klass]
            dev_img = None
            for k in self.image_kinds:
                img = self.image_arena[k].take((hi - lo) * sp.unit_bytes)
                if hi > lo:
                    if k == "device":
                        fill_normal16(self.seed, sp.stream, lo * epu, (hi - lo) * epu, self.cfg.model.init_std, self.dt,
                                      out=img.view(self.dt))
                        dev_img = img
                    elif dev_img is not None:
                        img.copy_(dev_img)
                    else:
                        tmp = fill_normal16(self.seed, sp.stream, lo * epu, (hi - lo) * epu, self.cfg.model.init_std, self.dt,
                                            device=self.device)
                        img.copy_(tmp.view(torch.uint8))
                        del tmp
                self.images[k][sp.name] = img
        torch.cuda.synchronize(self.device)

    def _alloc_kv(self, slack_garbage: bool, seq_lens) -> None:
        m, kvs = self.cfg.model, self.cfg.kv
        seed = self.seed + 500
        if seq_lens is None:
            seq_lens = [kvs.seq_len] * kvs.n_seqs
        table, seq_lens, last_use, n_blocks = make_page_table(kvs.n_seqs, seq_lens, kvs.block_size, kvs.pool_slack, seed)
        first = self.initial_layouts()["head"]
        widths = [e - s for (_, s, e, _) in first] + [e - s for st in self.steps for (_, s, e, _) in st.new["head"]]
        head_cap = max(widths)
        frag = m.head_dim * m.elem_bytes
        rows = m.n_layers * 2 * n_blocks * kvs.block_size
        kv = {"table": table, "seq_lens": seq_lens, "last_use": last_use, "n_blocks": n_blocks, "head_cap": head_cap,
              "frag": frag, "rows": rows, "anchors": {r: s for (r, s, e, _) in first}, "pools": {}, "backup": {},
              "layout": self.kv_layout}
        lay = dict(layout=self.kv_layout, block_size=kvs.block_size)
        for (r, s, e, _) in first:
            if not self.is_local(r):
                continue
            nb = rows * head_cap * frag
            if slack_garbage:
                pool = fill_bytes(seed, 100 + r, 0, (nb + 7) // 8 * 8, device=self.device)[:nb]
            else:
                pool = torch.zeros(nb, dtype=torch.uint8, device=self.device)
            if e > s:
                fill_kv_pool(pool, rows, head_cap, m.head_dim, 0, s, e - s, m.n_kv_heads, seed, 1, self.dt, **lay)
            kv["pools"][r] = pool
        torch.cuda.synchronize(self.device)
        kv["pools"] = self._open_remote(kv["pools"])
        # the backup of each rank that dies: its pool at the time of death compacted to its own heads (reading K4)
        for i, st in enumerate(self.steps):
            ds, de = [(s, e) for (r, s, e, _) in st.old["head"] if r == st.dead][0]
            hh = de - ds
            per_kind = {}
            if hh > 0:
                dev = torch.empty(rows * hh * frag, dtype=torch.uint8, device=self.device)
                fill_kv_pool(dev, rows, hh, m.head_dim, 0, ds, hh, m.n_kv_heads, seed, 1, self.dt, **lay)
                for k in self.image_kinds:
                    if k == "device":
                        per_kind[k] = dev
                    else:
                        pin = torch.empty(dev.numel(), dtype=torch.uint8, pin_memory=True)
                        pin.copy_(dev)
                        per_kind[k] = pin
                if "device" not in self.image_kinds:
                    del dev
            kv["backup"][i] = (per_kind, hh, ds)
        torch.cuda.synchronize(self.device)
        self.kv = kv

    # ------------------------------------------------------------------ marshalling
    def tensor_descs(self, step_idx: int, image: str) -> List[B.TensorDesc]:
        st = self.steps[step_idx]
        out = []
        for sp in self.specs:
            slabs = {}
            for r, t in self.slabs[sp.name].items():
                if r == st.dead or not any(rr == r for (rr, _, _, _) in st.old[sp.klass]):
                    continue
                anchor, cap = self.geom[sp.klass][r]
                slabs[r] = (t.data_ptr(), cap, anchor)
            lo, hi = self.reload_range[sp.klass]
            out.append(B.TensorDesc(sp.total_units, sp.unit_bytes, slabs, self.n_ranks, self.class_index[sp.klass],
                                    self.images[image][sp.name].data_ptr() if hi > lo else 0, lo, hi - lo))
        return out

    def prepared(self, step_idx: int, image: str):
        key = (step_idx, image)
        if key not in self._prepared:
            self._prepared[key] = B.PreparedParams(self.tensor_descs(step_idx, image))
        return self._prepared[key]

    # ------------------------------------------------------------------ one pass of the hot path (S1-S6)
    def reshard(self, ctx: B.Context, step_idx: int, image: str, copy_stream: int, reload_stream: int,
                replan: bool = True, table: Optional[np.ndarray] = None, block_budget: Optional[int] = None,
                kv_reload_stream: Optional[int] = None) -> Dict[str, object]:
        """S1 partition + S2 CMM plan (host, inside libetp.so), then S3-S5 on the parameters and S3-S6 on the KV cache.
        Asynchronous: returns after enqueueing; the caller synchronises both streams (and ``kv_reload_stream`` when the KV reload is
        given a stream of its own, so that its zero-copy gather shares the host link with the parameter DMAs instead of queueing
        behind them)."""
        st = self.steps[step_idx]
        if replan:
            cur = {k: [(r, s, e, 1) for (r, s, e, _) in st.old[k]] for k in st.old}
            st2 = self.plan_step(cur, st.dead)
            plans = st2.plans
        else:
            plans = st.plans
        rep_p = rep_k = None
        evicted: List[int] = []
        if self.specs:
            rep_p = self.prepared(step_idx, image).run(ctx, [plans[k] for k in self.klasses], copy_stream, reload_stream)
        new_table = None
        if self.kv is not None:
            kv, m = self.kv, self.cfg.model
            per_kind, hh, ds = kv["backup"][step_idx]
            new_table = kv["table"].copy() if table is None else table
            alive_pools = {r: p.data_ptr() for r, p in kv["pools"].items()
                           if r != st.dead and any(rr == r for (rr, _, _, _) in st.old["head"])}
            evicted, rep_k = B.etp_reshard_kv(
                ctx, n_layers=m.n_layers, n_blocks=kv["n_blocks"], block_size=self.cfg.kv.block_size, head_cap=kv["head_cap"],
                head_dim=m.head_dim, elem_bytes=m.elem_bytes, layout=kv["layout"], pools=alive_pools,
                head_anchor=kv["anchors"], n_ranks=self.n_ranks, table=new_table, seq_lens=kv["seq_lens"],
                last_use=kv["last_use"], head_plan=plans["head"],
                new_block_budget=kv["n_blocks"] if block_budget is None else block_budget,
                host_backup=per_kind[image].data_ptr() if hh > 0 else 0, host_heads=hh, host_head0=ds,
                copy_stream=copy_stream, reload_stream=reload_stream if kv_reload_stream is None else kv_reload_stream)
        return {"params": rep_p, "kv": rep_k, "evicted": evicted, "table": new_table, "plans": plans}

    # ------------------------------------------------------------------ S7: the layer outputs on the sharded state
    def linear(self, name: str, step_idx: int, after: bool = True) -> "B.PreparedLinear":
        """etp_shard_linear arguments for tensor ``name`` as it sits in the slabs before (``after=False``: every old rank
        still holds its shard) or after the reshard of step ``step_idx``."""
        key = (name, step_idx, after)
        if key not in self._prepared:
            sp = next(s for s in self.specs if s.name == name)
            st = self.steps[step_idx]
            layout = list(st.new[sp.klass]) if after else [(r, s, e, 1) for (r, s, e, _) in st.old[sp.klass]]
            slabs = {}
            for (r, _, _, _) in layout:
                anchor, cap = self.geom[sp.klass][r]
                slabs[r] = (self.slabs[name][r].data_ptr(), cap, anchor)
            sharded = sp.total_units * sp.features_per_unit
            K, N = (sharded, sp.row_elems) if sp.transposed else (sp.row_elems, sharded)
            desc = B.TensorDesc(sp.total_units, sp.unit_bytes, slabs, self.n_ranks, 0)
            self._prepared[key] = B.PreparedLinear(B.ROW_PARALLEL if sp.transposed else B.COL_PARALLEL, self.cfg.model.dtype,
                                                   K, N, desc, layout, sp.features_per_unit)
        return self._prepared[key]

    def state_bytes(self) -> Dict[str, int]:
        p = sum(sp.total_units * sp.unit_bytes for sp in self.specs)
        k = 0
        if self.kv is not None:
            live = int(((self.kv["seq_lens"].astype(np.int64) + self.cfg.kv.block_size - 1) // self.cfg.kv.block_size).sum())
            k = live * self.cfg.kv.block_size * self.cfg.model.n_layers * 2 * self.cfg.model.n_kv_heads * self.kv["frag"]
        return {"param_bytes": p, "kv_live_bytes": k}
