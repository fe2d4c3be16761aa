"""ORACLE (test infrastructure) — applying a plan to parameter slabs and a paged KV cache.

Follows DESIGN.md "O-A": snapshot semantics, element by element (the loops are in etp_apply.c),
slot addressing per reading L3, KV layout per reading K1, page-table rule per reading K5
("least recently used (LRU) eviction").  numpy arrays of uint8 / int32 only.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

from .planning import KEEP, RELOAD, TRANSFER, Task

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libetp_oracle.so")
_SRC = os.path.join(_HERE, "etp_apply.c")
_lib_handle = None


_SO_OMP = os.path.join(_HERE, "libetp_oracle_omp.so")
_lib_omp_handle = None


def build(force: bool = False, omp: bool = False) -> str:
    """gcc -O2, no intrinsics.  (Building the checker is not using it.)  ``omp``: the same file with -fopenmp, for the
    all-cores leg of the CPU baseline."""
    so = _SO_OMP if omp else _SO
    if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-Wall", "-shared", "-fPIC"] + (["-fopenmp"] if omp else []) + ["-o", so, _SRC])
    return so


def _declare(L):
    i64, p, i32 = ctypes.c_int64, ctypes.c_void_p, ctypes.c_int
    L.oracle_slot.restype = i64
    L.oracle_slot.argtypes = [i64, i64, i64]
    L.oracle_apply_param_task.restype = i64
    L.oracle_apply_param_task.argtypes = [i32, i64, i64, i64, p, i64, i64, p, i64, i64, p, i64]
    L.oracle_apply_kv_task.restype = i64
    L.oracle_apply_kv_task.argtypes = [i32, i64, i64, i32, i64, i64, i64, i64, i64,
                                       p, i64, p, i64, p, i64, i64, p, p, i64]
    L.oracle_threads.restype = i32
    L.oracle_apply_param_jobs.restype = i64
    L.oracle_apply_param_jobs.argtypes = [p, i64]
    L.oracle_apply_kv_jobs.restype = i64
    L.oracle_apply_kv_jobs.argtypes = [p, i64]
    return L


def _lib():
    global _lib_handle
    if _lib_handle is None:
        _lib_handle = _declare(ctypes.CDLL(build()))
    return _lib_handle


def _lib_omp():
    global _lib_omp_handle
    if _lib_omp_handle is None:
        _lib_omp_handle = _declare(ctypes.CDLL(build(omp=True)))
    return _lib_omp_handle


def omp_threads() -> int:
    """Threads the all-cores leg runs on (omp_get_max_threads of the -fopenmp build)."""
    return int(_lib_omp().oracle_threads())


def _ptr(a: Optional[np.ndarray]):
    if a is None:
        return None
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.c_void_p)


# ----------------------------------------------------------------------------- slot addressing (L3)
def slot(u: int, anchor: int, cap: int) -> int:
    """Rank r stores unit u at slot (u - anchor) mod cap of its slab (reading L3)."""
    return (u - anchor) % cap      # Python's % is already non-negative for cap > 0


def place_units(slab: np.ndarray, anchor: int, cap: int, unit_bytes: int, begin: int, end: int,
                unsharded: np.ndarray, unit0: int = 0) -> None:
    """Build an initial state: write units [begin,end) of the unsharded tensor into the slab."""
    assert end - begin <= cap
    for u in range(begin, end):
        s = slot(u, anchor, cap)
        slab[s * unit_bytes:(s + 1) * unit_bytes] = unsharded[(u - unit0) * unit_bytes:(u - unit0 + 1) * unit_bytes]


def read_units(slab: np.ndarray, anchor: int, cap: int, unit_bytes: int, begin: int, end: int) -> np.ndarray:
    out = np.empty((end - begin) * unit_bytes, dtype=np.uint8)
    for k, u in enumerate(range(begin, end)):
        s = slot(u, anchor, cap)
        out[k * unit_bytes:(k + 1) * unit_bytes] = slab[s * unit_bytes:(s + 1) * unit_bytes]
    return out


# ----------------------------------------------------------------------------- parameters (O-A)
def apply_params(tasks: Sequence[Task], snap: Dict[int, np.ndarray], geom: Dict[int, Tuple[int, int]],
                 unit_bytes: int, host_image: Optional[np.ndarray], host_unit0: int = 0
                 ) -> Tuple[Dict[int, np.ndarray], Dict[str, int]]:
    """snap[rank] = uint8 slab image (pre-reshard), geom[rank] = (anchor, cap).
    Returns (out slabs — full copies with the plan applied, byte counters)."""
    L = _lib()
    out = {r: a.copy() for r, a in snap.items()}
    stats = {"d2d_bytes": 0, "h2d_bytes": 0, "kept_bytes": 0}
    for (kind, src, dst, b, e) in tasks:
        if kind == KEEP:
            stats["kept_bytes"] += (e - b) * unit_bytes
            continue
        da, dc = geom[dst]
        assert e - b <= dc
        if kind == TRANSFER:
            sa, sc = geom[src]
            n = L.oracle_apply_param_task(TRANSFER, b, e, unit_bytes, _ptr(snap[src]), sa, sc,
                                          _ptr(out[dst]), da, dc, None, 0)
            stats["d2d_bytes"] += n
        else:
            assert host_image is not None, "RELOAD task but no host image"
            assert host_unit0 <= b and (e - host_unit0) * unit_bytes <= host_image.size
            n = L.oracle_apply_param_task(RELOAD, b, e, unit_bytes, None, 0, 1,
                                          _ptr(out[dst]), da, dc, _ptr(host_image), host_unit0)
            stats["h2d_bytes"] += n
    return out, stats


# ----------------------------------------------------------------------------- page table (K5)
def page_table_rewrite(table: np.ndarray, seq_lens: Sequence[int], last_use: Sequence[int],
                       block_size: int, budget: int):
    """"if the calculated KV demand exceeds the memory budget, the system will gradually release
    cold KVs using a least recently used (LRU) eviction policy".  Reading K5:
      (i)  live = sum ceil(len/bs) over non-evicted sequences; while live > budget evict the sequence with the
           smallest last_use (tie -> smaller index); its row becomes -1;
      (ii) every surviving block whose id >= budget, in ascending (seq, logical index), moves to the smallest
           id < budget not used by any surviving block (ids of evicted sequences are free).
    Returns (new_table, evicted seq ids in eviction order, [(seq, logical, old_id, new_id)] for ALL surviving blocks)."""
    table = np.asarray(table, dtype=np.int32)
    n_seqs = table.shape[0]
    per = [-(-int(seq_lens[s]) // block_size) for s in range(n_seqs)]
    alive = [True] * n_seqs
    live = sum(per)
    evicted: List[int] = []
    while live > budget:
        cand = [s for s in range(n_seqs) if alive[s] and per[s] > 0]
        if not cand:
            break
        v = min(cand, key=lambda s: (int(last_use[s]), s))
        alive[v] = False
        evicted.append(v)
        live -= per[v]
    new = table.copy()
    for s in evicted:
        new[s, :] = -1
    used = set()
    for s in range(n_seqs):
        if alive[s]:
            for i in range(per[s]):
                assert table[s, i] >= 0
                used.add(int(table[s, i]))
    free = [b for b in range(budget) if b not in used]    # ascending
    fi = 0
    pairs = []
    for s in range(n_seqs):
        if not alive[s]:
            continue
        for i in range(per[s]):
            b = int(table[s, i])
            if b >= budget:
                nb = free[fi]
                fi += 1
                new[s, i] = nb
            else:
                nb = b
            pairs.append((s, i, b, nb))
    return new, evicted, pairs


# ----------------------------------------------------------------------------- KV (O-K)
class KVGeom:
    def __init__(self, n_layers, n_blocks, block_size, head_cap, head_dim, elem_bytes, layout=0):
        self.n_layers, self.n_blocks, self.block_size = n_layers, n_blocks, block_size
        self.head_cap, self.head_dim, self.elem_bytes, self.layout = head_cap, head_dim, elem_bytes, layout
        self.frag_bytes = head_dim * elem_bytes

    def pool_bytes(self, heads: Optional[int] = None) -> int:
        h = self.head_cap if heads is None else heads
        return self.n_layers * 2 * self.n_blocks * self.block_size * h * self.frag_bytes

    def frag_off(self, l, c, b, t, slot_, heads: Optional[int] = None) -> int:
        """[layer][K|V][block][token][slot][dim] (layout 0) or [layer][K|V][block][slot][token][dim] (layout 1)."""
        h = self.head_cap if heads is None else heads
        lcb = (l * 2 + c) * self.n_blocks + b
        if self.layout == 0:
            return ((lcb * self.block_size + t) * h + slot_) * self.frag_bytes
        return ((lcb * h + slot_) * self.block_size + t) * self.frag_bytes


def apply_kv(head_tasks: Sequence[Task], snap: Dict[int, np.ndarray], anchors: Dict[int, int], g: KVGeom,
             host_backup: Optional[np.ndarray], host_heads: int, host_head0: int,
             pairs: Sequence[Tuple[int, int, int, int]]):
    """Same three cases as parameters with (layer, K/V, block, token, head) in place of the unit.
    ``pairs`` = surviving live blocks (seq, logical, old id, new id) from page_table_rewrite."""
    L = _lib()
    out = {r: a.copy() for r, a in snap.items()}
    old_ids = np.ascontiguousarray([p[2] for p in pairs], dtype=np.int32)
    new_ids = np.ascontiguousarray([p[3] for p in pairs], dtype=np.int32)
    stats = {"d2d_bytes": 0, "h2d_bytes": 0, "kept_bytes": 0}
    per_head_live = len(pairs) * g.n_layers * 2 * g.block_size * g.frag_bytes
    for (kind, src, dst, b, e) in head_tasks:
        if kind == KEEP:
            n = L.oracle_apply_kv_task(KEEP, b, e, g.layout, g.n_layers, g.n_blocks, g.block_size, g.head_cap,
                                       g.frag_bytes, _ptr(snap[dst]), anchors[dst], _ptr(out[dst]), anchors[dst],
                                       None, 0, 0, _ptr(old_ids), _ptr(new_ids), len(pairs))
            stats["d2d_bytes"] += n                 # relocated blocks of kept heads are same-rank copies
            stats["kept_bytes"] += per_head_live * (e - b) - n
        elif kind == TRANSFER:
            n = L.oracle_apply_kv_task(TRANSFER, b, e, g.layout, g.n_layers, g.n_blocks, g.block_size, g.head_cap,
                                       g.frag_bytes, _ptr(snap[src]), anchors[src], _ptr(out[dst]), anchors[dst],
                                       None, 0, 0, _ptr(old_ids), _ptr(new_ids), len(pairs))
            stats["d2d_bytes"] += n
        else:
            if host_backup is None:
                continue          # reading K4: fragments left untouched, sequences reported evicted by the caller
            assert host_head0 <= b and e <= host_head0 + host_heads
            n = L.oracle_apply_kv_task(RELOAD, b, e, g.layout, g.n_layers, g.n_blocks, g.block_size, g.head_cap,
                                       g.frag_bytes, None, 0, _ptr(out[dst]), anchors[dst],
                                       _ptr(host_backup), host_heads, host_head0,
                                       _ptr(old_ids), _ptr(new_ids), len(pairs))
            stats["h2d_bytes"] += n
    return out, stats


def kv_fragment(pool: np.ndarray, g: KVGeom, anchor: int, l: int, c: int, block: int, t: int, head: int,
                heads: Optional[int] = None) -> np.ndarray:
    sl = slot(head, anchor, g.head_cap if heads is None else heads)
    o = g.frag_off(l, c, block, t, sl, heads)
    return pool[o:o + g.frag_bytes]


# ----------------------------------------------------------------------------- all-cores leg (SURVEY.md 8(d) "Oracle timing")
_PARAM_JOB = np.dtype([(n, np.int64) for n in ("kind", "begin", "end", "unit_bytes", "snap_src", "src_anchor", "src_cap",
                                                "out_dst", "dst_anchor", "dst_cap", "host_image", "host_unit0")])
_KV_JOB = np.dtype([(n, np.int64) for n in ("kind", "h_begin", "h_end", "layout", "n_layers", "n_blocks", "block_size", "head_cap",
                                             "frag_bytes", "snap_src", "src_anchor", "out_dst", "dst_anchor", "host_backup",
                                             "host_heads", "host_head0", "old_ids", "new_ids", "n_pairs")])


def _addr(a: Optional[np.ndarray]) -> int:
    if a is None:
        return 0
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data


def apply_params_parallel(items, job_bytes: int = 4 << 20):
    """The same plan application as ``apply_params`` for a LIST of tensors at once, with the element-by-element loops of
    etp_apply.c run from an OpenMP ``parallel for`` over jobs (one job = a task, cut into unit sub-ranges of about
    ``job_bytes`` so the loop balances).  items: [(tasks, snap, geom, unit_bytes, host_image, host_unit0)].
    Returns ([out slabs per item], byte counters)."""
    L = _lib_omp()
    outs, jobs = [], []
    stats = {"d2d_bytes": 0, "h2d_bytes": 0, "kept_bytes": 0}
    for (tasks, snap, geom, unit_bytes, host_image, host_unit0) in items:
        out = {r: a.copy() for r, a in snap.items()}
        outs.append(out)
        step = max(1, job_bytes // unit_bytes)
        for (kind, src, dst, b, e) in tasks:
            if kind == KEEP:
                stats["kept_bytes"] += (e - b) * unit_bytes
                continue
            da, dc = geom[dst]
            assert e - b <= dc
            if kind == TRANSFER:
                sa, sc = geom[src]
                row = (TRANSFER, 0, 0, unit_bytes, _addr(snap[src]), sa, sc, _addr(out[dst]), da, dc, 0, 0)
                stats["d2d_bytes"] += (e - b) * unit_bytes
            else:
                assert host_image is not None and host_unit0 <= b and (e - host_unit0) * unit_bytes <= host_image.size
                row = (RELOAD, 0, 0, unit_bytes, 0, 0, 1, _addr(out[dst]), da, dc, _addr(host_image), host_unit0)
                stats["h2d_bytes"] += (e - b) * unit_bytes
            for u in range(b, e, step):
                jobs.append(row[:1] + (u, min(e, u + step)) + row[3:])
    arr = np.array(jobs, dtype=_PARAM_JOB) if jobs else np.zeros(0, dtype=_PARAM_JOB)
    n = L.oracle_apply_param_jobs(arr.ctypes.data_as(ctypes.c_void_p), len(jobs))
    assert n == stats["d2d_bytes"] + stats["h2d_bytes"]
    return outs, stats


def apply_kv_parallel(head_tasks: Sequence[Task], snap: Dict[int, np.ndarray], anchors: Dict[int, int], g: KVGeom,
                      host_backup: Optional[np.ndarray], host_heads: int, host_head0: int,
                      pairs: Sequence[Tuple[int, int, int, int]], pairs_per_job: int = 64):
    """``apply_kv`` with the live blocks of every head task cut into jobs of ``pairs_per_job`` blocks, run from the
    OpenMP parallel for of etp_apply.c (distinct live blocks have distinct new ids, so jobs write disjoint bytes)."""
    L = _lib_omp()
    out = {r: a.copy() for r, a in snap.items()}
    old_ids = np.ascontiguousarray([p[2] for p in pairs], dtype=np.int32)
    new_ids = np.ascontiguousarray([p[3] for p in pairs], dtype=np.int32)
    stats = {"d2d_bytes": 0, "h2d_bytes": 0, "kept_bytes": 0}
    per_head_live = len(pairs) * g.n_layers * 2 * g.block_size * g.frag_bytes
    jobs, kinds = [], []
    for (kind, src, dst, b, e) in head_tasks:
        if kind == RELOAD and host_backup is None:
            continue
        if kind == RELOAD:
            assert host_head0 <= b and e <= host_head0 + host_heads
            s_ptr, s_anchor, hb = 0, 0, _addr(host_backup)
        else:
            s_ptr, s_anchor, hb = _addr(snap[dst if kind == KEEP else src]), anchors[dst if kind == KEEP else src], 0
        if kind == KEEP:
            stats["kept_bytes"] += per_head_live * (e - b)
        for p0 in range(0, len(pairs), pairs_per_job):
            n = min(pairs_per_job, len(pairs) - p0)
            jobs.append((kind, b, e, g.layout, g.n_layers, g.n_blocks, g.block_size, g.head_cap, g.frag_bytes, s_ptr, s_anchor,
                         _addr(out[dst]), anchors[dst], hb, host_heads, host_head0, old_ids.ctypes.data + 4 * p0,
                         new_ids.ctypes.data + 4 * p0, n))
            kinds.append(kind)
    # per-kind byte counters need per-kind totals: run the kinds one after the other (three parallel loops)
    for kind, key in ((KEEP, "d2d_bytes"), (TRANSFER, "d2d_bytes"), (RELOAD, "h2d_bytes")):
        sel = [j for j, k in zip(jobs, kinds) if k == kind]
        if not sel:
            continue
        arr = np.array(sel, dtype=_KV_JOB)
        n = L.oracle_apply_kv_jobs(arr.ctypes.data_as(ctypes.c_void_p), len(sel))
        stats[key] += n
        if kind == KEEP:
            stats["kept_bytes"] -= n
    return out, stats
