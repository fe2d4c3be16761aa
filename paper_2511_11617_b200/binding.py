"""Thin ctypes binding of libetp.so (include/etp.h).  Argument marshalling only — every step of the hot path runs
inside the library.  Names follow the C ABI.  There is no CPU fallback: if the library is missing or no sm_100 device
is present, the device calls raise EtpError."""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, List, Optional, Sequence, Tuple

from . import _build

i32, i64, vp = C.c_int32, C.c_int64, C.c_void_p

ETP_OK = 0
STATUS = {0: "OK", 1: "INVALID_ARG", 2: "ALIGNMENT", 3: "CAPACITY", 4: "NO_SOURCE", 5: "UNSUPPORTED", 6: "CUDA", 7: "NOMEM"}
KEEP, TRANSFER, RELOAD = 0, 1, 2
SPLIT = {"floor": 0, "ceil_first": 1}
GRAN = {"head": 0, "ffn": 1, "expert": 2, "vocab": 3}
PLAN_CMM, PLAN_GREEDY, PLAN_FULL_RELOAD, PLAN_MIGRATION_AWARE = 0, 1, 2, 3
COL_PARALLEL, ROW_PARALLEL = 0, 1
DTYPE = {"bf16": 0, "fp16": 1}
KV_TOKEN_MAJOR, KV_HEAD_MAJOR = 0, 1
(OPT_SKIP_D2D, OPT_SKIP_RELOAD, OPT_TMA_MIN_BYTES, OPT_LDG_STEALS_BULK, OPT_RELOAD_CHUNK_BYTES, OPT_RESERVED_5,
 OPT_GRID_CTAS, OPT_GATHER_CTAS, OPT_TIME_KERNELS, OPT_LINEAR_CTA_PAIR, OPT_VALIDATE_INTERVALS, OPT_LINEAR_PDL, OPT_LINEAR_RING, OPT_ONLY_PHASE,
 OPT_MOE_CTA_PAIR, OPT_SMALL_STAGED) = range(16)


class EtpError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"ETP_ERR_{STATUS.get(status, status)}: {msg}")
        self.status = status


class etp_shard(C.Structure):
    _fields_ = [("rank", i32), ("alive", i32), ("begin", i64), ("end", i64)]


class etp_task(C.Structure):
    _fields_ = [("kind", i32), ("src_rank", i32), ("dst_rank", i32), ("reserved", i32), ("begin", i64), ("end", i64)]


class etp_plan_stats(C.Structure):
    _fields_ = [(n, i64) for n in ("total_units", "keep_units", "transfer_units", "reload_units", "reload_lower_bound", "n_tasks")]


class etp_slab(C.Structure):
    _fields_ = [("base", vp), ("cap_units", i64), ("anchor_unit", i64)]


class etp_tensor(C.Structure):
    _fields_ = [("total_units", i64), ("unit_bytes", i64), ("slabs", C.POINTER(etp_slab)), ("n_ranks", i32), ("plan_index", i32),
                ("host_image", vp), ("host_unit0", i64), ("host_units", i64)]


class etp_reshard_report(C.Structure):
    _fields_ = [("d2d_bytes", i64), ("h2d_bytes", i64), ("reload_dev_bytes", i64), ("kept_bytes", i64), ("n_jobs", i64), ("n_units", i64),
                ("n_memcpys", i64), ("n_phases", i32), ("n_kernel_launches", i32), ("lower_ms", C.c_double), ("remote_bytes", i64)]

    def as_dict(self) -> Dict[str, float]:
        return {n: getattr(self, n) for n, _ in self._fields_}


class etp_kv_geometry(C.Structure):
    _fields_ = [("n_layers", i32), ("n_blocks", i32), ("block_size", i32), ("head_cap", i32), ("head_dim", i32), ("elem_bytes", i32),
                ("layout", i32), ("n_ranks", i32), ("pools", C.POINTER(vp)), ("head_anchor", C.POINTER(i64)),
                ("host_backup", vp), ("host_heads", i32), ("host_head0", i64)]


class etp_page_table(C.Structure):
    _fields_ = [("n_seqs", i32), ("max_blocks", i32), ("block_table", C.POINTER(i32)), ("seq_lens", C.POINTER(i32)),
                ("last_use", C.POINTER(i64))]


class etp_linear_out(C.Structure):
    _fields_ = [("w", C.POINTER(etp_tensor)), ("out_features", i64), ("features_per_unit", i64), ("y", vp)]


class etp_linear_spec(C.Structure):
    _fields_ = [("mode", i32), ("reserved0", i32), ("in_features", i64), ("out_features", i64), ("w", C.POINTER(etp_tensor)),
                ("layout", C.POINTER(etp_shard)), ("n_shards", i32), ("reserved1", i32), ("features_per_unit", i64)]


class etp_linear_plan_stats(C.Structure):
    _fields_ = [("n_linears", i32), ("n_ctas", i32), ("n_items", i64), ("total_chunks", i64), ("max_cta_chunks", i64),
                ("n_split_tiles", i64), ("n_splits", i32 * 8)]


class etp_moe_instance(C.Structure):
    _fields_ = [("expert", i32), ("rank", i32), ("slot", i64), ("row_begin", i64), ("row_end", i64)]


class etp_replica(C.Structure):
    _fields_ = [("expert", i32), ("rank", i32)]


class etp_interval(C.Structure):
    _fields_ = [("src", vp), ("dst", vp), ("bytes", i64)]


EXPORTS = ["etp_ctx_create", "etp_ctx_create_multi", "etp_ctx_set_rank_devices", "etp_ctx_device_report", "etp_ctx_destroy", "etp_last_error", "etp_version", "etp_ctx_set_option", "etp_ctx_get_option",
           "etp_ctx_kernel_time", "etp_partition", "etp_cmm_plan", "etp_plan_create", "etp_plan_create_weighted", "etp_plan_tasks", "etp_plan_new_layout",
           "etp_plan_get_stats", "etp_plan_slab_span", "etp_plan_free", "etp_reshard_params", "etp_page_table_rewrite", "etp_reshard_kv", "etp_shard_linear",
           "etp_shard_linear_multi", "etp_linear_prepare", "etp_linear_run", "etp_linear_plan_info", "etp_linear_free",
           "etp_moe_linear", "etp_moe_linear_instances", "etp_moe_gate_up", "etp_eplb_place", "etp_eplb_apply", "etp_copy_intervals", "etp_intervals_validate",
           "etp_copy_intervals_static", "etp_debug_starved_wait"]

_lib = None


def lib() -> C.CDLL:
    """Loads (building first if stale) libetp.so.  Fails loudly if it cannot be built or loaded."""
    global _lib
    if _lib is None:
        so = _build.build()
        L = C.CDLL(so)
        L.etp_last_error.restype = C.c_char_p
        L.etp_version.restype = C.c_char_p
        L.etp_ctx_create.argtypes = [C.c_int, i64, C.POINTER(vp)]
        L.etp_ctx_create_multi.argtypes = [C.POINTER(i32), i32, C.POINTER(vp)]
        L.etp_ctx_set_rank_devices.argtypes = [vp, C.POINTER(i32), i32]
        L.etp_ctx_device_report.argtypes = [vp, i32, C.POINTER(etp_reshard_report)]
        L.etp_ctx_destroy.argtypes = [vp]
        L.etp_ctx_destroy.restype = None
        L.etp_ctx_set_option.argtypes = [vp, C.c_int, i64]
        L.etp_ctx_get_option.argtypes = [vp, C.c_int, C.POINTER(i64)]
        L.etp_ctx_kernel_time.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(i32)]
        L.etp_plan_slab_span.argtypes = [vp, i32, C.POINTER(i64), C.POINTER(i64)]
        L.etp_partition.argtypes = [C.c_int, i64, i32, C.c_int, i64, C.POINTER(i64)]
        L.etp_cmm_plan.argtypes = [C.POINTER(etp_shard), i32, C.POINTER(i64), i32, C.POINTER(vp)]
        L.etp_plan_create.argtypes = [C.c_int, C.POINTER(etp_shard), i32, C.POINTER(i64), i32, C.POINTER(vp)]
        L.etp_plan_create_weighted.argtypes = [C.c_int, C.POINTER(etp_shard), i32, C.POINTER(i64), i32, C.POINTER(i64), i32, C.POINTER(vp)]
        L.etp_plan_tasks.argtypes = [vp, C.POINTER(etp_task), i64, C.POINTER(i64)]
        L.etp_plan_new_layout.argtypes = [vp, C.POINTER(etp_shard), i32, C.POINTER(i32)]
        L.etp_plan_get_stats.argtypes = [vp, C.POINTER(etp_plan_stats)]
        L.etp_plan_free.argtypes = [vp]
        L.etp_plan_free.restype = None
        L.etp_reshard_params.argtypes = [vp, C.POINTER(etp_tensor), i32, C.POINTER(vp), i32, vp, vp, C.POINTER(etp_reshard_report)]
        L.etp_page_table_rewrite.argtypes = [C.POINTER(etp_page_table), i32, i32, C.POINTER(i32), C.POINTER(i32), C.POINTER(i32), i64,
                                             C.POINTER(i64)]
        L.etp_reshard_kv.argtypes = [vp, C.POINTER(etp_kv_geometry), C.POINTER(etp_page_table), vp, i32, C.POINTER(i32), C.POINTER(i32),
                                     vp, vp, C.POINTER(etp_reshard_report)]
        L.etp_shard_linear.argtypes = [vp, C.c_int, C.c_int, vp, i64, i64, i64, C.POINTER(etp_tensor), C.POINTER(etp_shard), i32, i64,
                                       vp, vp]
        L.etp_shard_linear_multi.argtypes = [vp, C.c_int, vp, i64, i64, C.POINTER(etp_linear_out), i32, C.POINTER(etp_shard), i32, vp]
        L.etp_linear_prepare.argtypes = [vp, C.c_int, C.POINTER(etp_linear_spec), i32, C.POINTER(vp)]
        L.etp_linear_run.argtypes = [vp, C.POINTER(vp), i64, C.POINTER(vp), vp]
        L.etp_linear_plan_info.argtypes = [vp, C.POINTER(etp_linear_plan_stats)]
        L.etp_linear_free.argtypes = [vp]
        L.etp_linear_free.restype = None
        L.etp_moe_linear.argtypes = [vp, C.c_int, C.c_int, vp, C.POINTER(i64), i32, i64, i64, C.POINTER(etp_tensor), C.POINTER(etp_shard),
                                     i32, vp, vp]
        L.etp_moe_linear_instances.argtypes = [vp, C.c_int, C.c_int, vp, C.POINTER(etp_moe_instance), i32, i64, i32, i64, i64,
                                               C.POINTER(etp_tensor), vp, vp]
        L.etp_moe_gate_up.argtypes = [vp, C.c_int, vp, C.POINTER(i64), C.POINTER(etp_moe_instance), i32, i64, i32, i64, i64,
                                      C.POINTER(etp_tensor), C.POINTER(etp_tensor), C.POINTER(etp_shard), i32, vp, vp]
        L.etp_eplb_apply.argtypes = [vp, C.POINTER(etp_tensor), i32, C.POINTER(etp_shard), i32, C.POINTER(etp_replica), i32, C.POINTER(i64), vp]
        L.etp_eplb_place.argtypes = [C.POINTER(i64), C.POINTER(i32), i32, C.POINTER(i64), C.POINTER(i32), i32, C.POINTER(etp_replica), i32,
                                     C.POINTER(i32)]
        L.etp_copy_intervals.argtypes = [vp, C.POINTER(etp_interval), i64, vp, C.POINTER(etp_reshard_report)]
        L.etp_intervals_validate.argtypes = [C.POINTER(etp_interval), i64]
        L.etp_copy_intervals_static.argtypes = [C.POINTER(etp_interval), i64, vp]
        L.etp_debug_starved_wait.argtypes = [vp, vp]
        _lib = L
    return _lib


def _check(status: int) -> None:
    if status != ETP_OK:
        raise EtpError(status, lib().etp_last_error().decode())


def etp_version() -> str:
    return lib().etp_version().decode()


# ------------------------------------------------------------------------------------------------ S1 / S2 (host)
def etp_partition(total_units: int, parts: int, policy: str = "floor", align_units: int = 1, granularity: str = "ffn") -> List[int]:
    out = (i64 * (parts + 1 if parts >= 0 else 1))()
    _check(lib().etp_partition(GRAN[granularity], total_units, parts, SPLIT[policy], align_units, out))
    return list(out)


Shard = Tuple[int, int, int, int]  # (rank, begin, end, alive) — the tuple order used by the tests' harness


def _shards(layout: Sequence[Shard]):
    arr = (etp_shard * max(len(layout), 1))()
    for k, (r, b, e, a) in enumerate(layout):
        arr[k] = etp_shard(int(r), int(a), int(b), int(e))
    return arr


class Plan:
    """Owns an etp_plan handle."""

    def __init__(self, handle: int):
        self.handle = vp(handle)

    def __del__(self):
        if getattr(self, "handle", None) and _lib is not None:
            _lib.etp_plan_free(self.handle)
            self.handle = None

    def tasks(self) -> List[Tuple[int, int, int, int, int]]:
        n = i64()
        _check(lib().etp_plan_tasks(self.handle, None, 0, C.byref(n)))
        arr = (etp_task * max(n.value, 1))()
        _check(lib().etp_plan_tasks(self.handle, arr, n.value, C.byref(n)))
        return [(t.kind, t.src_rank, t.dst_rank, t.begin, t.end) for t in arr[: n.value]]

    def new_layout(self) -> List[Shard]:
        n = i32()
        _check(lib().etp_plan_new_layout(self.handle, None, 0, C.byref(n)))
        arr = (etp_shard * max(n.value, 1))()
        _check(lib().etp_plan_new_layout(self.handle, arr, n.value, C.byref(n)))
        return [(s.rank, s.begin, s.end, s.alive) for s in arr[: n.value]]

    def slab_span(self, rank: int) -> Tuple[int, int]:
        """(first_unit, span_units) of the union of the rank's old and new interval."""
        a, n = i64(), i64()
        _check(lib().etp_plan_slab_span(self.handle, rank, C.byref(a), C.byref(n)))
        return a.value, n.value

    def stats(self) -> Dict[str, int]:
        st = etp_plan_stats()
        _check(lib().etp_plan_get_stats(self.handle, C.byref(st)))
        return {n: getattr(st, n) for n, _ in st._fields_}


def etp_plan_create(mode: int, old_layout: Sequence[Shard], M: int, target_bounds: Optional[Sequence[int]] = None,
                    link_cost: Optional[Sequence[Sequence[int]]] = None) -> Plan:
    """link_cost: square matrix [src][dst] of per-unit link prices (etp_plan_create_weighted), migration-aware mode only."""
    h = vp()
    tb = None
    if target_bounds is not None:
        tb = (i64 * len(target_bounds))(*[int(x) for x in target_bounds])
    if link_cost is None:
        _check(lib().etp_plan_create(mode, _shards(old_layout), len(old_layout), tb, M, C.byref(h)))
    else:
        n = len(link_cost)
        flat = (i64 * (n * n))(*[int(v) for row in link_cost for v in row])
        _check(lib().etp_plan_create_weighted(mode, _shards(old_layout), len(old_layout), tb, M, flat, n, C.byref(h)))
    return Plan(h.value)


def etp_cmm_plan(old_layout: Sequence[Shard], M: int, target_bounds: Optional[Sequence[int]] = None) -> Plan:
    h = vp()
    tb = None
    if target_bounds is not None:
        tb = (i64 * len(target_bounds))(*[int(x) for x in target_bounds])
    _check(lib().etp_cmm_plan(_shards(old_layout), len(old_layout), tb, M, C.byref(h)))
    return Plan(h.value)


def etp_page_table_rewrite(table, seq_lens, last_use, block_size: int, budget: int):
    """table: numpy int32 [n_seqs][max_blocks] (modified in place).  Returns (evicted list, pairs [(old, new)])."""
    import numpy as np
    assert table.dtype == np.int32 and table.flags["C_CONTIGUOUS"]
    sl = np.ascontiguousarray(seq_lens, dtype=np.int32)
    lu = np.ascontiguousarray(last_use, dtype=np.int64)
    n_seqs, max_blocks = table.shape
    pt = etp_page_table(n_seqs, max_blocks, table.ctypes.data_as(C.POINTER(i32)), sl.ctypes.data_as(C.POINTER(i32)),
                        lu.ctypes.data_as(C.POINTER(i64)))
    cap = int(((sl.astype(np.int64) + block_size - 1) // block_size).sum()) if block_size > 0 else 0
    pairs = np.zeros((max(cap, 1), 2), dtype=np.int32)
    ev = np.zeros(max(n_seqs, 1), dtype=np.int32)
    n_ev, n_pairs = i32(), i64()
    _check(lib().etp_page_table_rewrite(C.byref(pt), block_size, budget, ev.ctypes.data_as(C.POINTER(i32)), C.byref(n_ev),
                                        pairs.ctypes.data_as(C.POINTER(i32)), cap, C.byref(n_pairs)))
    return [int(v) for v in ev[: n_ev.value]], [(int(a), int(b)) for a, b in pairs[: n_pairs.value]]


def etp_eplb_place(expert_load: Sequence[int], home_rank: Sequence[int], rank_capacity: Sequence[int],
                   spare_slots: Sequence[int]) -> List[Tuple[int, int]]:
    """EPLB-style replica placement (host-only): [(expert, rank)] of the new instances in creation order."""
    E, R = len(expert_load), len(rank_capacity)
    ld = (i64 * max(E, 1))(*[int(v) for v in expert_load])
    hm = (i32 * max(E, 1))(*[int(v) for v in home_rank])
    cp = (i64 * R)(*[int(v) for v in rank_capacity])
    sl = (i32 * R)(*[int(v) for v in spare_slots])
    n = i32()
    _check(lib().etp_eplb_place(ld, hm, E, cp, sl, R, None, 0, C.byref(n)))
    out = (etp_replica * max(n.value, 1))()
    _check(lib().etp_eplb_place(ld, hm, E, cp, sl, R, out, n.value, C.byref(n)))
    return [(r.expert, r.rank) for r in out[: n.value]]


# ------------------------------------------------------------------------------------------------ device calls
class Context:
    """Owns an etp_ctx (descriptor arenas, events) on one CUDA device."""

    def __init__(self, device: int = 0, staging_bytes: int = 0, devices: Optional[Sequence[int]] = None):
        """``devices``: CUDA device of every LOGICAL device (etp_ctx_create_multi; entries may repeat); default one device."""
        h = vp()
        if devices is None:
            _check(lib().etp_ctx_create(device, staging_bytes, C.byref(h)))
            self.n_devices = 1
        else:
            arr = (i32 * len(devices))(*[int(d) for d in devices])
            _check(lib().etp_ctx_create_multi(arr, len(devices), C.byref(h)))
            self.n_devices = len(devices)
        self.handle = h

    def set_rank_devices(self, device_of_rank: Sequence[int]) -> None:
        """rank -> logical device that holds (and writes) its memory; -1 = a rank another process writes."""
        arr = (i32 * max(len(device_of_rank), 1))(*[int(d) for d in device_of_rank])
        _check(lib().etp_ctx_set_rank_devices(self.handle, arr, len(device_of_rank)))

    def device_report(self, logical_device: int) -> Dict[str, float]:
        rep = etp_reshard_report()
        _check(lib().etp_ctx_device_report(self.handle, logical_device, C.byref(rep)))
        return rep.as_dict()

    def close(self):
        if getattr(self, "handle", None):
            lib().etp_ctx_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_option(self, key: int, value: int) -> None:
        _check(lib().etp_ctx_set_option(self.handle, key, value))

    def get_option(self, key: int) -> int:
        v = i64()
        _check(lib().etp_ctx_get_option(self.handle, key, C.byref(v)))
        return v.value

    def kernel_time(self) -> Tuple[float, int]:
        """(ms, launches) of the copy-stream kernels of the last device call (needs OPT_TIME_KERNELS = 1)."""
        ms, n = C.c_double(), i32()
        _check(lib().etp_ctx_kernel_time(self.handle, C.byref(ms), C.byref(n)))
        return ms.value, n.value


class TensorDesc:
    """Python-side description of one sharded tensor: slabs = {rank: (device ptr, cap_units, anchor_unit)}."""

    def __init__(self, total_units: int, unit_bytes: int, slabs: Dict[int, Tuple[int, int, int]], n_ranks: int, plan_index: int,
                 host_image: int = 0, host_unit0: int = 0, host_units: int = 0):
        self.total_units, self.unit_bytes, self.slabs, self.n_ranks = total_units, unit_bytes, slabs, n_ranks
        self.plan_index, self.host_image, self.host_unit0, self.host_units = plan_index, host_image, host_unit0, host_units


def _marshal_tensors(tensors: Sequence[TensorDesc]):
    arr = (etp_tensor * max(len(tensors), 1))()
    keep = []
    for k, t in enumerate(tensors):
        sl = (etp_slab * max(t.n_ranks, 1))()
        for r in range(t.n_ranks):
            base, cap, anchor = t.slabs.get(r, (0, 0, 0))
            sl[r] = etp_slab(base or None, cap, anchor)
        keep.append(sl)
        arr[k] = etp_tensor(t.total_units, t.unit_bytes, sl, t.n_ranks, t.plan_index, t.host_image or None, t.host_unit0, t.host_units)
    return arr, keep


def etp_reshard_params(ctx: Context, tensors: Sequence[TensorDesc], plans: Sequence[Plan], copy_stream: int = 0,
                       reload_stream: int = 0) -> Dict[str, float]:
    arr, keep = _marshal_tensors(tensors)
    ph = (vp * max(len(plans), 1))(*[p.handle for p in plans])
    rep = etp_reshard_report()
    _check(lib().etp_reshard_params(ctx.handle, arr, len(tensors), ph, len(plans), copy_stream or None, reload_stream or None, C.byref(rep)))
    del keep
    return rep.as_dict()


class PreparedParams:
    """Pre-marshalled tensor array of etp_reshard_params, so that a timed loop pays only the C call."""

    def __init__(self, tensors: Sequence[TensorDesc]):
        self.arr, self._keep = _marshal_tensors(tensors)
        self.n = len(tensors)

    def run(self, ctx: Context, plans: Sequence[Plan], copy_stream: int = 0, reload_stream: int = 0) -> Dict[str, float]:
        ph = (vp * max(len(plans), 1))(*[p.handle for p in plans])
        rep = etp_reshard_report()
        _check(lib().etp_reshard_params(ctx.handle, self.arr, self.n, ph, len(plans), copy_stream or None, reload_stream or None,
                                        C.byref(rep)))
        return rep.as_dict()


def etp_reshard_kv(ctx: Context, *, n_layers: int, n_blocks: int, block_size: int, head_cap: int, head_dim: int, elem_bytes: int,
                   layout: int, pools: Dict[int, int], head_anchor: Dict[int, int], n_ranks: int, table, seq_lens, last_use,
                   head_plan: Plan, new_block_budget: int, host_backup: int = 0, host_heads: int = 0, host_head0: int = 0,
                   copy_stream: int = 0, reload_stream: int = 0):
    """table: numpy int32 [n_seqs][max_blocks], rewritten in place.  Returns (evicted seq ids, report dict)."""
    import numpy as np
    assert table.dtype == np.int32 and table.flags["C_CONTIGUOUS"]
    sl = np.ascontiguousarray(seq_lens, dtype=np.int32)
    lu = np.ascontiguousarray(last_use, dtype=np.int64)
    pool_arr = (vp * n_ranks)(*[(pools.get(r) or None) for r in range(n_ranks)])
    anchor_arr = (i64 * n_ranks)(*[int(head_anchor.get(r, 0)) for r in range(n_ranks)])
    g = etp_kv_geometry(n_layers, n_blocks, block_size, head_cap, head_dim, elem_bytes, layout, n_ranks, pool_arr, anchor_arr,
                        host_backup or None, host_heads, host_head0)
    n_seqs, max_blocks = table.shape
    pt = etp_page_table(n_seqs, max_blocks, table.ctypes.data_as(C.POINTER(i32)), sl.ctypes.data_as(C.POINTER(i32)),
                        lu.ctypes.data_as(C.POINTER(i64)))
    ev = np.zeros(max(n_seqs, 1), dtype=np.int32)
    n_ev = i32()
    rep = etp_reshard_report()
    _check(lib().etp_reshard_kv(ctx.handle, C.byref(g), C.byref(pt), head_plan.handle, new_block_budget, ev.ctypes.data_as(C.POINTER(i32)),
                                C.byref(n_ev), copy_stream or None, reload_stream or None, C.byref(rep)))
    return [int(v) for v in ev[: n_ev.value]], rep.as_dict()


def etp_shard_linear(ctx: Context, mode: int, dtype: str, x_ptr: int, tokens: int, in_features: int, out_features: int,
                     w: TensorDesc, layout: Sequence[Shard], features_per_unit: int, y_ptr: int, stream: int = 0) -> None:
    arr, keep = _marshal_tensors([w])
    _check(lib().etp_shard_linear(ctx.handle, mode, DTYPE[dtype], x_ptr, tokens, in_features, out_features, arr, _shards(layout),
                                  len(layout), features_per_unit, y_ptr, stream or None))
    del keep


class PreparedMultiLinear:
    """Pre-marshalled arguments of one etp_shard_linear_multi call: column-parallel linears (each a PreparedLinear of the same
    class and in_features) fused into one launch; run() takes one output pointer per linear."""

    def __init__(self, linears: Sequence["PreparedLinear"]):
        assert linears and all(l.mode == COL_PARALLEL and l.K == linears[0].K and l.dtype == linears[0].dtype for l in linears)
        self.lins = list(linears)
        self.K, self.dtype = linears[0].K, linears[0].dtype
        self.layout, self.n = linears[0].layout, linears[0].n
        self.outs = (etp_linear_out * len(linears))()
        for i, l in enumerate(linears):
            self.outs[i] = etp_linear_out(C.cast(l.arr, C.POINTER(etp_tensor)), l.N, l.fpu, None)

    def run(self, ctx: Context, x_ptr: int, tokens: int, y_ptrs: Sequence[int], stream: int = 0) -> None:
        for i, y in enumerate(y_ptrs):
            self.outs[i].y = y
        _check(lib().etp_shard_linear_multi(ctx.handle, self.dtype, x_ptr, tokens, self.K, self.outs, len(self.lins), self.layout, self.n,
                                            stream or None))


class LinearPlan:
    """Owns an etp_linear_plan: a prepared group of 1..8 independent shard linears (each a PreparedLinear: mode, shapes, weight
    descriptor, layout).  run() takes one x and one y pointer per linear (or a single x shared by all)."""

    def __init__(self, ctx: Context, linears: Sequence["PreparedLinear"]):
        assert linears and all(l.dtype == linears[0].dtype for l in linears)
        self.lins = list(linears)          # keeps the marshalled descriptors alive while prepare() reads them
        n = len(linears)
        specs = (etp_linear_spec * n)()
        for i, l in enumerate(linears):
            specs[i] = etp_linear_spec(l.mode, 0, l.K, l.N, C.cast(l.arr, C.POINTER(etp_tensor)), l.layout, l.n, 0, l.fpu)
        h = vp()
        _check(lib().etp_linear_prepare(ctx.handle, linears[0].dtype, specs, n, C.byref(h)))
        self.handle, self.n, self.ctx = h, n, ctx
        self._x, self._y = (vp * n)(), (vp * n)()

    def run(self, x_ptrs, tokens: int, y_ptrs: Sequence[int], stream: int = 0) -> None:
        if isinstance(x_ptrs, int):
            x_ptrs = [x_ptrs] * self.n
        for i in range(self.n):
            self._x[i], self._y[i] = x_ptrs[i], y_ptrs[i]
        _check(lib().etp_linear_run(self.handle, self._x, tokens, self._y, stream or None))

    def info(self) -> Dict[str, object]:
        st = etp_linear_plan_stats()
        _check(lib().etp_linear_plan_info(self.handle, C.byref(st)))
        d = {n: getattr(st, n) for n, _ in st._fields_ if n != "n_splits"}
        d["n_splits"] = list(st.n_splits)[: st.n_linears]
        return d

    def close(self) -> None:
        if getattr(self, "handle", None) and _lib is not None:      # also after the ctx was closed: the free needs only the plan
            _lib.etp_linear_free(self.handle)
        self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def etp_moe_linear(ctx: Context, mode: int, dtype: str, x_ptr: int, row_offsets: Sequence[int], in_features: int, out_features: int,
                   w: TensorDesc, layout: Sequence[Shard], y_ptr: int, stream: int = 0) -> None:
    """row_offsets: n_experts + 1 host offsets into the expert-grouped rows of x / y."""
    arr, keep = _marshal_tensors([w])
    n = len(row_offsets) - 1
    offs = (i64 * (n + 1))(*[int(v) for v in row_offsets])
    _check(lib().etp_moe_linear(ctx.handle, mode, DTYPE[dtype], x_ptr, offs, n, in_features, out_features, arr, _shards(layout),
                                len(layout), y_ptr, stream or None))
    del keep


def _instances(instances):
    """[(expert, rank, slot, row_begin, row_end)] -> ctypes array"""
    arr = (etp_moe_instance * max(len(instances), 1))()
    for i, (e, r, s, b, en) in enumerate(instances):
        arr[i] = etp_moe_instance(int(e), int(r), int(s), int(b), int(en))
    return arr


def etp_moe_linear_instances(ctx: Context, mode: int, dtype: str, x_ptr: int, instances, n_rows: int, n_experts: int, in_features: int,
                             out_features: int, w: TensorDesc, y_ptr: int, stream: int = 0) -> None:
    arr, keep = _marshal_tensors([w])
    _check(lib().etp_moe_linear_instances(ctx.handle, mode, DTYPE[dtype], x_ptr, _instances(instances), len(instances), n_rows, n_experts,
                                          in_features, out_features, arr, y_ptr, stream or None))
    del keep


def etp_moe_gate_up(ctx: Context, dtype: str, x_ptr: int, in_features: int, ffn: int, w_gate: TensorDesc, w_up: TensorDesc, h_ptr: int,
                    row_offsets: Optional[Sequence[int]] = None, layout: Optional[Sequence[Shard]] = None, instances=None,
                    n_rows: int = 0, stream: int = 0) -> None:
    """Fused gate | up + SwiGLU.  Either (row_offsets, layout) or (instances, n_rows)."""
    ag, kg = _marshal_tensors([w_gate])
    au, ku = _marshal_tensors([w_up])
    n_experts = w_gate.total_units
    if instances is not None:
        _check(lib().etp_moe_gate_up(ctx.handle, DTYPE[dtype], x_ptr, None, _instances(instances), len(instances), n_rows, n_experts,
                                     in_features, ffn, ag, au, None, 0, h_ptr, stream or None))
    else:
        offs = (i64 * len(row_offsets))(*[int(v) for v in row_offsets])
        _check(lib().etp_moe_gate_up(ctx.handle, DTYPE[dtype], x_ptr, offs, None, 0, 0, n_experts, in_features, ffn, ag, au,
                                     _shards(layout), len(layout), h_ptr, stream or None))
    del kg, ku


def etp_eplb_apply(ctx: Context, tensors: Sequence[TensorDesc], layout: Sequence[Shard], replicas: Sequence[Tuple[int, int]],
                   stream: int = 0) -> List[int]:
    """Copies every replica's expert into the lowest spare slot of its rank, in every tensor; returns the slots."""
    arr, keep = _marshal_tensors(tensors)
    reps = (etp_replica * max(len(replicas), 1))(*[etp_replica(int(e), int(r)) for (e, r) in replicas])
    slots = (i64 * max(len(replicas), 1))()
    _check(lib().etp_eplb_apply(ctx.handle, arr, len(tensors), _shards(layout), len(layout), reps, len(replicas), slots, stream or None))
    del keep
    return [int(s) for s in slots[: len(replicas)]]


class PreparedLinear:
    """Pre-marshalled arguments of one etp_shard_linear call (weight descriptor + layout), so that a timed loop pays only
    the C call."""

    def __init__(self, mode: int, dtype: str, in_features: int, out_features: int, w: TensorDesc, layout: Sequence[Shard],
                 features_per_unit: int):
        self.mode, self.dtype, self.K, self.N, self.fpu = mode, DTYPE[dtype], in_features, out_features, features_per_unit
        self.arr, self._keep = _marshal_tensors([w])
        self.layout, self.n = _shards(layout), len(layout)

    def run(self, ctx: Context, x_ptr: int, tokens: int, y_ptr: int, stream: int = 0) -> None:
        _check(lib().etp_shard_linear(ctx.handle, self.mode, self.dtype, x_ptr, tokens, self.K, self.N, self.arr, self.layout,
                                      self.n, self.fpu, y_ptr, stream or None))


class IntervalList:
    """Pre-marshalled etp_interval array (src, dst, bytes as absolute addresses / byte counts), optionally in page-locked
    memory so that the library's DMA reads it in place; a timed loop then pays only the C call."""

    def __init__(self, src_ptrs, dst_ptrs, sizes, pin: bool = False):
        import numpy as np
        self.n = len(sizes)
        if pin:
            import torch
            self._t = torch.empty((max(self.n, 1), 3), dtype=torch.int64).pin_memory()
            self.rec = self._t.numpy()
        else:
            self.rec = np.empty((max(self.n, 1), 3), dtype=np.int64)
        self.rec[: self.n, 0], self.rec[: self.n, 1], self.rec[: self.n, 2] = src_ptrs, dst_ptrs, sizes

    def run(self, ctx: Context, stream: int = 0) -> Dict[str, float]:
        rep = etp_reshard_report()
        _check(lib().etp_copy_intervals(ctx.handle, self.rec.ctypes.data_as(C.POINTER(etp_interval)), self.n, stream or None, C.byref(rep)))
        return rep.as_dict()

    def run_static(self, stream: int = 0) -> None:
        """etp_copy_intervals_static: no Context, nothing allocated (scratch in the library's static device array)."""
        _check(lib().etp_copy_intervals_static(self.rec.ctypes.data_as(C.POINTER(etp_interval)), self.n, stream or None))

    def validate(self) -> None:
        """etp_intervals_validate (host-only, no context): raises EtpError as etp_copy_intervals would."""
        _check(lib().etp_intervals_validate(self.rec.ctypes.data_as(C.POINTER(etp_interval)), self.n))


def etp_intervals_validate(src_ptrs, dst_ptrs, sizes) -> None:
    IntervalList(src_ptrs, dst_ptrs, sizes).validate()


def etp_copy_intervals(ctx: Context, src_ptrs, dst_ptrs, sizes, stream: int = 0) -> Dict[str, float]:
    """src_ptrs / dst_ptrs / sizes: numpy int64 arrays of absolute device addresses and byte counts."""
    return IntervalList(src_ptrs, dst_ptrs, sizes).run(ctx, stream)


def etp_copy_intervals_static(src_ptrs, dst_ptrs, sizes, stream: int = 0) -> None:
    """The copy of etp_copy_intervals for callers that must not allocate device memory (a recovery path running while the serving
    engine's pool owns all free HBM, code inside somebody else's CUDA context): no Context, at most 4096 intervals per call, runs on
    the current CUDA device.  Calls share one static scratch array: keep them on one stream or order them yourself (include/etp.h)."""
    IntervalList(src_ptrs, dst_ptrs, sizes).run_static(stream)


def etp_debug_starved_wait(ctx: Context, stream: int = 0) -> None:
    """Launches a kernel that waits on a barrier nobody arrives on: raises EtpError(ETP_ERR_CUDA) with the fault record after about
    10 s.  The CUDA context of the process is lost afterwards: throw-away processes only."""
    _check(lib().etp_debug_starved_wait(ctx.handle, stream or None))
