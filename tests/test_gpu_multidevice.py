"""The destination-partitioned executor on ONE physical GPU: every logical
device of the ctx aliases cuda:0, so the per-device streams, descriptor arenas, cross-device hazard events and the fork /
join with the caller's streams all run for real, and the result must be bit-exact to the oracle exactly as in the
single-device tests.  Also the one-process-per-GPU form: two contexts that each write only "their" ranks (rank map -1 for
the others) and pull from everybody's slabs."""
import dataclasses

import numpy as np
import pytest
import torch

import paper_2511_11617_b200 as etp
from oracle import planning as OP
from oracle import state as OS
from tests import harness as H
from tests.gpu_util import DevBuf, LibSide, Streams, make_plans, pinned
from tests.test_gpu_reshard import MID, compare_params, tensor_descs, upload_param_world

pytestmark = pytest.mark.gpu


def bytes_by_destination(world, step_idx, rank_dev, n_dev):
    """(d2d, reload) bytes per logical device from the ORACLE's task lists: a task belongs to the device of its dst rank."""
    st = world.steps[step_idx]
    d2d, rel = [0] * n_dev, [0] * n_dev
    for sp in world.specs:
        for (kind, src, dst, b, e) in st.tasks[sp.klass]:
            d = rank_dev[dst]
            if d < 0:
                continue
            if kind == OP.TRANSFER:
                d2d[d] += (e - b) * sp.unit_bytes
            elif kind == OP.RELOAD:
                rel[d] += (e - b) * sp.unit_bytes
    return d2d, rel


def run_params(ctx, world, bufs, images, step_idx, streams):
    step = world.steps[step_idx]
    plans = make_plans(step)
    klasses = sorted(plans)
    descs = tensor_descs(world, bufs, images, step, {k: i for i, k in enumerate(klasses)})
    return etp.etp_reshard_params(ctx, descs, [plans[k] for k in klasses], streams.copy.cuda_stream, streams.reload.cuda_stream)


@pytest.mark.parametrize("mode", ["span", "tight"])
@pytest.mark.parametrize("image", ["pinned", "device"])
@pytest.mark.parametrize("n_dev", [2, 3])
def test_params_partitioned_by_destination_device(mode, image, n_dev):
    world = H.build_param_world(MID, side=LibSide, mode=mode, failed=(2,))
    expect, stats = H.oracle_reshard_params(world, 0)
    bufs, images = upload_param_world(world, image)
    rank_dev = [r % n_dev for r in range(4)]
    ctx = etp.Context(devices=[0] * n_dev)
    try:
        ctx.set_rank_devices(rank_dev)
        s = Streams()
        rep = run_params(ctx, world, bufs, images, 0, s)
        s.sync()                                   # the caller's two streams only: the library joined its own into them
        compare_params(world, bufs, expect, {2})
        assert rep["d2d_bytes"] == stats["d2d_bytes"] and rep["h2d_bytes"] + rep["reload_dev_bytes"] == stats["h2d_bytes"]
        assert rep["remote_bytes"] == 0
        if mode == "tight":
            assert rep["n_phases"] >= 2
        d2d, rel = bytes_by_destination(world, 0, rank_dev, n_dev)
        per = [ctx.device_report(d) for d in range(n_dev)]
        assert [p["d2d_bytes"] for p in per] == d2d                      # each device wrote exactly its own ranks' incoming bytes
        assert [p["h2d_bytes"] + p["reload_dev_bytes"] for p in per] == rel
        assert sum(p["n_kernel_launches"] for p in per) == rep["n_kernel_launches"]
        assert all((p["n_kernel_launches"] > 0) == (p["d2d_bytes"] + p["reload_dev_bytes"] > 0) for p in per)
    finally:
        ctx.close()


@pytest.mark.parametrize("layout", [0, 1])
def test_kv_partitioned_by_destination_device(layout):
    cfg = dataclasses.replace(MID, model=dataclasses.replace(MID.model, n_layers=2))
    world = H.build_kv_world(cfg, side=LibSide, layout=layout, seq_lens=[300, 7, 1000], head_cap=4)
    st, g = world.steps[0], world.g
    live = int(((world.seq_lens + 15) // 16).sum())
    budget = live + 3                                                     # relocations of kept heads (same-rank copies) too
    new_table, evicted, pairs = OS.page_table_rewrite(world.table, world.seq_lens, world.last_use, g.block_size, budget)
    snap = {r: p for r, p in world.pools.items() if r != st.dead}
    expect, stats = OS.apply_kv(st.tasks["head"], snap, world.anchors, g, world.host_backup, world.host_heads, world.host_head0, pairs)
    bufs = {r: DevBuf(p) for r, p in snap.items()}
    img = pinned(world.host_backup)
    ctx = etp.Context(devices=[0, 0])
    try:
        ctx.set_rank_devices([0, 1, 1, 0])
        table = world.table.copy()
        s = Streams()
        ev, rep = etp.etp_reshard_kv(ctx, n_layers=g.n_layers, n_blocks=g.n_blocks, block_size=g.block_size, head_cap=g.head_cap,
                                     head_dim=g.head_dim, elem_bytes=g.elem_bytes, layout=g.layout, pools={r: b.ptr for r, b in bufs.items()},
                                     head_anchor=world.anchors, n_ranks=4, table=table, seq_lens=world.seq_lens, last_use=world.last_use,
                                     head_plan=make_plans(st)["head"], new_block_budget=budget, host_backup=img.data_ptr(),
                                     host_heads=world.host_heads, host_head0=world.host_head0, copy_stream=s.copy.cuda_stream,
                                     reload_stream=s.reload.cuda_stream)
        s.sync()
        assert ev == evicted and np.array_equal(table, new_table)
        for r, b in bufs.items():
            assert b.guards_intact() and b.payload().tobytes() == expect[r].tobytes(), f"pool of rank {r} differs from the oracle image"
        assert rep["d2d_bytes"] == stats["d2d_bytes"] and rep["h2d_bytes"] == stats["h2d_bytes"]
        per = [ctx.device_report(d) for d in range(2)]
        assert sum(p["d2d_bytes"] for p in per) == stats["d2d_bytes"] and sum(p["h2d_bytes"] for p in per) == stats["h2d_bytes"]
    finally:
        ctx.close()


@pytest.mark.parametrize("form", ["two_contexts", "three_devices"])
@pytest.mark.parametrize("budget_delta", [3, -10])
def test_kv_phase_by_phase_keeps_the_original_table(form, budget_delta):
    """ETP_OPT_ONLY_PHASE on a KV reshard that needs several hazard phases AND relocates blocks (tight head_cap = the wider shard,
    so a reloaded head lands in the slot another rank still has to read; a block budget that moves live blocks, and with -10 also
    evicts).  Every phase call must lower the plan from the ORIGINAL page table: the call therefore leaves the caller's table
    alone (include/etp.h) - were it rewritten by the phase-1 call, phase 2 would see identity {old, new} pairs and read the
    source pools at the new block ids.  Run as two contexts that each write their own ranks, and as one ctx over three logical
    devices; after the last phase the caller's etp_page_table_rewrite gives the table, and pools / evictions match the oracle."""
    cfg = dataclasses.replace(MID, model=dataclasses.replace(MID.model, n_layers=2))
    world = H.build_kv_world(cfg, side=LibSide, layout=0, seq_lens=[300, 7, 1000])      # head_cap = max shard width (3): tight
    st, g = world.steps[0], world.g
    assert g.head_cap == 3
    live = int(((world.seq_lens + 15) // 16).sum())
    budget = live + budget_delta
    new_table, evicted, pairs = OS.page_table_rewrite(world.table, world.seq_lens, world.last_use, g.block_size, budget)
    assert any(p[2] != p[3] for p in pairs) and (budget_delta > 0 or evicted)          # (seq, index, old id, new id)
    snap = {r: p for r, p in world.pools.items() if r != st.dead}
    expect, stats = OS.apply_kv(st.tasks["head"], snap, world.anchors, g, world.host_backup, world.host_heads, world.host_head0, pairs)
    bufs = {r: DevBuf(p) for r, p in snap.items()}
    img = pinned(world.host_backup)
    if form == "two_contexts":
        ctxs, maps = [etp.Context(0), etp.Context(0)], ([0, -1, -1, 0], [-1, 0, 0, -1])
    else:
        ctxs, maps = [etp.Context(devices=[0, 0, 0])], ([0, 1, 2, 0],)
    try:
        for c, m in zip(ctxs, maps):
            c.set_rank_devices(m)
        streams = [Streams() for _ in ctxs]
        table = world.table.copy()
        phase, n_phases, reps = 0, 1, [None] * len(ctxs)
        while phase < n_phases:
            for i, (c, s) in enumerate(zip(ctxs, streams)):
                c.set_option(etp.OPT_ONLY_PHASE, phase + 1)
                ev, reps[i] = etp.etp_reshard_kv(c, n_layers=g.n_layers, n_blocks=g.n_blocks, block_size=g.block_size, head_cap=g.head_cap,
                                                 head_dim=g.head_dim, elem_bytes=g.elem_bytes, layout=g.layout,
                                                 pools={r: b.ptr for r, b in bufs.items()}, head_anchor=world.anchors, n_ranks=4, table=table,
                                                 seq_lens=world.seq_lens, last_use=world.last_use, head_plan=make_plans(st)["head"],
                                                 new_block_budget=budget, host_backup=img.data_ptr(), host_heads=world.host_heads,
                                                 host_head0=world.host_head0, copy_stream=s.copy.cuda_stream, reload_stream=s.reload.cuda_stream)
                n_phases = reps[i]["n_phases"]
                assert ev == evicted                                    # reported by every phase call
                assert np.array_equal(table, world.table)               # ... and the table is still the original one
            for s in streams:
                s.sync()                                                # the barrier between hazard phases
            phase += 1
        assert n_phases >= 2
        ev2, pairs2 = etp.etp_page_table_rewrite(table, world.seq_lens, world.last_use, g.block_size, budget)
        assert ev2 == evicted and np.array_equal(table, new_table)
        for r, b in bufs.items():
            assert b.guards_intact() and b.payload().tobytes() == expect[r].tobytes(), f"pool of rank {r} differs from the oracle image"
        assert sum(r["d2d_bytes"] for r in reps) == stats["d2d_bytes"] and sum(r["h2d_bytes"] for r in reps) == stats["h2d_bytes"]
    finally:
        for c in ctxs:
            c.close()


@pytest.mark.parametrize("mode", ["span", "tight"])
def test_one_context_per_rank_group_pulls_only_its_own_destinations(mode):
    """The one-process-per-GPU form in one process: context A writes ranks {0, 3}, context B ranks {1, 2} (the others are -1
    in its rank map: valid sources, never written).  Single-phase plans need no coordination at all; multi-phase plans are
    run phase by phase (ETP_OPT_ONLY_PHASE) with a synchronisation in between, as two processes would with a barrier."""
    world = H.build_param_world(MID, side=LibSide, mode=mode, failed=(1,))
    expect, stats = H.oracle_reshard_params(world, 0)
    bufs, images = upload_param_world(world, "pinned")
    maps = ([0, -1, -1, 0], [-1, 0, 0, -1])
    ctxs = [etp.Context(0), etp.Context(0)]
    try:
        for c, m in zip(ctxs, maps):
            c.set_rank_devices(m)
        streams = [Streams(), Streams()]
        reps = [None, None]
        if mode == "span":
            reps = [run_params(c, world, bufs, images, 0, s) for c, s in zip(ctxs, streams)]
            assert all(r["n_phases"] == 1 for r in reps)
        else:
            phase, n_phases = 0, 1
            while phase < n_phases:
                for i, (c, s) in enumerate(zip(ctxs, streams)):
                    c.set_option(etp.OPT_ONLY_PHASE, phase + 1)
                    reps[i] = run_params(c, world, bufs, images, 0, s)      # lowers the whole plan, enqueues this phase only
                    n_phases = reps[i]["n_phases"]
                for s in streams:
                    s.sync()                                                # the barrier between hazard phases
                phase += 1
            assert n_phases >= 2
        for s in streams:
            s.sync()
        compare_params(world, bufs, expect, {1})
        moved = stats["d2d_bytes"] + stats["h2d_bytes"]
        for rep, m in zip(reps, maps):
            d2d, rel = bytes_by_destination(world, 0, m, 1)
            assert rep["d2d_bytes"] == d2d[0] and rep["h2d_bytes"] == rel[0]
            assert rep["remote_bytes"] == moved - d2d[0] - rel[0]
        assert sum(r["d2d_bytes"] for r in reps) == stats["d2d_bytes"] and sum(r["h2d_bytes"] for r in reps) == stats["h2d_bytes"]
    finally:
        for c in ctxs:
            c.close()


def _ipc_worker(rank, rank_map, tensors, world_blob, image_kind, done):
    """A process that owns NOTHING: every slab is a CUDA-IPC mapping of the parent's allocation.  It writes only its ranks."""
    import pickle
    torch.cuda.set_device(0)
    world = pickle.loads(world_blob)

    class Buf:
        def __init__(self, t):
            self.t = t
            self.ptr = t.data_ptr()

    bufs = {name: {r: Buf(t) for r, t in per.items()} for name, per in tensors.items()}
    images = {sp.name: pinned(world.unsharded[sp.name]) for sp in world.specs}
    ctx = etp.Context(0)
    ctx.set_rank_devices(rank_map)
    s = Streams()
    rep = run_params(ctx, world, bufs, images, 0, s)
    s.sync()
    ctx.close()
    done.put((rank, rep["d2d_bytes"], rep["h2d_bytes"], rep["remote_bytes"]))


def test_two_processes_pull_through_cuda_ipc_mappings():
    """Two worker PROCESSES on the one GPU, each with its own ctx and a rank map that makes it write half of the ranks; the
    slabs are CUDA-IPC mappings of allocations they do not own (what a process per GPU sees of its peers' memory).  Neither
    kernel waits for the other; the parent compares the shared slabs with the oracle once both have exited."""
    import pickle
    import torch.multiprocessing as mp
    world = H.build_param_world(MID, side=LibSide, mode="span", failed=(1,))
    expect, stats = H.oracle_reshard_params(world, 0)
    tensors = {sp.name: {r: torch.from_numpy(a).cuda() for r, a in world.slabs[sp.name].items()} for sp in world.specs}
    torch.cuda.synchronize()
    mpc = mp.get_context("spawn")
    done = mpc.Queue()
    blob = pickle.dumps(world)
    maps = ([0, -1, -1, 0], [-1, 0, 0, -1])
    procs = [mpc.Process(target=_ipc_worker, args=(i, maps[i], tensors, blob, "pinned", done)) for i in range(2)]
    for p in procs:
        p.start()
    got = [done.get(timeout=300) for _ in procs]
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    torch.cuda.synchronize()
    for sp in world.specs:
        for r, t in tensors[sp.name].items():
            if r != 1:
                assert t.cpu().numpy().tobytes() == expect[sp.name][r].tobytes(), f"{sp.name} rank {r}: slab differs from the oracle image"
    assert sum(g[1] for g in got) == stats["d2d_bytes"] and sum(g[2] for g in got) == stats["h2d_bytes"]
    assert all(g[3] > 0 for g in got)


def _torchrun(script_args, n=2, timeout=900):
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, ETP_BENCH_ALIAS_GPU0="1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", "29617"] + script_args
    return subprocess.run(cmd, cwd=root, env=env, capture_output=True, text=True, timeout=timeout)


@pytest.mark.parametrize("n", [2, 3])
def test_sharded_state_one_process_per_rank_group(n):
    """tests/sharded_check.py under torchrun: the sharded ModelState (CUDA-IPC mapped peers) resharded by N processes, whole state
    against the plain definition in every process."""
    r = _torchrun(["tests/sharded_check.py", "2", "2", "8"], n=n)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-3000:]
    assert r.stdout.count("SHARDED_OK") == n


def test_bench_sharded_moves_the_same_bytes_as_one_process():
    """`bench.py --gpus 2 --sharded` (two processes aliased to cuda:0) prints the contract line, strong scaling, and moves exactly
    the bytes the single-process run of the same reduced workload moves."""
    import json
    common = ["bench.py", "--sharded", "--config", "2", "--layers", "2", "--seqs", "4", "--steps", "2", "--warmup", "1"]
    two = _torchrun(common + ["--gpus", "2"], n=2)
    assert two.returncode == 0, two.stdout[-3000:] + two.stderr[-3000:]
    one = _torchrun(common + ["--gpus", "1"], n=1)
    assert one.returncode == 0, one.stdout[-3000:] + one.stderr[-3000:]
    l2 = json.loads([l for l in two.stdout.splitlines() if l.startswith("{")][-1])
    l1 = json.loads([l for l in one.stdout.splitlines() if l.startswith("{")][-1])
    assert l2["n_gpus"] == 2 and l2["scaling"] == "strong" and l2["config"]["aliased_to_gpu0"] is True
    assert l2["config"]["moved_GB_per_step"] == l1["config"]["moved_GB_per_step"] > 0
    assert l2["e2e"]["h2d_bytes_per_step"] == l1["e2e"]["h2d_bytes_per_step"] > 0
