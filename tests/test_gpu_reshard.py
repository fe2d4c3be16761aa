"""Parity proper: the CUDA path (through the C ABI) against the CPU oracle, byte for byte.

Whole slabs / whole pools are compared (not only the new shards), so a byte written outside the plan fails
(reading L6), and every device buffer sits between guard bands."""
import dataclasses

import numpy as np
import pytest
import torch

import paper_2511_11617_b200 as etp
from oracle import state as OS
from tests import harness as H
from tests.gpu_util import DevBuf, LibSide, Streams, make_plans, pinned
from workloads import get_config
from workloads.configs import FFN, HEAD, VOCAB, Config, KVShape, ModelShape, Scenario
from workloads.gen import microbench_intervals

pytestmark = pytest.mark.gpu

# a shape whose transfers span several 256-KiB bulk jobs and 32-KiB ring stages with ragged tails
MID = Config(1, "mid", ModelShape("mid-dense", 2, 1024, 16, 8, 64, ffn=2731, vocab=5003, dtype="bf16"),
             KVShape(3, 1000), Scenario(4, (1,), old_widths={FFN: (700, 650, 720, 661)}), tokens=4)


@pytest.fixture(scope="module")
def ctx():
    c = etp.Context(0)
    yield c
    c.close()


def upload_param_world(world, image="pinned"):
    bufs, descs, images = {}, {}, {}
    for sp in world.specs:
        bufs[sp.name] = {r: DevBuf(a) for r, a in world.slabs[sp.name].items()}
        if image == "pinned":
            images[sp.name] = pinned(world.unsharded[sp.name])
        else:
            images[sp.name] = torch.from_numpy(world.unsharded[sp.name]).cuda()
    return bufs, images


def tensor_descs(world, bufs, images, step, class_index):
    n_ranks = max(r for (r, _, _, _) in world.steps[0].old[world.specs[0].klass]) + 1
    out = []
    for sp in world.specs:
        slabs = {}
        for r, b in bufs[sp.name].items():
            if r == step.dead:
                continue
            anchor, cap = world.geom[sp.name][r]
            slabs[r] = (b.ptr, cap, anchor)
        out.append(etp.TensorDesc(sp.total_units, sp.unit_bytes, slabs, n_ranks, class_index[sp.klass],
                                  images[sp.name].data_ptr(), 0, sp.total_units))
    return out


def run_param_step(ctx, world, bufs, images, step_idx, streams, mode=0):
    step = world.steps[step_idx]
    plans = make_plans(step, mode)
    klasses = sorted(plans)
    class_index = {k: i for i, k in enumerate(klasses)}
    descs = tensor_descs(world, bufs, images, step, class_index)
    rep = etp.etp_reshard_params(ctx, descs, [plans[k] for k in klasses], streams.copy.cuda_stream, streams.reload.cuda_stream)
    streams.sync()
    return rep


def compare_params(world, bufs, expect, dead_ranks):
    for sp in world.specs:
        for r, b in bufs[sp.name].items():
            assert b.guards_intact(), f"{sp.name} rank {r}: guard band overwritten"
            if r in dead_ranks:
                continue
            got = b.payload()
            assert got.tobytes() == expect[sp.name][r].tobytes(), f"{sp.name} rank {r}: slab differs from the oracle image"


@pytest.mark.parametrize("mode", ["span", "tight", "full"])
@pytest.mark.parametrize("policy", ["floor", "ceil_first"])
@pytest.mark.parametrize("dead", [0, 1, 2, 3])
def test_config1_params_bit_exact(ctx, mode, policy, dead):
    cfg = get_config("1")
    world = H.build_param_world(cfg, side=LibSide, mode=mode, new_policy=policy, failed=(dead,))
    expect, stats = H.oracle_reshard_params(world, 0)
    bufs, images = upload_param_world(world)
    rep = run_param_step(ctx, world, bufs, images, 0, Streams())
    compare_params(world, bufs, expect, {dead})
    assert rep["d2d_bytes"] == stats["d2d_bytes"] and rep["h2d_bytes"] == stats["h2d_bytes"]
    assert rep["kept_bytes"] == stats["kept_bytes"]
    assert rep["n_kernel_launches"] >= (1 if stats["d2d_bytes"] else 0)
    if mode != "tight":
        assert rep["n_phases"] == 1


@pytest.mark.parametrize("image", ["pinned", "device"])
@pytest.mark.parametrize("tma_min", [None, 16, 1 << 62])
@pytest.mark.parametrize("steal", [0, 1])
def test_mid_params_bit_exact_every_copy_path(ctx, image, tma_min, steal):
    """Multi-tile sizes with ragged tails; TMA-only, vector-only and mixed routing of the same plan; with
    ETP_OPT_LDG_STEALS_BULK the vector warps also drain the bulk queue (both engines race for the same items)."""
    world = H.build_param_world(MID, side=LibSide, mode="span")
    expect, stats = H.oracle_reshard_params(world, 0)
    bufs, images = upload_param_world(world, image)
    default = ctx.get_option(etp.OPT_TMA_MIN_BYTES)
    try:
        if tma_min is not None:
            ctx.set_option(etp.OPT_TMA_MIN_BYTES, tma_min)
        ctx.set_option(etp.OPT_LDG_STEALS_BULK, steal)
        rep = run_param_step(ctx, world, bufs, images, 0, Streams())
    finally:
        ctx.set_option(etp.OPT_TMA_MIN_BYTES, default)
        ctx.set_option(etp.OPT_LDG_STEALS_BULK, 0)
    compare_params(world, bufs, expect, {1})
    assert rep["d2d_bytes"] == stats["d2d_bytes"]
    assert rep["h2d_bytes"] + rep["reload_dev_bytes"] == stats["h2d_bytes"]


@pytest.mark.parametrize("planner", ["greedy", "full_reload"])
def test_comparison_planners_bit_exact(ctx, planner):
    """PAPER.md:204 / Table II: the Greedy (no P2P for gaps) and Full Reload (no reuse) planners through the same lowering and
    the same reload pipeline, against the oracle applying the oracle's own plan of that kind; Full Reload moves no byte D2D."""
    from oracle import planning as OP
    fn, mode = {"greedy": (OP.greedy_plan, etp.PLAN_GREEDY), "full_reload": (OP.full_reload_plan, etp.PLAN_FULL_RELOAD)}[planner]

    class Side(LibSide):
        @staticmethod
        def plan(old, M, tb=None):
            return fn(old, M, tb)

    world = H.build_param_world(MID, side=Side, mode="span")
    expect, stats = H.oracle_reshard_params(world, 0)
    assert stats["d2d_bytes"] == 0
    bufs, images = upload_param_world(world)
    rep = run_param_step(ctx, world, bufs, images, 0, Streams(), mode=mode)
    compare_params(world, bufs, expect, {1})
    assert rep["d2d_bytes"] == 0 and rep["h2d_bytes"] == stats["h2d_bytes"]
    if planner == "full_reload":
        assert rep["kept_bytes"] == 0 and rep["h2d_bytes"] == sum(sp.total_units * sp.unit_bytes for sp in world.specs)


@pytest.mark.parametrize("mode", ["span", "tight"])
def test_sequential_failures_bit_exact(ctx, mode):
    """Config-5a style chain (PAPER.md:206 k -> k-1 switches) on the mid shape: 4 -> 3 -> 2, in place."""
    world = H.build_param_world(MID, side=LibSide, mode=mode, failed=(2, 0))
    bufs, images = upload_param_world(world)
    cur, dead = world.slabs, set()
    streams = Streams()
    for i in range(2):
        expect, _ = H.oracle_reshard_params(world, i, cur)
        rep = run_param_step(ctx, world, bufs, images, i, streams)
        dead.add(world.steps[i].dead)
        compare_params(world, bufs, expect, dead)
        cur = expect
        if mode == "tight":
            assert rep["n_phases"] >= 1


def test_same_stream_and_skip_options(ctx):
    world = H.build_param_world(MID, side=LibSide, mode="span")
    expect, stats = H.oracle_reshard_params(world, 0)
    bufs, images = upload_param_world(world)
    s = Streams()
    s.reload = s.copy                       # one stream for both legs
    run_param_step(ctx, world, bufs, images, 0, s)
    compare_params(world, bufs, expect, {1})
    # SKIP_D2D + SKIP_RELOAD touch nothing
    bufs2, images2 = upload_param_world(world)
    ctx.set_option(etp.OPT_SKIP_D2D, 1)
    ctx.set_option(etp.OPT_SKIP_RELOAD, 1)
    try:
        run_param_step(ctx, world, bufs2, images2, 0, Streams())
    finally:
        ctx.set_option(etp.OPT_SKIP_D2D, 0)
        ctx.set_option(etp.OPT_SKIP_RELOAD, 0)
    compare_params(world, bufs2, world.slabs, {1})


def test_param_errors(ctx):
    world = H.build_param_world(get_config("1"), side=LibSide, mode="span")
    bufs, images = upload_param_world(world)
    step = world.steps[0]
    plans = make_plans(step)
    klasses = sorted(plans)
    ci = {k: i for i, k in enumerate(klasses)}
    descs = tensor_descs(world, bufs, images, step, ci)
    pl = [plans[k] for k in klasses]
    s = Streams()
    bad = tensor_descs(world, bufs, images, step, ci)
    bad[0].host_image = 0
    with pytest.raises(etp.EtpError) as e:
        etp.etp_reshard_params(ctx, bad, pl, s.copy.cuda_stream, s.reload.cuda_stream)
    assert e.value.status == 4              # NO_SOURCE
    bad = tensor_descs(world, bufs, images, step, ci)
    r0 = min(bad[4].slabs)
    p, cap, a = bad[4].slabs[r0]
    bad[4].slabs[r0] = (p + 8, cap, a)
    with pytest.raises(etp.EtpError) as e:
        etp.etp_reshard_params(ctx, bad, pl, s.copy.cuda_stream, s.reload.cuda_stream)
    assert e.value.status == 2              # ALIGNMENT
    bad = tensor_descs(world, bufs, images, step, ci)
    for r in bad[4].slabs:
        p, cap, a = bad[4].slabs[r]
        bad[4].slabs[r] = (p, 3, a)
    with pytest.raises(etp.EtpError) as e:
        etp.etp_reshard_params(ctx, bad, pl, s.copy.cuda_stream, s.reload.cuda_stream)
    assert e.value.status == 3              # CAPACITY
    s.sync()
    compare_params(world, bufs, world.slabs, {step.dead})     # failed calls wrote nothing
    del descs


# ------------------------------------------------------------------------------------------------ KV
def run_kv(ctx, world, budget, backup="pinned", head_cap=None, plan=None):
    st = world.steps[0]
    g = world.g
    new_table, evicted, pairs = OS.page_table_rewrite(world.table, world.seq_lens, world.last_use, g.block_size, budget)
    snap = {r: p for r, p in world.pools.items() if r != st.dead}
    hb = world.host_backup if backup else None
    expect, stats = OS.apply_kv(st.tasks["head"], snap, world.anchors, g, hb, world.host_heads, world.host_head0, pairs)
    bufs = {r: DevBuf(p) for r, p in snap.items()}
    if backup == "pinned":
        img = pinned(world.host_backup)
    elif backup == "device":
        img = torch.from_numpy(world.host_backup).cuda()
    else:
        img = None
    plan = plan or make_plans(st)["head"]
    n_ranks = max(world.pools) + 1
    table = world.table.copy()
    s = Streams()
    ev, rep = etp.etp_reshard_kv(ctx, n_layers=g.n_layers, n_blocks=g.n_blocks, block_size=g.block_size, head_cap=g.head_cap,
                                 head_dim=g.head_dim, elem_bytes=g.elem_bytes, layout=g.layout,
                                 pools={r: b.ptr for r, b in bufs.items()}, head_anchor=world.anchors, n_ranks=n_ranks,
                                 table=table, seq_lens=world.seq_lens, last_use=world.last_use, head_plan=plan,
                                 new_block_budget=budget, host_backup=img.data_ptr() if img is not None else 0,
                                 host_heads=world.host_heads, host_head0=world.host_head0,
                                 copy_stream=s.copy.cuda_stream, reload_stream=s.reload.cuda_stream)
    s.sync()
    assert np.array_equal(table, new_table)
    for r, b in bufs.items():
        assert b.guards_intact()
        assert b.payload().tobytes() == expect[r].tobytes(), f"pool of rank {r} differs from the oracle image"
    return ev, evicted, rep, stats


@pytest.mark.parametrize("layout", [0, 1])
@pytest.mark.parametrize("dead", [0, 1, 2, 3])
@pytest.mark.parametrize("budget", [None, 12])
def test_config1_kv_bit_exact(ctx, layout, dead, budget):
    world = H.build_kv_world(get_config("1"), side=LibSide, layout=layout, failed=(dead,))
    bud = world.g.n_blocks if budget is None else budget
    ev, evicted, rep, stats = run_kv(ctx, world, bud)
    assert ev == evicted
    assert rep["d2d_bytes"] == stats["d2d_bytes"] and rep["h2d_bytes"] == stats["h2d_bytes"]


@pytest.mark.parametrize("layout", [0, 1])
@pytest.mark.parametrize("backup", ["pinned", "device"])
@pytest.mark.parametrize("policy", ["floor", "ceil_first"])
def test_mid_kv_bit_exact(ctx, layout, backup, policy):
    """Ragged sequence lengths (a 1-block sequence, a partial last block), 8 KV heads 4 -> 3, head_cap with slack."""
    cfg = dataclasses.replace(MID, model=dataclasses.replace(MID.model, n_layers=2))
    world = H.build_kv_world(cfg, side=LibSide, layout=layout, new_policy=policy, seq_lens=[300, 7, 1000], head_cap=4)
    ev, evicted, rep, stats = run_kv(ctx, world, world.g.n_blocks, backup)
    assert ev == evicted == []
    assert rep["d2d_bytes"] == stats["d2d_bytes"]
    assert rep["h2d_bytes"] + rep["reload_dev_bytes"] == stats["h2d_bytes"]


def test_kv_budget_shrink_and_no_backup(ctx):
    cfg = dataclasses.replace(MID, model=dataclasses.replace(MID.model, n_layers=1))
    world = H.build_kv_world(cfg, side=LibSide, layout=0, seq_lens=[300, 7, 1000], head_cap=4)
    live = int(((world.seq_lens + 15) // 16).sum())
    ev, evicted, rep, stats = run_kv(ctx, world, live - 10)
    assert ev == evicted and len(ev) >= 1
    # reading K4: no backup -> reload heads untouched, every live sequence reported
    ev, evicted, rep, stats = run_kv(ctx, world, world.g.n_blocks, backup=None)
    assert sorted(ev) == [0, 1, 2] and rep["h2d_bytes"] == 0


# ------------------------------------------------------------------------------------------------ scale-up (a rank joins)
@pytest.mark.parametrize("tight", [False, True])
def test_scale_up_a_repaired_rank_joins(ctx, tight):
    """PAPER.md:168 (scale-up after a GPU is repaired), reading C6: the joining rank is an ALIVE rank with an empty interval.
    3 -> 4 ranks of 1201 units x 4112 B; nothing is reloaded, every target tiles from transfers and keeps; with tight slabs
    (cap = the wider of old and new shard) shards wrap and the plan needs hazard phases."""
    from oracle import planning as OP
    Hn, ub = 1201, 4112
    old = [(0, 0, 400, 1), (1, 400, 800, 1), (2, 800, Hn, 1), (3, Hn, Hn, 1)]
    tasks, new = OP.cmm_plan(old, 4)
    assert OP.plan_stats(tasks)["reload_units"] == 0 and new[3][2] - new[3][1] > 0
    geom = {}
    for (r, b, e, _), (_, nb, ne, _) in zip(old, new):
        if tight:
            geom[r] = (b if e > b else nb, max(e - b, ne - nb))
        else:
            lo, hi = (min(b, nb), max(e, ne)) if e > b else (nb, ne)
            geom[r] = (lo, hi - lo)
    rng = np.random.default_rng(11)
    w = rng.integers(0, 256, Hn * ub, dtype=np.uint8)
    slabs = {}
    for (r, b, e, _) in old:
        anchor, cap = geom[r]
        slab = rng.integers(0, 256, cap * ub, dtype=np.uint8)
        OS.place_units(slab, anchor, cap, ub, b, e, w)
        slabs[r] = slab
    expect, stats = OS.apply_params(tasks, slabs, geom, ub, None, 0)
    for (r, b, e, _) in new:                       # the plain definition: every new shard is the unsharded slice
        assert np.array_equal(OS.read_units(expect[r], *geom[r], ub, b, e), w[b * ub:e * ub])
    bufs = {r: DevBuf(a) for r, a in slabs.items()}
    plan = etp.etp_cmm_plan(old, 4)
    assert plan.tasks() == [tuple(t) for t in tasks]
    desc = etp.TensorDesc(Hn, ub, {r: (bufs[r].ptr, geom[r][1], geom[r][0]) for r in bufs}, 4, 0)
    st = Streams()
    rep = etp.etp_reshard_params(ctx, [desc], [plan], st.copy.cuda_stream, st.reload.cuda_stream)
    st.sync()
    assert rep["d2d_bytes"] == stats["d2d_bytes"] and rep["h2d_bytes"] == 0
    assert rep["n_phases"] >= 2 if tight else rep["n_phases"] == 1
    for r, b in bufs.items():
        assert b.guards_intact()
        assert np.array_equal(b.payload(), expect[r]), f"rank {r}: slab differs from the oracle image"


# ------------------------------------------------------------------------------------------------ migration-aware plan
class MigSide(LibSide):
    """plans with the owner of every target chosen to minimise transfers (reading M1); bounds as the scenario gives them"""
    name = "libetp-migration-aware"

    @staticmethod
    def plan(old, M, tb=None):
        p = etp.etp_plan_create(etp.PLAN_MIGRATION_AWARE, old, M, tb)
        return p.tasks(), p.new_layout()


@pytest.mark.parametrize("layout", [0, 1])
@pytest.mark.parametrize("dead", [0, 1, 2])
def test_kv_with_migration_aware_head_plan(ctx, layout, dead):
    """Paged KV under a permuted head layout: config 1 (4 heads on 4 ranks), one rank dies, the migration-aware plan keeps
    more heads in place than the in-order one; a rank may now own a head interval disjoint from its old one, so a reload can
    land on a slot another rank still has to read (write-after-read phases across the copy and reload streams)."""
    from oracle import planning as OP
    cfg = get_config("1")
    world = H.build_kv_world(cfg, side=MigSide, layout=layout, failed=(dead,))
    st = world.steps[0]
    old = [tuple(x) for x in st.old["head"]]
    tb = [b for (_, b, _, _) in st.new["head"]] + [st.new["head"][-1][2]]
    tasks, new = OP.migration_aware_plan(old, len(st.new["head"]), tb)
    assert [tuple(t) for t in st.tasks["head"]] == [tuple(t) for t in tasks] and [tuple(x) for x in st.new["head"]] == new
    base = OP.plan_stats(OP.cmm_plan(old, len(new), tb)[0])
    assert OP.plan_stats(tasks)["transfer_units"] <= base["transfer_units"]
    plan = etp.etp_plan_create(etp.PLAN_MIGRATION_AWARE, old, len(new), tb)
    ev, evicted, rep, stats = run_kv(ctx, world, world.g.n_blocks, plan=plan)
    assert ev == evicted == []
    assert rep["d2d_bytes"] == stats["d2d_bytes"] and rep["h2d_bytes"] == stats["h2d_bytes"]


# ------------------------------------------------------------------------------------------------ migration-aware plan (parameters)
@pytest.mark.parametrize("slabs_mode", ["span", "full"])
def test_migration_aware_plan_reshard_and_linear(ctx, slabs_mode):
    """Reading M1: config 5a's second failure in miniature - 7 ranks of 200 units, rank 0 dies, 6 targets.
    The migration-aware plan permutes the owners (the new layout is not in rank order) and transfers fewer units than
    Algorithm 1's in-order owners; the reshard is bit-exact to the oracle applying the oracle's own migration-aware plan, and
    the column-parallel linear on the permuted layout still matches the unsharded reference."""
    from oracle import linear as OL
    from oracle import planning as OP
    K = 1032                                             # in-features; unit = one out-feature row
    Hn, ub = 1400, K * 2
    ranks = [0, 1, 2, 3, 4, 6, 7]
    old = [(r, 200 * i, 200 * (i + 1), 0 if r == 0 else 1) for i, r in enumerate(ranks)]
    tasks, new = OP.migration_aware_plan(old, 6)
    base = OP.plan_stats(OP.cmm_plan(old, 6)[0])
    st = OP.plan_stats(tasks)
    assert st["reload_units"] == base["reload_units"] == 200 and st["transfer_units"] < base["transfer_units"]
    assert [r for (r, _, _, _) in new] != sorted(r for (r, _, _, _) in new)
    plan = etp.etp_plan_create(etp.PLAN_MIGRATION_AWARE, old, 6)
    assert plan.tasks() == tasks and plan.new_layout() == new
    geom = {}
    for (r, b, e, a) in old:
        if not a:
            continue
        if slabs_mode == "full":
            geom[r] = (0, Hn)
        else:
            first, span = plan.slab_span(r)
            geom[r] = (first, span)
    from workloads.gen import as_u8, fill_normal16
    w = as_u8(fill_normal16(77, 1, 0, Hn * K, 0.02, torch.bfloat16)).copy()
    rng = np.random.default_rng(3)
    slabs = {}
    for (r, b, e, a) in old:
        if a:
            slab = np.full(geom[r][1] * ub, 0xFF, dtype=np.uint8)      # NaN patterns outside the shard
            OS.place_units(slab, *geom[r], ub, b, e, w)
            slabs[r] = slab
    expect, stats = OS.apply_params(tasks, slabs, geom, ub, w, 0)
    for (r, b, e, _) in new:
        assert np.array_equal(OS.read_units(expect[r], *geom[r], ub, b, e), w[b * ub:e * ub])
    bufs = {r: DevBuf(a) for r, a in slabs.items()}
    image = pinned(w)
    desc = etp.TensorDesc(Hn, ub, {r: (bufs[r].ptr, geom[r][1], geom[r][0]) for r in bufs}, 8, 0, image.data_ptr(), 0, Hn)
    s = Streams()
    rep = etp.etp_reshard_params(ctx, [desc], [plan], s.copy.cuda_stream, s.reload.cuda_stream)
    s.sync()
    assert rep["d2d_bytes"] == stats["d2d_bytes"] == st["transfer_units"] * ub and rep["h2d_bytes"] == 200 * ub
    for r, b in bufs.items():
        assert b.guards_intact()
        assert np.array_equal(b.payload(), expect[r]), f"rank {r}: slab differs from the oracle image"
    # S7 on the permuted layout
    T = 4
    x = as_u8(fill_normal16(77, 2, 0, T * K, 1.0, torch.bfloat16)).copy()
    xb, yb = DevBuf(x), DevBuf(np.full(T * Hn * 2, 0xEE, dtype=np.uint8))
    etp.etp_shard_linear(ctx, etp.COL_PARALLEL, "bf16", xb.ptr, T, K, Hn, desc, new, 1, yb.ptr)
    torch.cuda.synchronize()
    y = OL.decode16(yb.payload(), "bf16").reshape(T, Hn)
    ref = OL.linear_ref(OL.decode16(x, "bf16").reshape(T, K), OL.decode16(w, "bf16").reshape(Hn, K))
    assert np.isfinite(y).all() and OL.max_rel_err(y, ref) <= 5e-3


# ------------------------------------------------------------------------------------------------ interval copy (5b)
@pytest.mark.parametrize("n,hi", [(0, 1 << 20), (1, 1 << 20), (300, 4 << 20), (20000, 8 << 10),
                                  (40000, 8 << 10), (70000, 96 << 10)])    # >= 32768 intervals: device-side lowering, 1 and 2 chunks
@pytest.mark.parametrize("tma_min", [None, 16, 1 << 62])
def test_copy_intervals_bit_exact(ctx, n, hi, tma_min):
    """Config 5b recipe at a size the host reproduces in seconds: log-uniform sizes from 16 B, random 16-B aligned
    offsets, overlapping sources, disjoint destinations with random gaps (gaps must keep their old bytes).  From 32768
    intervals on the descriptors are built on the device (etp_lower_dev.cu); tma_min routes the same plan through the bulk
    queue only, the vector queue only (linear + small segments), or both."""
    src_arena = 64 << 20
    if n:
        so, do, sz, dst_arena = microbench_intervals(n, 16, hi, 1234 + n, src_arena, max_total=(1 << 30) if n > 30000 else (256 << 20))
    else:
        so = do = sz = np.zeros(0, dtype=np.int64)
        dst_arena = 1024
    rng = np.random.default_rng(5)
    src = rng.integers(0, 256, src_arena, dtype=np.uint8)
    dst0 = rng.integers(0, 256, dst_arena, dtype=np.uint8)
    expect = dst0.copy()
    for a, b, m in zip(so, do, sz):
        expect[b:b + m] = src[a:a + m]
    S, D = DevBuf(src), DevBuf(dst0)
    default = ctx.get_option(etp.OPT_TMA_MIN_BYTES)
    stream = torch.cuda.Stream()
    try:
        if tma_min is not None:
            ctx.set_option(etp.OPT_TMA_MIN_BYTES, tma_min)
        rep = etp.etp_copy_intervals(ctx, so + S.ptr, do + D.ptr, sz, stream.cuda_stream)
    finally:
        ctx.set_option(etp.OPT_TMA_MIN_BYTES, default)
    stream.synchronize()
    assert D.guards_intact() and S.guards_intact()
    assert D.payload().tobytes() == expect.tobytes()
    assert rep["d2d_bytes"] == int(sz.sum())
    assert S.payload().tobytes() == src.tobytes()


@pytest.mark.parametrize("size,n", [(16, 5000), (256, 4099), (4096, 777), (32768, 65)])
@pytest.mark.parametrize("staged", [1, 0])
def test_copy_intervals_small_batches(ctx, size, n, staged):
    """The descriptor-bound corner of config 5b: every interval the same small size, so every vector work item is a
    batch of up to 128 intervals (or 32 KiB): staged through the idle ring with per-lane bulk copies (ETP_OPT_SMALL_STAGED, the
    default when a launch has no bulk intervals) or walked with the shuffle search; ragged last batch, last round and last word."""
    ctx.set_option(etp.OPT_SMALL_STAGED, staged)
    try:
        _small_batches(ctx, size, n)
    finally:
        ctx.set_option(etp.OPT_SMALL_STAGED, 1)


def _small_batches(ctx, size, n):
    rng = np.random.default_rng(size + n)
    src_arena = 8 << 20
    src = rng.integers(0, 256, src_arena, dtype=np.uint8)
    so = rng.integers(0, (src_arena - size) // 16, n).astype(np.int64) * 16
    gaps = rng.integers(0, 4, n).astype(np.int64) * 16
    do_sorted = np.cumsum(gaps + size) - size
    do = do_sorted[rng.permutation(n)]
    sz = np.full(n, size, dtype=np.int64)
    dst0 = rng.integers(0, 256, int(do_sorted[-1] + size + 64), dtype=np.uint8)
    expect = dst0.copy()
    for a, b in zip(so, do):
        expect[b:b + size] = src[a:a + size]
    S, D = DevBuf(src), DevBuf(dst0)
    stream = torch.cuda.Stream()
    rep = etp.etp_copy_intervals(ctx, so + S.ptr, do + D.ptr, sz, stream.cuda_stream)
    stream.synchronize()
    assert D.guards_intact() and S.guards_intact()
    assert D.payload().tobytes() == expect.tobytes()
    assert rep["d2d_bytes"] == n * size


def test_copy_intervals_errors(ctx):
    S, D = DevBuf(np.zeros(4096, np.uint8)), DevBuf(np.full(4096, 7, np.uint8))
    for so, do, sz, status in [(8, 0, 16, 2), (0, 0, 24, 2), (0, 0, -16, 1)]:
        with pytest.raises(etp.EtpError) as e:
            etp.etp_copy_intervals(ctx, np.array([S.ptr + so]), np.array([D.ptr + do]), np.array([sz]))
        assert e.value.status == status
    # the contract of include/etp.h: destinations mutually disjoint and disjoint from every source -> INVALID_ARG, nothing enqueued
    a = np.array
    cases = [
        (a([S.ptr, S.ptr + 512]), a([D.ptr, D.ptr + 48]), a([64, 64])),                  # two destinations overlap by 16 bytes
        (a([S.ptr, S.ptr + 512, S.ptr + 64]), a([D.ptr + 1024, D.ptr, D.ptr + 1040]), a([32, 64, 16])),   # ... out of order in the list
        (a([S.ptr, D.ptr + 96]), a([D.ptr + 64, D.ptr + 2048]), a([64, 64])),          # a destination overlaps another interval's source
        (a([D.ptr + 16]), a([D.ptr]), a([64])),                                           # ... its own source (a shifting copy)
    ]
    for sp, dp, sz in cases:
        with pytest.raises(etp.EtpError) as e:
            etp.etp_copy_intervals(ctx, sp, dp, sz)
        assert e.value.status == 1
    torch.cuda.synchronize()
    assert (D.payload() == 7).all() and D.guards_intact()
    # touching but not overlapping is fine; with validation off the caller is trusted
    etp.etp_copy_intervals(ctx, a([S.ptr, S.ptr + 64]), a([D.ptr, D.ptr + 64]), a([64, 64]))
    ctx.set_option(etp.OPT_VALIDATE_INTERVALS, 0)
    try:
        etp.etp_copy_intervals(ctx, a([S.ptr]), a([D.ptr + 128]), a([64]))
    finally:
        ctx.set_option(etp.OPT_VALIDATE_INTERVALS, 1)
    torch.cuda.synchronize()
    assert (D.payload()[:192] == 0).all() and (D.payload()[192:] == 7).all()


@pytest.mark.parametrize("n", [5000, 100_000])
def test_copy_intervals_validation_at_scale(ctx, n):
    """The disjointness check on many intervals (radix sort of (start, index) pairs, two threads from 65536): a valid random plan
    passes and is copied exactly; ONE planted overlap - a destination moved 16 bytes into its neighbour, or a source pointed into
    some destination - is reported with the right interval, and nothing is enqueued."""
    rng = np.random.default_rng(n)
    sz = rng.integers(1, 9, n).astype(np.int64) * 16
    do_sorted = np.cumsum(sz + rng.integers(0, 3, n) * 16) - sz
    perm = rng.permutation(n)
    do = do_sorted[perm]
    sz_p = sz[perm]
    src_arena = 1 << 20
    so = rng.integers(0, (src_arena - 256) // 16, n).astype(np.int64) * 16
    src = rng.integers(0, 256, src_arena, dtype=np.uint8)
    dst0 = np.full(int(do_sorted[-1] + sz[-1] + 64), 9, dtype=np.uint8)
    S, D = DevBuf(src), DevBuf(dst0)
    etp.etp_copy_intervals(ctx, so + S.ptr, do + D.ptr, sz_p)
    torch.cuda.synchronize()
    expect = dst0.copy()
    for a, b, m in zip(so, do, sz_p):
        expect[b:b + m] = src[a:a + m]
    assert D.payload().tobytes() == expect.tobytes() and D.guards_intact()
    D2 = DevBuf(dst0)
    k = int(np.argmax(do == do_sorted[n // 2]))                   # the interval whose destination is the (n/2)-th in address order
    bad_d = do.copy()
    bad_d[k] -= 16                                                # now overlaps the end of its predecessor (gap 0 or more: force it)
    pred = int(np.argmax(do == do_sorted[n // 2 - 1]))
    bad_d[k] = do[pred] + sz_p[pred] - 16
    with pytest.raises(etp.EtpError) as e:
        etp.etp_copy_intervals(ctx, so + S.ptr, bad_d + D2.ptr, sz_p)
    assert e.value.status == 1 and str(pred) in str(e.value) and str(k) in str(e.value)
    bad_s = so + S.ptr
    bad_s[7] = D2.ptr + do[k]                                     # a source inside another interval's destination
    with pytest.raises(etp.EtpError) as e:
        etp.etp_copy_intervals(ctx, bad_s, do + D2.ptr, sz_p)
    assert e.value.status == 1
    torch.cuda.synchronize()
    assert (D2.payload() == 9).all() and D2.guards_intact()


def test_back_to_back_calls_without_a_sync(ctx):
    """Two calls in flight on one ctx (the descriptor arena is double-buffered): a KV reshard whose zero-copy gather sits on
    the reload stream behind a large pinned-host copy, then - without any synchronisation - a multi-phase parameter reshard
    (tight slabs: several launches on the copy stream).  The work-queue heads of the first call's gather must not be reset
    or shared by the second call's launches (they live in the call's own arena slot)."""
    cfg = dataclasses.replace(MID, model=dataclasses.replace(MID.model, n_layers=2))
    kvw = H.build_kv_world(cfg, side=LibSide, layout=0, seq_lens=[300, 7, 1000], head_cap=4)
    st = kvw.steps[0]
    g = kvw.g
    new_table, evicted, pairs = OS.page_table_rewrite(kvw.table, kvw.seq_lens, kvw.last_use, g.block_size, g.n_blocks)
    snap = {r: p for r, p in kvw.pools.items() if r != st.dead}
    kexpect, _ = OS.apply_kv(st.tasks["head"], snap, kvw.anchors, g, kvw.host_backup, kvw.host_heads, kvw.host_head0, pairs)
    kbufs = {r: DevBuf(p) for r, p in snap.items()}
    img = pinned(kvw.host_backup)
    world = H.build_param_world(MID, side=LibSide, mode="tight", failed=(2,))
    pexpect, _ = H.oracle_reshard_params(world, 0)
    pbufs, pimages = upload_param_world(world)
    plans = make_plans(world.steps[0])
    klasses = sorted(plans)
    descs = tensor_descs(world, pbufs, pimages, world.steps[0], {k: i for i, k in enumerate(klasses)})
    s = Streams()
    big = torch.empty(1 << 30, dtype=torch.uint8).pin_memory()
    sink = torch.empty(1 << 30, dtype=torch.uint8, device="cuda")
    table = kvw.table.copy()
    with torch.cuda.stream(s.reload):
        sink.copy_(big, non_blocking=True)              # ~20 ms of DMA ahead of the gather on the reload stream
    ev, _ = etp.etp_reshard_kv(ctx, n_layers=g.n_layers, n_blocks=g.n_blocks, block_size=g.block_size, head_cap=g.head_cap,
                               head_dim=g.head_dim, elem_bytes=g.elem_bytes, layout=g.layout, pools={r: b.ptr for r, b in kbufs.items()},
                               head_anchor=kvw.anchors, n_ranks=max(kvw.pools) + 1, table=table, seq_lens=kvw.seq_lens,
                               last_use=kvw.last_use, head_plan=make_plans(st)["head"], new_block_budget=g.n_blocks,
                               host_backup=img.data_ptr(), host_heads=kvw.host_heads, host_head0=kvw.host_head0,
                               copy_stream=s.copy.cuda_stream, reload_stream=s.reload.cuda_stream)
    rep = etp.etp_reshard_params(ctx, descs, [plans[k] for k in klasses], s.copy.cuda_stream, s.reload.cuda_stream)
    assert rep["n_phases"] >= 2 and rep["n_kernel_launches"] >= 1
    s.sync()
    assert ev == evicted and np.array_equal(table, new_table)
    for r, b in kbufs.items():
        assert b.guards_intact() and b.payload().tobytes() == kexpect[r].tobytes(), f"pool of rank {r} differs from the oracle image"
    compare_params(world, pbufs, pexpect, {2})


def test_failed_kv_call_leaves_the_table_alone(ctx):
    """A call that fails in lowering (head_cap too small for the new shard; backup that does not cover the reloaded heads) must
    not have rewritten the caller's page table or reported evictions, and must not have moved a byte."""
    cfg = dataclasses.replace(MID, model=dataclasses.replace(MID.model, n_layers=1))
    world = H.build_kv_world(cfg, side=LibSide, layout=0, seq_lens=[300, 7, 1000], head_cap=4)
    st, g = world.steps[0], world.g
    live = int(((world.seq_lens + 15) // 16).sum())
    snap = {r: p for r, p in world.pools.items() if r != st.dead}
    bufs = {r: DevBuf(p) for r, p in snap.items()}
    img = pinned(world.host_backup)
    s = Streams()
    for kw, status in ((dict(head_cap=2), 3), (dict(host_head0=world.host_head0 + 1), 4), (dict(block_size=0), 1)):
        table = world.table.copy()
        args = dict(n_layers=g.n_layers, n_blocks=g.n_blocks, block_size=g.block_size, head_cap=g.head_cap, head_dim=g.head_dim,
                    elem_bytes=g.elem_bytes, layout=g.layout, pools={r: b.ptr for r, b in bufs.items()}, head_anchor=world.anchors,
                    n_ranks=max(world.pools) + 1, table=table, seq_lens=world.seq_lens, last_use=world.last_use,
                    head_plan=make_plans(st)["head"], new_block_budget=live - 10, host_backup=img.data_ptr(),
                    host_heads=world.host_heads, host_head0=world.host_head0, copy_stream=s.copy.cuda_stream,
                    reload_stream=s.reload.cuda_stream)
        args.update(kw)
        with pytest.raises(etp.EtpError) as e:
            etp.etp_reshard_kv(ctx, **args)
        assert e.value.status == status, (kw, e.value)
        assert np.array_equal(table, world.table), f"{kw}: the failed call rewrote the page table"
    s.sync()
    for r, b in bufs.items():
        assert b.guards_intact() and b.payload().tobytes() == snap[r].tobytes()
