"""Parity of kernel (c) etp_shard_linear (tcgen05/TMEM/TMA) against the oracle's UNSHARDED fp64 linear reference.

north_star: "the shard-linear outputs must match an unsharded fp32 reference within max relative error 5e-3"; reading G1
(DESIGN.md): max|y - ref| / max|ref| over the whole output.  The weight is handed to the kernel exactly as a reshard leaves
it: slot-addressed slabs (wrapped shards included), unequal widths, slack slots full of NaN bit patterns so that a read
outside a shard poisons the output."""
import numpy as np
import pytest
import torch

import paper_2511_11617_b200 as etp
from oracle import linear as OL
from oracle import state as OS
from tests import harness as H
from tests.gpu_util import DevBuf, LibSide, Streams, make_plans
from workloads import get_config
from workloads.gen import as_u8, fill_normal16, torch_dtype

pytestmark = pytest.mark.gpu

TOL = 5e-3          # north_star
SEED = 25111617


@pytest.fixture(scope="module")
def ctx():
    c = etp.Context(0)
    yield c
    c.close()


def widths_to_layout(widths, ranks=None):
    ranks = list(range(len(widths))) if ranks is None else ranks
    out, b = [], 0
    for r, w in zip(ranks, widths):
        out.append((r, b, b + w, 1))
        b += w
    return out


def shard_into_slabs(w_u8, unit_bytes, layout, geom):
    """slabs[r]: cap*unit_bytes bytes of 0xFF (16-bit NaN patterns) with the rank's units placed by the slot rule."""
    slabs = {}
    for (r, b, e, alive) in layout:
        anchor, cap = geom[r]
        slab = np.full(cap * unit_bytes, 0xFF, dtype=np.uint8)
        OS.place_units(slab, anchor, cap, unit_bytes, b, e, w_u8)
        slabs[r] = slab
    return slabs


def run_linear(ctx, mode, dtype, x_u8, T, K, N, w_desc, layout, fpu, stream=0):
    xb = DevBuf(x_u8)
    yb = DevBuf(np.full(T * N * 2, 0xEE, dtype=np.uint8))
    etp.etp_shard_linear(ctx, mode, dtype, xb.ptr, T, K, N, w_desc, layout, fpu, yb.ptr, stream)
    torch.cuda.synchronize()
    assert xb.guards_intact() and yb.guards_intact()
    return yb.payload()


def reference(dtype, x_u8, w_u8, T, K, N, transposed):
    x = OL.decode16(x_u8, dtype).reshape(T, K)
    w = OL.decode16(w_u8, dtype)
    w = w.reshape(K, N).T if transposed else w.reshape(N, K)
    return OL.linear_ref(x, w)


def check(y_u8, ref, dtype, T, N):
    y = OL.decode16(y_u8, dtype).reshape(T, N)
    assert np.isfinite(y).all(), "non-finite output: the kernel read outside a shard or left outputs unwritten"
    err = OL.max_rel_err(y, ref)
    assert err <= TOL, f"max relative error {err:.3e} > {TOL}"
    # sharper, derived from the arithmetic: fp32 accumulation + ONE rounding to 16 bit.  bf16 keeps 8 significant bits
    # (spacing 2^-7 relative, so round-to-nearest errs by at most 2^-8), fp16 keeps 11 (at most 2^-11).
    half_ulp = 2.0 ** -8 if dtype == "bf16" else 2.0 ** -11
    assert err <= half_ulp + 1e-4, f"max relative error {err:.3e} exceeds one 16-bit rounding"
    return err


CASES = [
    # mode, dtype, T, in, out, fpu, widths (units), geometry mode
    ("col", "bf16", 4, 256, 512, 1, (171, 171, 170), "tight"),
    ("col", "fp16", 4, 256, 256, 32, (3, 3, 2), "wrap"),
    ("col", "bf16", 4, 200, 1000, 1, (333, 334, 333), "wrap"),             # K tail (200 = 3 chunks + 8), ragged m tiles
    ("row", "bf16", 4, 688, 256, 1, (229, 229, 230), "tight"),             # config-1 down_t: K runs with tails
    ("row", "fp16", 4, 256, 256, 64, (1, 1, 2), "wrap"),                   # config-1 wo_t
    ("row", "bf16", 4, 1000, 200, 1, (100, 500, 400), "wrap"),             # out not a multiple of 64 / 128
    ("col", "bf16", 33, 512, 640, 1, (200, 240, 200), "wrap"),             # BN = 64
    ("row", "bf16", 50, 520, 384, 1, (260, 260), "tight"),
    ("col", "bf16", 100, 1000, 777, 1, (111, 222, 333, 111), "wrap"),      # BN = 256, ragged token tile
    ("row", "fp16", 300, 1000, 776, 1, (111, 222, 333, 334), "wrap"),      # two token tiles
    ("col", "bf16", 4, 5120, 5120, 640, (3, 3, 2), "tight"),               # Qwen3-14B wq, 4 tokens: split-K path
    ("row", "bf16", 4, 5120, 5120, 640, (3, 3, 2), "tight"),               # Qwen3-14B wo_t
    ("col", "bf16", 512, 2048, 2304, 1, (768, 769, 767), "wrap"),          # several items per CTA (accumulator stages)
    ("row", "bf16", 512, 2307 + 5, 2048, 1, (770, 771, 771), "wrap"),
    ("col", "bf16", 1000, 1024, 3000, 1, (1000, 1001, 999), "wrap"),       # CTA pairs: odd m-tile counts per run, 4 token tiles
    ("row", "bf16", 700, 3000, 1000, 1, (1000, 1001, 999), "wrap"),        # CTA pairs: out = 3.9 pair tiles, ragged tokens
    ("row", "bf16", 2560, 1000, 2040, 1, (300, 400, 300), "wrap"),         # 8 x 10 = 80 pair items over 74 pairs: the 6 items of
                                                                           # the last round are cut into 8 K ranges each (tail split)
    ("col", "bf16", 2560, 1000, 2040, 1, (680, 680, 680), "tight"),        # same item count, column-parallel: no tail split (G3)
]


@pytest.mark.parametrize("mode,dtype,T,K,N,fpu,widths,gmode", [c for c in CASES if c[2] > 64])
def test_shard_linear_forced_tile_modes_at_large_T(ctx, mode, dtype, T, K, N, fpu, widths, gmode):
    """> 64 tokens: CTA pairs (cta_group::2) with 256- and 128-token tiles and the single-CTA 128 x 256 path, each forced."""
    for forced in (0, 256, 128):            # 1 (default) picks pairs or single tiles by rounds of the persistent grid
        ctx.set_option(etp.OPT_LINEAR_CTA_PAIR, forced)
        try:
            test_shard_linear_matches_unsharded_reference(ctx, mode, dtype, T, K, N, fpu, widths, gmode)
        finally:
            ctx.set_option(etp.OPT_LINEAR_CTA_PAIR, 1)


@pytest.mark.parametrize("mode,dtype,T,K,N,fpu,widths,gmode", CASES)
def test_shard_linear_matches_unsharded_reference(ctx, mode, dtype, T, K, N, fpu, widths, gmode):
    transposed = mode == "row"
    sharded = K if transposed else N
    units = sharded // fpu
    assert units * fpu == sharded and sum(widths) == units
    row_len = N if transposed else K
    unit_bytes = fpu * row_len * 2
    dt = torch_dtype(dtype)
    std = 0.02
    w_u8 = as_u8(fill_normal16(SEED, 700 + T, 0, K * N, std, dt)).copy()
    x_u8 = as_u8(fill_normal16(SEED, 701 + T, 0, T * K, 1.0, dt)).copy()
    layout = widths_to_layout(widths)
    geom = {}
    for (r, b, e, _) in layout:
        if gmode == "tight":
            geom[r] = (b, e - b)                         # anchor = first unit, cap = width: no wrap
        else:
            cap = (e - b) + 1 + r
            geom[r] = (b - (cap - (e - b) // 2) % cap, cap)   # the shard starts mid-slab and wraps
    slabs = shard_into_slabs(w_u8, unit_bytes, layout, geom)
    bufs = {r: DevBuf(a) for r, a in slabs.items()}
    desc = etp.TensorDesc(units, unit_bytes, {r: (bufs[r].ptr, geom[r][1], geom[r][0]) for r in bufs}, len(widths), 0)
    y_u8 = run_linear(ctx, etp.ROW_PARALLEL if transposed else etp.COL_PARALLEL, dtype, x_u8, T, K, N, desc, layout, fpu)
    ref = reference(dtype, x_u8, w_u8, T, K, N, transposed)
    check(y_u8, ref, dtype, T, N)
    assert all(b.guards_intact() for b in bufs.values())
    for r, b in bufs.items():
        assert np.array_equal(b.payload(), slabs[r]), "the weight slabs are read-only for the linear"


@pytest.mark.parametrize("T", [4, 40, 100, 700])
def test_shard_linear_multi_fuses_qkv(ctx, T):
    """etp_shard_linear_multi: q | k | v (one granularity class: 8 KV-head groups, 5 / 1 / 1 rows of 32 per group... here 160 /
    32 / 32 features per unit) over unequal shards 3/3/2 with wrapped slabs, ONE launch; every output against the unsharded
    reference, and - where the kernel takes no K split (> 64 tokens) - bitwise equal to three separate etp_shard_linear calls."""
    dt = torch_dtype("bf16")
    K, units = 520, 8
    fpus = (160, 32, 32)
    layout = widths_to_layout((3, 3, 2))
    x_u8 = as_u8(fill_normal16(SEED, 780 + T, 0, T * K, 1.0, dt)).copy()
    xb = DevBuf(x_u8)
    lins, ybufs, refs, keep = [], [], [], []
    for i, fpu in enumerate(fpus):
        N = units * fpu
        ub = fpu * K * 2
        w_u8 = as_u8(fill_normal16(SEED, 790 + i, 0, N * K, 0.02, dt)).copy()
        geom = {}
        for (r, b, e, _) in layout:
            cap = (e - b) + 1 + r + i
            geom[r] = (b - (cap - (e - b) // 2) % cap, cap)
        slabs = shard_into_slabs(w_u8, ub, layout, geom)
        bufs = {r: DevBuf(a) for r, a in slabs.items()}
        keep.append(bufs)
        desc = etp.TensorDesc(units, ub, {r: (bufs[r].ptr, geom[r][1], geom[r][0]) for r in bufs}, 3, 0)
        lins.append(etp.PreparedLinear(etp.COL_PARALLEL, "bf16", K, N, desc, layout, fpu))
        ybufs.append(DevBuf(np.full(T * N * 2, 0xEE, dtype=np.uint8)))
        refs.append(reference("bf16", x_u8, w_u8, T, K, N, False))
    multi = etp.PreparedMultiLinear(lins)
    multi.run(ctx, xb.ptr, T, [y.ptr for y in ybufs])
    torch.cuda.synchronize()
    for lin, yb, ref in zip(lins, ybufs, refs):
        assert yb.guards_intact()
        check(yb.payload(), ref, "bf16", T, lin.N)
    if T > 64:
        for lin, yb in zip(lins, ybufs):
            y1 = DevBuf(np.full(T * lin.N * 2, 0xEE, dtype=np.uint8))
            lin.run(ctx, xb.ptr, T, y1.ptr)
            torch.cuda.synchronize()
            assert np.array_equal(y1.payload(), yb.payload())
    with pytest.raises(etp.EtpError) as e:      # different granularity classes cannot be fused
        other = etp.PreparedLinear(etp.COL_PARALLEL, "bf16", K, 4 * 32, etp.TensorDesc(4, 32 * K * 2, {0: (keep[0][0].ptr, 4, 0)}, 3, 0),
                                   layout, 32)
        etp.PreparedMultiLinear([lins[0], other]).run(ctx, xb.ptr, T, [ybufs[0].ptr, ybufs[1].ptr])
    assert e.value.status == 1


def test_column_parallel_is_bitwise_independent_of_the_split(ctx):
    """Reading G3: the K order of a column-parallel output does not depend on how out-features are cut."""
    T, K, N = 4, 1024, 1536
    dt = torch_dtype("bf16")
    w_u8 = as_u8(fill_normal16(SEED, 720, 0, K * N, 0.02, dt)).copy()
    x_u8 = as_u8(fill_normal16(SEED, 721, 0, T * K, 1.0, dt)).copy()
    outs = []
    for widths in ((384, 384, 384, 384), (512, 512, 512), (1536,), (100, 1000, 436)):
        layout = widths_to_layout(widths)
        geom = {r: (b, e - b) for (r, b, e, _) in layout}
        slabs = shard_into_slabs(w_u8, K * 2, layout, geom)
        bufs = {r: DevBuf(a) for r, a in slabs.items()}
        desc = etp.TensorDesc(N, K * 2, {r: (bufs[r].ptr, geom[r][1], geom[r][0]) for r in bufs}, len(widths), 0)
        outs.append(run_linear(ctx, etp.COL_PARALLEL, "bf16", x_u8, T, K, N, desc, layout, 1))
    for o in outs[1:]:
        assert np.array_equal(o, outs[0])


def linear_checks_for_world(ctx, world, bufs, layouts_by_class, tokens, dead=None):
    """Every sharded linear of the world on `layouts_by_class` against the unsharded reference.  Returns {name: y bytes}."""
    cfg = world.cfg
    dtype = cfg.model.dtype
    dt = torch_dtype(dtype)
    outs = {}
    n_ranks = max(r for (r, _, _, _) in world.steps[0].old[world.specs[0].klass]) + 1
    for sp in world.specs:
        if sp.name in ("embed",):
            continue                                   # a lookup table, not a linear
        sharded = sp.total_units * sp.features_per_unit
        K, N = (sharded, sp.row_elems) if sp.transposed else (sp.row_elems, sharded)
        x_u8 = as_u8(fill_normal16(H.seed_for(cfg), 5000 + sp.stream, 0, tokens * K, 1.0, dt)).copy()
        # before the failure every rank still holds its shard (the plan input marks the failing rank alive = 0)
        layout = [(r, b, e, 1) for (r, b, e, a) in layouts_by_class[sp.klass] if (a or dead is None) and r != dead]
        slabs = {r: (bufs[sp.name][r].ptr, world.geom[sp.name][r][1], world.geom[sp.name][r][0]) for (r, _, _, _) in layout}
        desc = etp.TensorDesc(sp.total_units, sp.unit_bytes, slabs, n_ranks, 0)
        y = run_linear(ctx, etp.ROW_PARALLEL if sp.transposed else etp.COL_PARALLEL, dtype, x_u8, tokens, K, N, desc, layout,
                       sp.features_per_unit)
        ref = reference(dtype, x_u8, world.unsharded[sp.name], tokens, K, N, sp.transposed)
        check(y, ref, dtype, tokens, N)
        outs[sp.name] = y
    return outs


@pytest.mark.parametrize("mode", ["tight", "span"])
def test_config1_layer_outputs_survive_the_reshard(ctx, mode):
    """Config 1 (BASELINE.json configs[0]): 4 unequal ranks, rank 2 fails, reshard to 3, "shard-linear check on a batch of
    4 tokens": every linear computes the unsharded layer output before AND after the reshard; column-parallel bitwise equal."""
    from tests import test_gpu_reshard as TR
    cfg = get_config("1")
    world = H.build_param_world(cfg, side=LibSide, mode=mode)
    bufs, images = TR.upload_param_world(world)
    step = world.steps[0]
    before = linear_checks_for_world(ctx, world, bufs, step.old, cfg.tokens)
    TR.run_param_step(ctx, world, bufs, images, 0, Streams())
    after = linear_checks_for_world(ctx, world, bufs, step.new, cfg.tokens, dead=step.dead)
    for sp in world.specs:
        if sp.name in before and not sp.transposed:
            assert np.array_equal(before[sp.name], after[sp.name]), sp.name


def test_moe_layer_on_resharded_experts(ctx):
    """Reading G5 at a size the oracle finishes in seconds: 12 experts over 4 ranks (3/3/3/3), rank 1 fails, experts are
    repartitioned 4/4/4; router logits N(0,1), top-4.  Every routed expert's gate / up / down runs through etp_shard_linear on
    the bytes the reshard left in the slabs; the layer output matches the oracle's unsharded fp64 MoE layer within 5e-3."""
    import dataclasses
    from tests import moe_util as MU
    from tests import test_gpu_reshard as TR
    from workloads.configs import Config, KVShape, ModelShape, Scenario
    shape = ModelShape("tiny-moe", 1, 256, 8, 4, 32, n_experts=12, expert_ffn=128, top_k=4)
    cfg = Config(9, "moe-small", shape, KVShape(2, 64), Scenario(4, (1,)))
    world = H.build_param_world(cfg, side=LibSide, mode="tight")
    bufs, images = TR.upload_param_world(world)
    TR.run_param_step(ctx, world, bufs, images, 0, Streams())
    expect, _ = H.oracle_reshard_params(world, 0)
    TR.compare_params(world, bufs, expect, {1})
    new = world.steps[0].new["expert"]
    dt = torch_dtype(shape.dtype)
    T, E, F, Hd = 24, shape.n_experts, shape.expert_ffn, shape.hidden
    x = fill_normal16(SEED, 740, 0, T * Hd, 1.0, dt).view(T, Hd).cuda()
    logits = fill_normal16(SEED, 741, 0, T * E, 1.0, dt).view(T, E).cuda()
    names = {"gate": "l0.exp_gate", "up": "l0.exp_up", "down_t": "l0.exp_down_t"}

    def locate(kind, e):
        r = next(rr for (rr, b, en, _) in new if b <= e < en)
        anchor, cap = world.geom[names[kind]][r]
        return bufs[names[kind]][r].ptr, anchor, cap, F * Hd * 2

    y, order, wts, calls = MU.moe_layer_per_expert(ctx, shape.dtype, x, logits, shape.top_k, F, locate)
    assert calls == 3 * len(np.unique(order))
    mats = {k: OL.decode16(world.unsharded[n], shape.dtype).reshape(E, F, Hd) for k, n in names.items()}
    x64 = OL.decode16(as_u8(x.cpu()), shape.dtype).reshape(T, Hd)
    lg64 = OL.decode16(as_u8(logits.cpu()), shape.dtype).reshape(T, E)
    MU.check_against_oracle(y, order, wts, x64, lg64, mats["gate"], mats["up"], mats["down_t"], shape.top_k)
    # the grouped kernel (etp_moe_linear): one launch per projection over all experts, same oracle, and bitwise the same
    # 16-bit projections as the per-expert calls would give is NOT required - only the tolerance is
    n_ranks = 4
    descs = {k: etp.TensorDesc(E, F * Hd * 2, {r: (bufs[n][r].ptr, world.geom[n][r][1], world.geom[n][r][0]) for (r, _, _, _) in new},
                               n_ranks, 0) for k, n in names.items()}
    y2, order2, wts2, counts, (g, u, yp, tok, exp_of_row) = MU.moe_layer_grouped(ctx, shape.dtype, x, logits, shape.top_k, F, descs, new)
    assert counts.sum() == T * shape.top_k and np.array_equal(order2, order)
    MU.check_against_oracle(y2, order2, wts2, x64, lg64, mats["gate"], mats["up"], mats["down_t"], shape.top_k)
    # every grouped projection row by row against the unsharded expert matrix (reading G4: each linear on its own)
    gg = OL.decode16(as_u8(g.cpu()), shape.dtype).reshape(-1, F)
    tok_h, exp_h = tok.cpu().numpy(), exp_of_row.cpu().numpy()
    ref_g = np.stack([mats["gate"][e] @ x64[t] for t, e in zip(tok_h, exp_h)])
    assert np.isfinite(gg).all() and OL.max_rel_err(gg, ref_g) <= TOL
    assert all(b.guards_intact() for n in names.values() for b in bufs[n].values())


@pytest.mark.parametrize("T,E,F,Hd,top_k,widths,gmode", [
    (4, 8, 128, 256, 2, (3, 3, 2), "tight"),          # a few rows per expert: 16-row tiles, experts without rows
    (300, 6, 192, 320, 3, (2, 1, 3), "wrap"),         # F not a multiple of 128 (a tile runs into the next expert's rows), wrapped shards
    (1500, 5, 256, 136, 2, (5,), "tight"),            # > 256 rows per expert: several row tiles; K tail (136 = 2 chunks + 8)
    (900, 4, 384, 192, 2, (1, 2, 1), "wrap"),         # 3 feature tiles: the second CTA pair has one tile past the last feature
])
@pytest.mark.parametrize("moe_pair", [0, 1, 2])
def test_moe_linear_grouped_vs_reference(ctx, T, E, F, Hd, top_k, widths, gmode, moe_pair):
    """etp_moe_linear on synthetic expert tensors (NaN-filled slack slots): every row of the column-parallel (gate-like) and
    row-parallel (down-like) grouped outputs against the fp64 product with ITS expert's unsharded matrix.  moe_pair: single-CTA
    tiles only / the library's choice / CTA pairs (cta_group::2) forced even for a few rows."""
    ctx.set_option(etp.OPT_MOE_CTA_PAIR, moe_pair)
    try:
        _moe_linear_grouped(ctx, T, E, F, Hd, top_k, widths, gmode, "fp16" if (T + moe_pair) % 2 else "bf16")   # both dtypes over the grid
    finally:
        ctx.set_option(etp.OPT_MOE_CTA_PAIR, 1)


def _moe_linear_grouped(ctx, T, E, F, Hd, top_k, widths, gmode, dtype="bf16"):
    dt = torch_dtype(dtype)
    rng = np.random.default_rng(T + E)
    layout = widths_to_layout(widths)
    geom = {}
    for (r, b, e, _) in layout:
        if gmode == "tight":
            geom[r] = (b, e - b)
        else:
            cap = (e - b) + 1 + r
            geom[r] = (b - (cap - (e - b) // 2) % cap, cap)
    ub = F * Hd * 2
    assign = np.sort(rng.integers(0, E, T * top_k)) if T > 4 else np.array([1, 1, 1, 4, 4, 6, 6, 6])
    counts = np.bincount(assign, minlength=E)
    offs = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    R = int(offs[-1])
    for mode, (K, N) in ((etp.COL_PARALLEL, (Hd, F)), (etp.ROW_PARALLEL, (F, Hd))):
        w_u8 = as_u8(fill_normal16(SEED, 760 + mode, 0, E * F * Hd, 0.02, dt)).copy()
        x_u8 = as_u8(fill_normal16(SEED, 770 + mode, 0, R * K, 1.0, dt)).copy()
        slabs = shard_into_slabs(w_u8, ub, layout, geom)
        bufs = {r: DevBuf(a) for r, a in slabs.items()}
        desc = etp.TensorDesc(E, ub, {r: (bufs[r].ptr, geom[r][1], geom[r][0]) for r in bufs}, len(widths), 0)
        xb, yb = DevBuf(x_u8), DevBuf(np.full(R * N * 2, 0xEE, dtype=np.uint8))
        etp.etp_moe_linear(ctx, mode, dtype, xb.ptr, offs, K, N, desc, layout, yb.ptr)
        torch.cuda.synchronize()
        assert xb.guards_intact() and yb.guards_intact() and all(b.guards_intact() for b in bufs.values())
        x64 = OL.decode16(x_u8, dtype).reshape(R, K)
        w64 = OL.decode16(w_u8, dtype).reshape(E, F, Hd)        # col: [E][out=F][in=Hd]; row: [E][in=F][out=Hd]
        ref = np.stack([(w64[e] @ x64[r]) if mode == etp.COL_PARALLEL else (x64[r] @ w64[e]) for r, e in enumerate(assign)])
        check(yb.payload(), ref, dtype, R, N)


def test_shard_linear_argument_errors(ctx):
    T, K, N = 4, 64, 128
    w = DevBuf(np.zeros(N * K * 2, dtype=np.uint8))
    x = DevBuf(np.zeros(T * K * 2, dtype=np.uint8))
    y = DevBuf(np.zeros(T * N * 2, dtype=np.uint8))
    desc = etp.TensorDesc(N, K * 2, {0: (w.ptr, N, 0)}, 1, 0)
    ok = [(0, 0, N, 1)]
    etp.etp_shard_linear(ctx, etp.COL_PARALLEL, "bf16", x.ptr, T, K, N, desc, ok, 1, y.ptr)
    torch.cuda.synchronize()
    with pytest.raises(etp.EtpError) as e:   # layout with a gap
        etp.etp_shard_linear(ctx, etp.COL_PARALLEL, "bf16", x.ptr, T, K, N, desc, [(0, 0, N - 1, 1)], 1, y.ptr)
    assert e.value.status == 1
    with pytest.raises(etp.EtpError) as e:   # unit_bytes inconsistent with the shapes
        etp.etp_shard_linear(ctx, etp.COL_PARALLEL, "bf16", x.ptr, T, K + 8, N, desc, ok, 1, y.ptr)
    assert e.value.status == 1
    with pytest.raises(etp.EtpError) as e:   # misaligned x
        etp.etp_shard_linear(ctx, etp.COL_PARALLEL, "bf16", x.ptr + 2, T, K, N, desc, ok, 1, y.ptr)
    assert e.value.status == 2
    with pytest.raises(etp.EtpError) as e:   # shard wider than its slab
        d2 = etp.TensorDesc(N, K * 2, {0: (w.ptr, N - 1, 0)}, 1, 0)
        etp.etp_shard_linear(ctx, etp.COL_PARALLEL, "bf16", x.ptr, T, K, N, d2, ok, 1, y.ptr)
    assert e.value.status == 3


def test_moe_linear_argument_errors(ctx):
    E, F, Hd = 4, 64, 128
    w = DevBuf(np.zeros(E * F * Hd * 2, dtype=np.uint8))
    x = DevBuf(np.zeros(8 * Hd * 2, dtype=np.uint8))
    y = DevBuf(np.full(8 * F * 2, 0xEE, dtype=np.uint8))
    desc = etp.TensorDesc(E, F * Hd * 2, {0: (w.ptr, E, 0)}, 1, 0)
    lay = [(0, 0, E, 1)]
    etp.etp_moe_linear(ctx, etp.COL_PARALLEL, "bf16", x.ptr, [0, 3, 3, 8, 8], Hd, F, desc, lay, y.ptr)
    torch.cuda.synchronize()
    assert not y.payload().any()                        # zero weights: every routed row written, as zeros
    etp.etp_moe_linear(ctx, etp.COL_PARALLEL, "bf16", x.ptr, [0, 0, 0, 0, 0], Hd, F, desc, lay, y.ptr)   # no rows: a no-op
    for offs, status in (([1, 3, 3, 8, 8], 1), ([0, 3, 2, 8, 8], 1), ([0, 3, 8], 1)):
        with pytest.raises(etp.EtpError) as e:          # offsets must start at 0, not decrease, and cover every expert
            etp.etp_moe_linear(ctx, etp.COL_PARALLEL, "bf16", x.ptr, offs, Hd, F, desc, lay, y.ptr)
        assert e.value.status == status
    with pytest.raises(etp.EtpError) as e:              # unit_bytes inconsistent with the shapes
        etp.etp_moe_linear(ctx, etp.COL_PARALLEL, "bf16", x.ptr, [0, 3, 3, 8, 8], Hd + 8, F, desc, lay, y.ptr)
    assert e.value.status == 1
    with pytest.raises(etp.EtpError) as e:              # row-parallel experts need in_features % 64 == 0
        d2 = etp.TensorDesc(E, 72 * Hd * 2, {0: (w.ptr, E, 0)}, 1, 0)
        etp.etp_moe_linear(ctx, etp.ROW_PARALLEL, "bf16", x.ptr, [0, 3, 3, 8, 8], 72, Hd, d2, lay, y.ptr)
    assert e.value.status == 5
    with pytest.raises(etp.EtpError) as e:              # layout with a gap
        etp.etp_moe_linear(ctx, etp.COL_PARALLEL, "bf16", x.ptr, [0, 3, 3, 8, 8], Hd, F, desc, [(0, 0, E - 1, 1)], y.ptr)
    assert e.value.status == 1
    with pytest.raises(etp.EtpError) as e:              # misaligned x
        etp.etp_moe_linear(ctx, etp.COL_PARALLEL, "bf16", x.ptr + 2, [0, 3, 3, 8, 8], Hd, F, desc, lay, y.ptr)
    assert e.value.status == 2
    assert x.guards_intact() and y.guards_intact() and w.guards_intact()


def smoke_shard_linear(ctx):
    """Used by __graft_entry__.smoke(): config 1's layer on the resharded state, 4 tokens, against the oracle reference."""
    from tests import test_gpu_reshard as TR
    cfg = get_config("1")
    world = H.build_param_world(cfg, side=LibSide, mode="tight")
    bufs, images = TR.upload_param_world(world)
    TR.run_param_step(ctx, world, bufs, images, 0, Streams())
    outs = linear_checks_for_world(ctx, world, bufs, world.steps[0].new, cfg.tokens, dead=world.steps[0].dead)
    print(f"smoke shard_linear OK: {len(outs)} linears of config 1 on the resharded layout within {TOL} of the unsharded reference")
    # the other tcgen05 kernels, one small case each against the fp64 references: CTA pairs of kernel (c) (> 64 tokens, row-parallel with
    # ragged widths), the grouped MoE kernels (fused gate|up through CTA pairs, plain single-CTA tiles)
    test_shard_linear_matches_unsharded_reference(ctx, "row", "bf16", 300, 1000, 776, 1, (111, 222, 333, 334), "wrap")
    ctx.set_option(etp.OPT_MOE_CTA_PAIR, 2)
    try:
        _moe_gate_up_fused(ctx, (130, 64, 257, 5), 4, 192, 320, (1, 3))
    finally:
        ctx.set_option(etp.OPT_MOE_CTA_PAIR, 1)
    _moe_linear_grouped(ctx, 4, 8, 128, 256, 2, (3, 3, 2), "tight")
    print("smoke tcgen05 OK: CTA-pair shard linear at 300 tokens, fused MoE gate|up (CTA pairs), grouped MoE linear at a few rows per expert")


# ------------------------------------------------------------------------------------------------ prepared groups (etp_linear_prepare / etp_linear_run)
def _make_linear(mode, K, N, fpu, widths, seed_i, gmode="wrap", dtype="bf16"):
    """One sharded weight on the device (NaN-filled slack) -> (PreparedLinear, w bytes, DevBufs to keep alive)."""
    transposed = mode == "row"
    units = (K if transposed else N) // fpu
    assert sum(widths) == units
    row_len = N if transposed else K
    ub = fpu * row_len * 2
    dt = torch_dtype(dtype)
    w_u8 = as_u8(fill_normal16(SEED, 900 + seed_i, 0, K * N, 0.02, dt)).copy()
    layout = widths_to_layout(widths)
    geom = {}
    for (r, b, e, _) in layout:
        if gmode == "tight":
            geom[r] = (b, e - b)
        else:
            cap = (e - b) + 1 + r
            geom[r] = (b - (cap - (e - b) // 2) % cap, cap)
    slabs = shard_into_slabs(w_u8, ub, layout, geom)
    bufs = {r: DevBuf(a) for r, a in slabs.items()}
    desc = etp.TensorDesc(units, ub, {r: (bufs[r].ptr, geom[r][1], geom[r][0]) for r in bufs}, len(widths), 0)
    lin = etp.PreparedLinear(etp.ROW_PARALLEL if transposed else etp.COL_PARALLEL, dtype, K, N, desc, layout, fpu)
    return lin, w_u8, bufs


GROUP = [   # a layer in miniature: q | k | v share the attention class layout, o_t is row-parallel over it, gate | up | down_t over the FFN class
    ("col", 520, 1280, 160, (3, 3, 2)), ("col", 520, 256, 32, (3, 3, 2)), ("col", 520, 256, 32, (3, 3, 2)),
    ("row", 1280, 520, 160, (3, 3, 2)), ("col", 520, 1403, 1, (468, 468, 467)), ("col", 520, 1403, 1, (468, 468, 467)),
    ("row", 1403 + 5, 520, 1, (470, 469, 469)),
]


@pytest.mark.parametrize("T", [1, 4, 16, 17, 64, 100])
@pytest.mark.parametrize("pdl", [1, 0])
def test_linear_group_mixed_modes_one_launch(ctx, T, pdl):
    """etp_linear_prepare / etp_linear_run: seven independent linears of both modes, every one with its OWN x and y, in one
    persistent launch (<= 64 tokens; one launch per linear at 100): each output against the unsharded fp64 reference at one
    16-bit rounding, the load-balanced item table sane, slack slots (NaN) never read, guard bands intact."""
    lins, ws, keep, xs, ys, refs = [], [], [], [], [], []
    dt = torch_dtype("bf16")
    for i, (mode, K, N, fpu, widths) in enumerate(GROUP):
        lin, w_u8, bufs = _make_linear(mode, K, N, fpu, widths, i)
        x_u8 = as_u8(fill_normal16(SEED, 950 + 10 * i + T, 0, T * K, 1.0, dt)).copy()
        lins.append(lin), ws.append(w_u8), keep.append(bufs)
        xs.append(DevBuf(x_u8))
        ys.append(DevBuf(np.full(T * N * 2, 0xEE, dtype=np.uint8)))
        refs.append(reference("bf16", x_u8, w_u8, T, K, N, mode == "row"))
    ctx.set_option(etp.OPT_LINEAR_PDL, pdl)
    try:
        plan = etp.LinearPlan(ctx, lins)
        info = plan.info()
        assert info["n_linears"] == 7 and 1 <= info["n_ctas"] <= 2 * 148 and info["n_items"] >= 7    # up to two CTAs per SM
        assert info["max_cta_chunks"] * info["n_ctas"] >= info["total_chunks"] > 0
        st = torch.cuda.Stream()
        for _ in range(3):                       # back to back on one stream: launch i+1 overlaps the tail of launch i
            plan.run([x.ptr for x in xs], T, [y.ptr for y in ys], st.cuda_stream)
        st.synchronize()
    finally:
        ctx.set_option(etp.OPT_LINEAR_PDL, 1)
    for (mode, K, N, fpu, widths), x, y, ref in zip(GROUP, xs, ys, refs):
        assert x.guards_intact() and y.guards_intact()
        check(y.payload(), ref, "bf16", T, N)
    plan.close()


def test_linear_chain_under_programmatic_dependent_launch(ctx):
    """What griddepcontrol.wait is for: linear B reads the OUTPUT of linear A, both launched back to back on one stream with the
    programmatic-serialization attribute (B's prologue and weight ring start while A is still running).  B's result must be
    bitwise what it is when A is synchronised first - 30 chains in a row, every intermediate overwritten each time."""
    T, K, Nmid = 8, 2048, 4096
    dt = torch_dtype("bf16")
    a, wa, ka = _make_linear("col", K, Nmid, 1, (1366, 1365, 1365), 40, "tight")
    b, wb, kb = _make_linear("row", Nmid, K, 1, (1366, 1365, 1365), 41, "tight")
    pa, pb = etp.LinearPlan(ctx, [a]), etp.LinearPlan(ctx, [b])
    st = torch.cuda.Stream()
    xs = [torch.from_numpy(as_u8(fill_normal16(SEED, 990 + i, 0, T * K, 1.0, dt)).copy()).cuda() for i in range(30)]
    mid = torch.zeros(T * Nmid * 2, dtype=torch.uint8, device="cuda")
    outs = [torch.zeros(T * K * 2, dtype=torch.uint8, device="cuda") for _ in range(30)]
    torch.cuda.synchronize()
    for x, o in zip(xs, outs):                   # chained, no synchronisation anywhere
        pa.run(x.data_ptr(), T, [mid.data_ptr()], st.cuda_stream)
        pb.run(mid.data_ptr(), T, [o.data_ptr()], st.cuda_stream)
    st.synchronize()
    chained = [o.cpu().numpy().copy() for o in outs]
    for i, x in enumerate(xs):                   # the same with a synchronisation after every launch
        pa.run(x.data_ptr(), T, [mid.data_ptr()], st.cuda_stream)
        st.synchronize()
        m_u8 = mid.cpu().numpy().copy()
        pb.run(mid.data_ptr(), T, [outs[i].data_ptr()], st.cuda_stream)
        st.synchronize()
        assert np.array_equal(outs[i].cpu().numpy(), chained[i]), f"chain {i}: B ran ahead of A's output"
        if i == 0:
            check(m_u8, reference("bf16", xs[0].cpu().numpy(), wa, T, K, Nmid, False), "bf16", T, Nmid)
            check(chained[0], reference("bf16", m_u8, wb, T, Nmid, K, True), "bf16", T, K)
    pa.close(), pb.close()


def test_linear_plans_on_two_streams_do_not_share_a_workspace(ctx):
    """One ctx, two streams, the same split-K plan in flight on both (per-stream partial tiles and tickets): both results are
    bitwise those of the serial runs."""
    T, K, N = 4, 8192, 1024
    dt = torch_dtype("bf16")
    lin, w_u8, keep = _make_linear("col", K, N, 1, (342, 341, 341), 60, "tight")
    plan = etp.LinearPlan(ctx, [lin])
    assert plan.info()["n_splits"][0] > 1
    xs = [torch.from_numpy(as_u8(fill_normal16(SEED, 1100 + i, 0, T * K, 1.0, dt)).copy()).cuda() for i in range(2)]
    serial = []
    for x in xs:
        y = torch.zeros(T * N * 2, dtype=torch.uint8, device="cuda")
        plan.run(x.data_ptr(), T, [y.data_ptr()], 0)
        torch.cuda.synchronize()
        serial.append(y.cpu().numpy().copy())
    check(serial[0], reference("bf16", xs[0].cpu().numpy(), w_u8, T, K, N, False), "bf16", T, N)
    s = [torch.cuda.Stream(), torch.cuda.Stream()]
    ys = [[torch.zeros(T * N * 2, dtype=torch.uint8, device="cuda") for _ in range(20)] for _ in range(2)]
    torch.cuda.synchronize()
    for k in range(20):
        for i in range(2):
            plan.run(xs[i].data_ptr(), T, [ys[i][k].data_ptr()], s[i].cuda_stream)
    torch.cuda.synchronize()
    for i in range(2):
        for k in range(20):
            assert np.array_equal(ys[i][k].cpu().numpy(), serial[i]), f"stream {i}, run {k}"
    plan.close()


@pytest.mark.parametrize("mode,K,N", [("col", 2048, 1536), ("row", 2048, 1536)])
def test_linear_right_behind_a_slab_write_on_the_same_stream(ctx, mode, K, N):
    """The <= 64-token kernel prefetches its first ring of weight tiles before griddepcontrol.wait when it is launched with the
    programmatic-serialization attribute, and the previous kernel's writes are only guaranteed visible after that wait.  The
    library therefore sends the first linear launch behind one of its own slab writes on that stream in plain stream order
    (ETP_OPT_LINEAR_PDL in include/etp.h).  Here the whole weight is REWRITTEN in place by etp_copy_intervals and the linear is
    enqueued right behind it, no sync, eight times with fresh weights: every output must follow the weights of its round."""
    T = 4
    dt = torch_dtype("bf16")
    widths = (K // 4, K // 2, K // 4) if mode == "row" else (N // 4, N // 2, N // 4)
    lin, w_u8, bufs = _make_linear(mode, K, N, 1, widths, 80, "tight")
    plan = etp.LinearPlan(ctx, [lin])
    x = torch.from_numpy(as_u8(fill_normal16(SEED, 1300, 0, T * K, 1.0, dt)).copy()).cuda()
    stream = torch.cuda.Stream()
    layout = widths_to_layout(widths)
    ub = (N if mode == "row" else K) * 2
    rounds = []
    for i in range(8):
        w_i = as_u8(fill_normal16(SEED, 1310 + i, 0, K * N, 0.02, dt)).copy()
        staged = torch.from_numpy(w_i).cuda()
        y = torch.zeros(T * N * 2, dtype=torch.uint8, device="cuda")
        rounds.append((w_i, staged, y))
    torch.cuda.synchronize()
    for w_i, staged, y in rounds:
        src = np.array([staged.data_ptr() + b * ub for (r, b, e, _) in layout], dtype=np.int64)
        dst = np.array([bufs[r].ptr for (r, b, e, _) in layout], dtype=np.int64)
        sz = np.array([(e - b) * ub for (r, b, e, _) in layout], dtype=np.int64)
        etp.etp_copy_intervals(ctx, src, dst, sz, stream.cuda_stream)
        plan.run(x.data_ptr(), T, [y.data_ptr()], stream.cuda_stream)
    stream.synchronize()
    for i, (w_i, staged, y) in enumerate(rounds):
        check(y.cpu().numpy(), reference("bf16", x.cpu().numpy(), w_i, T, K, N, mode == "row"), "bf16", T, N)
    plan.close()


def test_linear_plan_may_be_freed_after_its_ctx():
    """etp_linear_free touches only the plan's own device table (the device id is kept in the plan), so freeing a plan after
    etp_ctx_destroy is safe; the wrapper no longer leaks such plans."""
    own = etp.Context(0)
    lin, w_u8, keep = _make_linear("col", 256, 512, 1, (171, 171, 170), 70, "tight")
    plan = etp.LinearPlan(own, [lin])
    x = torch.from_numpy(as_u8(fill_normal16(SEED, 1200, 0, 4 * 256, 1.0, torch_dtype("bf16"))).copy()).cuda()
    y = torch.zeros(4 * 512 * 2, dtype=torch.uint8, device="cuda")
    plan.run(x.data_ptr(), 4, [y.data_ptr()], 0)
    torch.cuda.synchronize()
    check(y.cpu().numpy(), reference("bf16", x.cpu().numpy(), w_u8, 4, 256, 512, False), "bf16", 4, 512)
    own.close()
    assert plan.handle
    plan.close()
    assert plan.handle is None
    free0 = torch.cuda.mem_get_info()[0]
    assert free0 > 0                       # the device is still usable


def test_linear_prepare_errors(ctx):
    lin, _, keep = _make_linear("col", 256, 512, 1, (171, 171, 170), 70, "tight")
    with pytest.raises(etp.EtpError) as e:
        etp.LinearPlan(ctx, [lin] * 9)
    assert e.value.status == 1
    bad = etp.PreparedLinear(etp.COL_PARALLEL, "bf16", 256, 512, etp.TensorDesc(512, 512, {r: (b.ptr, 171, 0) for r, b in keep.items()}, 3, 0),
                             [(0, 0, 100, 1), (1, 150, 512, 1)], 1)
    with pytest.raises(etp.EtpError) as e:
        etp.LinearPlan(ctx, [bad])
    assert e.value.status == 1                  # the layout does not tile the units
    plan = etp.LinearPlan(ctx, [lin])
    y = DevBuf(np.zeros(4 * 512 * 2, np.uint8))
    x = DevBuf(np.zeros(4 * 256 * 2, np.uint8))
    with pytest.raises(etp.EtpError) as e:
        plan.run([x.ptr + 2], 4, [y.ptr])
    assert e.value.status == 2
    plan.run([x.ptr], 0, [y.ptr])               # zero tokens: nothing to do
    plan.close()


# ------------------------------------------------------------------------------------------------ fused gate|up, EPLB replicas
def _moe_world(E, F, Hd, widths, slack, seed_i):
    """gate / up / down_t expert tensors of one layer sharded over len(widths) ranks with `slack` spare slots per rank (NaN-filled):
    returns (w bytes per kind, TensorDescs per kind, layout, geom, DevBufs per kind)."""
    dt = torch_dtype("bf16")
    layout = widths_to_layout(widths)
    geom = {r: (b, (e - b) + slack) for (r, b, e, _) in layout}
    ub = F * Hd * 2
    ws, descs, bufs = {}, {}, {}
    for i, kind in enumerate(("gate", "up", "down_t")):
        ws[kind] = as_u8(fill_normal16(SEED, 1200 + 10 * seed_i + i, 0, E * F * Hd, 0.02 if kind != "down_t" else 0.05, dt)).copy()
        slabs = shard_into_slabs(ws[kind], ub, layout, geom)
        bufs[kind] = {r: DevBuf(a) for r, a in slabs.items()}
        descs[kind] = etp.TensorDesc(E, ub, {r: (bufs[kind][r].ptr, geom[r][1], geom[r][0]) for r in bufs[kind]}, len(widths), 0)
    return ws, descs, layout, geom, bufs


@pytest.mark.parametrize("rows_per_expert,E,F,Hd,widths", [
    ((0, 3, 17, 0, 1, 40), 6, 128, 256, (2, 2, 2)),           # 16-row tiles, experts without rows
    ((130, 64, 257, 5), 4, 192, 320, (1, 3)),                 # F not a multiple of 128: tiles run into the next slot; 128-row tiles
    ((300, 900), 2, 256, 136, (2,)),                          # several row tiles per expert; K tail
    ((256, 257, 0, 64, 321), 5, 384, 192, (2, 3)),            # 3 feature tiles (odd: half a CTA pair is idle), rows around the 256 / 64 edges
])
@pytest.mark.parametrize("moe_pair", [0, 1, 2])
def test_moe_gate_up_fused_matches_fp64_swiglu(ctx, rows_per_expert, E, F, Hd, widths, moe_pair):
    """etp_moe_gate_up: h = silu(gate x) * (up x) in one launch (two TMEM accumulators, activation in the epilogue), every row
    against oracle.linear.swiglu_ref in fp64 - fp32 accumulation and ONE 16-bit rounding, so the error is at most one rounding
    (tighter than the three-launch layer, which rounds gate and up to 16 bit first).  moe_pair as in the test above."""
    ctx.set_option(etp.OPT_MOE_CTA_PAIR, moe_pair)
    try:
        _moe_gate_up_fused(ctx, rows_per_expert, E, F, Hd, widths)
    finally:
        ctx.set_option(etp.OPT_MOE_CTA_PAIR, 1)


def _moe_gate_up_fused(ctx, rows_per_expert, E, F, Hd, widths):
    ws, descs, layout, geom, bufs = _moe_world(E, F, Hd, widths, 1, E)
    offs = np.concatenate([[0], np.cumsum(rows_per_expert)]).astype(np.int64)
    R = int(offs[-1])
    dt = torch_dtype("bf16")
    x_u8 = as_u8(fill_normal16(SEED, 1300 + E, 0, R * Hd, 1.0, dt)).copy()
    xb, hb = DevBuf(x_u8), DevBuf(np.full(R * F * 2, 0xEE, dtype=np.uint8))
    etp.etp_moe_gate_up(ctx, "bf16", xb.ptr, Hd, F, descs["gate"], descs["up"], hb.ptr, row_offsets=offs, layout=layout)
    torch.cuda.synchronize()
    assert xb.guards_intact() and hb.guards_intact()
    x64 = OL.decode16(x_u8, "bf16").reshape(R, Hd)
    g64, u64 = (OL.decode16(ws[k], "bf16").reshape(E, F, Hd) for k in ("gate", "up"))
    ref = np.concatenate([OL.swiglu_ref(x64[offs[e]:offs[e + 1]], g64[e], u64[e]) for e in range(E)])
    check(hb.payload(), ref, "bf16", R, F)


@pytest.mark.parametrize("moe_pair", [1, 2])
def test_moe_layer_with_eplb_replicas_is_bitwise_the_unreplicated_layer(ctx, moe_pair):
    """moe_pair = 2: the same through the CTA-pair kernels (forced; a replica changes an expert's row tiles, not its results)."""
    ctx.set_option(etp.OPT_MOE_CTA_PAIR, moe_pair)
    try:
        _moe_layer_with_eplb_replicas(ctx)
    finally:
        ctx.set_option(etp.OPT_MOE_CTA_PAIR, 1)


def _moe_layer_with_eplb_replicas(ctx):
    """Reading E1 end to end: seeded Zipf loads -> etp_eplb_place (== oracle) -> etp_eplb_apply copies the hot experts into
    spare slots (slot choice == oracle.eplb.replica_slots; the replica's bytes are the expert's, nothing else changes) ->
    the layer through etp_moe_gate_up + etp_moe_linear_instances with every expert's rows split over its instances.  A row is
    computed by exactly one instance from identical weights, so the output must be BITWISE the unreplicated layer's, and it
    matches the oracle's fp64 MoE layer within 5e-3."""
    from oracle import eplb
    from tests import moe_util as MU
    E, F, Hd, top_k, T = 12, 128, 256, 2, 96
    widths = (4, 4, 4)
    ws, descs, layout, geom, bufs = _moe_world(E, F, Hd, widths, 2, 77)
    dt = torch_dtype("bf16")
    x = fill_normal16(SEED, 1400, 0, T * Hd, 1.0, dt).view(T, Hd).cuda()
    logits = fill_normal16(SEED, 1401, 0, T * E, 1.0, dt).view(T, E).cuda()
    logits[:, 1] += 3.0                                            # a hot expert on rank 0, a warm one on rank 2
    logits[:, 9] += 1.5
    order, wts = MU.route(logits, top_k)
    flat_e = order.reshape(-1)
    perm = torch.argsort(flat_e, stable=True)
    tok = perm // top_k
    counts = torch.bincount(flat_e, minlength=E).cpu().numpy()
    offs = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    R = int(offs[-1])
    home = [next(r for (r, b, e, _) in layout if b <= ex < e) for ex in range(E)]
    capacity, spare = [2, 3, 2], [2, 2, 2]                         # rank 1 got the smaller dense shard: more idle compute
    replicas = etp.etp_eplb_place([int(c) for c in counts], home, capacity, spare)
    o_rep, o_inst = eplb.place([int(c) for c in counts], home, capacity, spare)
    assert replicas == o_rep and len(replicas) >= 1
    before = {k: {r: b.payload().copy() for r, b in bufs[k].items()} for k in bufs}
    slots = etp.etp_eplb_apply(ctx, [descs["gate"], descs["up"], descs["down_t"]], layout, replicas)
    torch.cuda.synchronize()
    assert slots == eplb.replica_slots(layout, geom, replicas)
    ub = F * Hd * 2
    for k in bufs:                                                  # the replica slots hold the expert's bytes, everything else is untouched
        for r, b in bufs[k].items():
            exp = before[k][r].copy()
            for (ex, d), s in zip(replicas, slots):
                if d == r:
                    exp[s * ub:(s + 1) * ub] = ws[k][ex * ub:(ex + 1) * ub]
            assert b.guards_intact() and np.array_equal(b.payload(), exp), f"{k} rank {r}"
    with pytest.raises(etp.EtpError) as err:                        # the same (expert, rank) twice: refused, nothing enqueued
        etp.etp_eplb_apply(ctx, [descs["gate"], descs["up"], descs["down_t"]], layout, list(replicas) + [replicas[0]])
    assert err.value.status == 1 and "twice" in str(err.value)
    # instances: home first, then replicas in creation order; rows split evenly (oracle.eplb.split_rows)
    slot_of = {(ex, d): s for (ex, d), s in zip(replicas, slots)}
    inst = []
    for ex in range(E):
        ranks = o_inst[ex]
        for (b, e), r in zip(eplb.split_rows(int(counts[ex]), len(ranks)), ranks):
            s = slot_of.get((ex, r), (ex - geom[r][0]) % geom[r][1] if r == home[ex] else None)
            inst.append((ex, r, s, int(offs[ex]) + b, int(offs[ex]) + e))
    assert max(len(r) for r in o_inst) >= 2
    xp = x[tok].contiguous()

    def layer(use_instances):
        h = torch.full((R, F), float("nan"), dtype=dt, device="cuda")
        yp = torch.full((R, Hd), float("nan"), dtype=dt, device="cuda")
        if use_instances:
            etp.etp_moe_gate_up(ctx, "bf16", xp.data_ptr(), Hd, F, descs["gate"], descs["up"], h.data_ptr(), instances=inst, n_rows=R)
            etp.etp_moe_linear_instances(ctx, etp.ROW_PARALLEL, "bf16", h.data_ptr(), inst, R, E, F, Hd, descs["down_t"], yp.data_ptr())
        else:
            etp.etp_moe_gate_up(ctx, "bf16", xp.data_ptr(), Hd, F, descs["gate"], descs["up"], h.data_ptr(), row_offsets=offs, layout=layout)
            etp.etp_moe_linear(ctx, etp.ROW_PARALLEL, "bf16", h.data_ptr(), offs, F, Hd, descs["down_t"], layout, yp.data_ptr())
        torch.cuda.synchronize()
        return h, yp

    h0, y0 = layer(False)
    h1, y1 = layer(True)
    assert torch.equal(h0.view(torch.int16), h1.view(torch.int16)) and torch.equal(y0.view(torch.int16), y1.view(torch.int16))
    w_flat = wts.reshape(-1)[perm].float()
    y = torch.zeros(T, Hd, dtype=torch.float32, device="cuda")
    y.index_add_(0, tok, w_flat[:, None] * y1.float())
    mats = {k: OL.decode16(ws[k], "bf16").reshape(E, F, Hd) for k in ws}
    MU.check_against_oracle(y, order.cpu().numpy(), wts.cpu().numpy(), OL.decode16(as_u8(x.cpu()), "bf16").reshape(T, Hd),
                            OL.decode16(as_u8(logits.cpu()), "bf16").reshape(T, E), mats["gate"], mats["up"], mats["down_t"], top_k)
    with pytest.raises(etp.EtpError) as e:                          # two instances may not share a row
        etp.etp_moe_linear_instances(ctx, etp.ROW_PARALLEL, "bf16", h1.data_ptr(), [(0, 0, 0, 0, 5), (1, 0, 1, 4, 8)], R, E, F, Hd,
                                     descs["down_t"], y1.data_ptr())
    assert e.value.status == 1
