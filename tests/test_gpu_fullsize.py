"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (ModelState, two streams, single-phase
slabs, device-resident and pinned reload sources).

Two kinds of check per config:
  * the plain definition over the WHOLE state, evaluated on the device from the seeded generator (every byte of the
    unsharded tensors / KV reference is a pure function of its index, workloads/gen.py): every unit of every new shard ==
    the unsharded tensor's unit; every slot outside the new shards still holds what it held before; every (layer, K|V, live
    block, token, new head) fragment == the reference fragment.  These hold at any size.
  * the CPU oracle (oracle/state.py, element by element) on sampled layers: their slabs / pool planes are copied to the
    host before the reshard, the oracle applies the plan, and the result is compared byte for byte with what the GPU left.
"""
import numpy as np
import pytest
import torch

import paper_2511_11617_b200 as etp
from oracle import planning as OP
from oracle import state as OS
from paper_2511_11617_b200.state import ModelState
from workloads import get_config
from workloads.configs import scaled
from workloads.gen import fill_bytes, fill_kv_pool, fill_normal16

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    c = etp.Context(0)
    yield c
    c.close()


_ORACLE_PLANS = {}


def oracle_tasks(state, st, klass, total_units):
    """The ORACLE's plan of one class for this step: Algorithm 1 on the policy's bounds, or - when the state was planned
    migration-aware (reading M1) - the oracle's own exhaustive search (cached: 5040 owner orders x the wide-shard placements)."""
    old = tuple(tuple(s) for s in st.old[klass])
    M = len(st.new[klass])
    if state.plan_mode == etp.PLAN_MIGRATION_AWARE:
        key = (old, M)
        if key not in _ORACLE_PLANS:
            _ORACLE_PLANS[key] = OP.migration_aware_plan(list(old), M)
        tasks, new = _ORACLE_PLANS[key]
        assert [tuple(x) for x in st.new[klass]] == new, "the library's migration-aware layout differs from the oracle's"
        return tasks
    return OP.cmm_plan(list(old), M, OP.partition(total_units, M, state.cfg.scenario.new_policy))[0]


def slot_runs(begin, end, anchor, cap):
    """[(first unit, n units, first slot)] of units [begin, end) in a slot-addressed slab (test-side restatement of L3)."""
    out, u = [], begin
    while u < end:
        s = (u - anchor) % cap
        n = min(end - u, cap - s)
        out.append((u, n, s))
        u += n
    return out


def holdings(state, klass, upto_step):
    """rank -> list of (unit interval) the rank's slab holds VALID data for after steps [0, upto_step) — new shard — plus
    the stale units it held before and that were not overwritten.  Returned as {rank: {slot: unit}} would be O(units); we
    return interval lists instead: (valid [(b, e)], stale candidates in order of age [(b, e), ...])."""
    first = state.initial_layouts()[klass]
    hist = {r: [(s, e)] for (r, s, e, _) in first}
    for i in range(upto_step):
        for (r, s, e, _) in state.steps[i].new[klass]:
            hist[r].append((s, e))
    return hist


def expected_slab(state, sp, r, upto_step, garbage):
    """Device tensor: what rank r's slab of tensor sp must hold after steps [0, upto_step): start from the initial image
    (garbage or zeros + the initial shard), then overlay each later shard the rank owned, oldest first; a newer unit
    landing on a slot replaces the older one (the slot rule makes the address a function of the unit alone)."""
    anchor, cap = state.geom[sp.klass][r]
    eb = state.cfg.model.elem_bytes
    epu = sp.unit_bytes // eb
    nb = cap * sp.unit_bytes
    if garbage:
        exp = fill_bytes(state.seed, 10_000 + sp.stream * 16 + r, 0, (nb + 7) // 8 * 8, device=state.device)[:nb].clone()
    else:
        exp = torch.zeros(nb, dtype=torch.uint8, device=state.device)
    for (b, e) in holdings(state, sp.klass, upto_step)[r]:
        for (u, n, s) in slot_runs(b, e, anchor, cap):
            fill_normal16(state.seed, sp.stream, u * epu, n * epu, state.cfg.model.init_std, state.dt,
                          out=exp[s * sp.unit_bytes:(s + n) * sp.unit_bytes].view(state.dt))
    return exp


def check_params_whole_state(state, upto_step, garbage):
    dead = {st.dead for st in state.steps[:upto_step]}
    n = 0
    for sp in state.specs:
        for r, slab in state.slabs[sp.name].items():
            if r in dead:
                continue
            exp = expected_slab(state, sp, r, upto_step, garbage)
            if not torch.equal(slab, exp):
                bad = torch.nonzero(slab != exp)[:4].flatten().tolist()
                raise AssertionError(f"{sp.name} rank {r}: slab differs from the plain definition at bytes {bad}")
            n += slab.numel()
            del exp
    return n


def snapshot_layer_params(state, layer):
    """Host copies of every slab of `layer`'s tensors (pre-reshard image for the oracle)."""
    return {sp.name: {r: t.cpu().numpy().copy() for r, t in state.slabs[sp.name].items()} for sp in state.specs if sp.layer == layer}


def oracle_layer_params(state, step_idx, snap):
    """oracle/state.apply_params on the snapshot of one layer; returns {name: {rank: expected slab bytes}}."""
    st = state.steps[step_idx]
    out = {}
    for sp in state.specs:
        if sp.name not in snap:
            continue
        M = len(st.new[sp.klass])
        tasks = oracle_tasks(state, st, sp.klass, sp.total_units)
        lo, hi = state.reload_range[sp.klass]
        epu = sp.unit_bytes // state.cfg.model.elem_bytes
        img = None
        if hi > lo:
            img = fill_normal16(state.seed, sp.stream, lo * epu, (hi - lo) * epu, state.cfg.model.init_std, state.dt,
                                device=state.device).view(torch.uint8).cpu().numpy()
        alive = {r: a for r, a in snap[sp.name].items() if r != st.dead}
        exp, _ = OS.apply_params(tasks, alive, state.geom[sp.klass], sp.unit_bytes, img, lo)
        out[sp.name] = exp
    return out


def compare_layer_params(state, expect):
    for name, per_rank in expect.items():
        for r, e in per_rank.items():
            got = state.slabs[name][r].cpu().numpy()
            assert np.array_equal(got, e), f"{name} rank {r}: GPU slab != oracle image"


# ------------------------------------------------------------------------------------------------ paged KV
def kv_dims(state):
    m, kv = state.cfg.model, state.kv
    return m.n_layers * 2, kv["n_blocks"], state.cfg.kv.block_size, kv["head_cap"], kv["frag"]


def live_block_ids(state):
    t = state.kv["table"]
    return torch.from_numpy(np.unique(t[t >= 0]).astype(np.int64)).to(state.device)


def expected_pool(state, r, upto_step, garbage):
    """What rank r's pool must hold after steps [0, upto_step) with an identity page table: the initial image (its old
    heads in EVERY block, as ModelState fills them), then, step by step, the heads of its new shard in the LIVE blocks only
    (free blocks are never copied, reading K6)."""
    planes, n_blocks, bs, cap, frag = kv_dims(state)
    m = state.cfg.model
    seed = state.seed + 500
    rows = planes * n_blocks * bs
    nb = rows * cap * frag
    first = {rr: (s, e) for (rr, s, e, _) in state.initial_layouts()["head"]}
    anchor = state.kv["anchors"][r]
    if garbage:
        exp = fill_bytes(seed, 100 + r, 0, (nb + 7) // 8 * 8, device=state.device)[:nb].clone()
    else:
        exp = torch.zeros(nb, dtype=torch.uint8, device=state.device)
    s, e = first[r]
    layout = state.kv["layout"]
    if e > s:
        fill_kv_pool(exp, rows, cap, m.head_dim, 0, s, e - s, m.n_kv_heads, seed, 1, state.dt, layout=layout, block_size=bs)
    live = live_block_ids(state)
    ev = exp.view(planes, n_blocks, bs, cap, frag) if layout == 0 else exp.view(planes, n_blocks, cap, bs, frag)
    held = set(range(s, e))
    for i in range(upto_step):
        new = [(b, e2) for (rr, b, e2, _) in state.steps[i].new["head"] if rr == r]
        for (b, e2) in new:
            for h in range(b, e2):
                if h in held:
                    continue                                   # KEEP: never touched
                one = torch.empty(rows * frag, dtype=torch.uint8, device=state.device)
                fill_kv_pool(one, rows, 1, m.head_dim, 0, h, 1, m.n_kv_heads, seed, 1, state.dt)
                ov = one.view(planes, n_blocks, bs, frag)
                if layout == 0:
                    ev[:, live, :, (h - anchor) % cap, :] = ov[:, live]
                else:
                    ev[:, live, (h - anchor) % cap, :, :] = ov[:, live]
                del one, ov
            held = set(range(b, e2))
    return exp


def check_kv_whole_state(state, upto_step, garbage):
    dead = {st.dead for st in state.steps[:upto_step]}
    n = 0
    for r, pool in state.kv["pools"].items():
        if r in dead:
            continue
        exp = expected_pool(state, r, upto_step, garbage)
        if not torch.equal(pool, exp):
            bad = torch.nonzero(pool != exp)[:4].flatten().tolist()
            raise AssertionError(f"KV pool of rank {r} differs from the plain definition at bytes {bad}")
        n += pool.numel()
        del exp
    return n


def layer_slice(state, t, layer, heads):
    planes, n_blocks, bs, cap, frag = kv_dims(state)
    per_layer = 2 * n_blocks * bs * heads * frag
    return t[layer * per_layer:(layer + 1) * per_layer]


def snapshot_layer_kv(state, layer):
    cap = state.kv["head_cap"]
    return {r: layer_slice(state, p, layer, cap).cpu().numpy().copy() for r, p in state.kv["pools"].items()}


def oracle_layer_kv(state, step_idx, layer, snap, image, budget=None):
    st = state.steps[step_idx]
    m, kv = state.cfg.model, state.kv
    planes, n_blocks, bs, cap, frag = kv_dims(state)
    g1 = OS.KVGeom(1, n_blocks, bs, cap, m.head_dim, m.elem_bytes, kv["layout"])
    sc = state.cfg.scenario
    H = m.n_kv_heads
    tasks = oracle_tasks(state, st, "head", H)
    _, evicted, pairs = OS.page_table_rewrite(kv["table"], kv["seq_lens"], kv["last_use"], bs, n_blocks if budget is None else budget)
    assert budget is not None or not evicted
    per_kind, hh, ds = kv["backup"][step_idx]
    backup = layer_slice(state, per_kind[image], layer, hh).cpu().numpy() if hh > 0 else None
    alive = {r: a for r, a in snap.items() if r != st.dead and any(rr == r for (rr, _, _, _) in st.old["head"])}
    exp, stats = OS.apply_kv(tasks, alive, kv["anchors"], g1, backup, hh, ds, pairs)
    return exp, stats


def compare_layer_kv(state, layer, expect):
    cap = state.kv["head_cap"]
    for r, e in expect.items():
        got = layer_slice(state, state.kv["pools"][r], layer, cap).cpu().numpy()
        assert np.array_equal(got, e), f"KV pool of rank {r}, layer {layer}: GPU planes != oracle image"


# ------------------------------------------------------------------------------------------------ S7 on sampled outputs
def check_linear_sampled(ctx, state, step_idx, layer, tokens, n_tok=12, n_feat=24):
    """etp_shard_linear on the resharded slabs of one layer at `tokens` tokens; n_tok x n_feat sampled outputs per linear are
    recomputed in fp64 from the generator's values of the UNSHARDED weight rows (oracle/linear.py) - max rel err <= 5e-3."""
    from oracle import linear as OL
    from workloads.gen import as_u8, normal16_at
    dtn = state.cfg.model.dtype
    rng = np.random.default_rng(1234 + layer)
    worst = 0.0
    for sp in state.specs:
        if sp.layer != layer:
            continue
        lin = state.linear(sp.name, step_idx, after=True)
        K, N = lin.K, lin.N
        x = fill_normal16(state.seed, 9100 + sp.stream, 0, tokens * K, 1.0, state.dt, device=state.device)
        y = torch.full((tokens * N,), float("nan"), dtype=state.dt, device=state.device)
        lin.run(ctx, x.data_ptr(), tokens, y.data_ptr(), 0)
        torch.cuda.synchronize()
        assert torch.isfinite(y.float()).all(), f"{sp.name}: unwritten or poisoned outputs"
        ts = np.unique(np.concatenate([[0, tokens - 1], rng.integers(0, tokens, n_tok)]))
        ns = np.unique(np.concatenate([[0, N - 1], rng.integers(0, N, n_feat)]))
        xs = OL.decode16(as_u8(x.view(tokens, K)[torch.from_numpy(ts).to(state.device)]), dtn).reshape(len(ts), K)
        k = torch.arange(K, dtype=torch.int64, device=state.device)
        nn = torch.from_numpy(ns).to(state.device)
        idx = (k[None, :] * N + nn[:, None]) if sp.transposed else (nn[:, None] * K + k[None, :])     # element index in the unsharded tensor
        ws = OL.decode16(as_u8(normal16_at(idx, state.seed, sp.stream, state.cfg.model.init_std, state.dt)), dtn).reshape(len(ns), K)
        ref = OL.linear_ref(xs, ws)
        got = OL.decode16(as_u8(y.view(tokens, N)[torch.from_numpy(ts).to(state.device)][:, nn]), dtn).reshape(len(ts), len(ns))
        err = OL.max_rel_err(got, ref)
        assert err <= 5e-3, f"{sp.name} T={tokens}: max relative error {err:.3e} on sampled outputs"
        worst = max(worst, err)
    return worst


def check_moe_layer(ctx, state, step_idx, layer, tokens=16):
    """Reading G5 at full size (config 4): one MoE layer on the resharded expert slabs, per-expert etp_shard_linear calls on
    the routed tokens (tests/moe_util.py), against the oracle's fp64 MoE layer on the generator's UNSHARDED expert matrices."""
    from oracle import linear as OL
    from tests import moe_util as MU
    from workloads.gen import as_u8
    m = state.cfg.model
    E, F, Hd, dtn = m.n_experts, m.expert_ffn, m.hidden, m.dtype
    names = {"gate": f"l{layer}.exp_gate", "up": f"l{layer}.exp_up", "down_t": f"l{layer}.exp_down_t"}
    spec = {k: next(s for s in state.specs if s.name == n) for k, n in names.items()}
    new = state.steps[step_idx].new["expert"]
    x = fill_normal16(state.seed, 9300 + layer, 0, tokens * Hd, 1.0, state.dt, device=state.device).view(tokens, Hd)
    logits = fill_normal16(state.seed, 9400 + layer, 0, tokens * E, 1.0, state.dt, device=state.device).view(tokens, E)

    def locate(kind, e):
        r = next(rr for (rr, b, en, _) in new if b <= e < en)
        anchor, cap = state.geom["expert"][r]
        return state.slabs[names[kind]][r].data_ptr(), anchor, cap, spec[kind].unit_bytes

    y, order, wts, _ = MU.moe_layer_per_expert(ctx, dtn, x, logits, m.top_k, F, locate)

    class Unsharded:
        """expert -> fp64 [F][Hd] straight from the position-addressable generator (never from a slab)."""
        def __init__(self, sp):
            self.sp = sp
        def __getitem__(self, e):
            w = fill_normal16(state.seed, self.sp.stream, e * F * Hd, F * Hd, m.init_std, state.dt, device=state.device)
            return OL.decode16(as_u8(w), dtn).reshape(F, Hd)

    err = MU.check_against_oracle(y, order, wts, OL.decode16(as_u8(x), dtn).reshape(tokens, Hd),
                                  OL.decode16(as_u8(logits), dtn).reshape(tokens, E), Unsharded(spec["gate"]),
                                  Unsharded(spec["up"]), Unsharded(spec["down_t"]), m.top_k)
    # the grouped kernel (etp_moe_linear) at a serving-size batch: 2048 tokens x top-8 = 16384 routed rows over 128 experts,
    # three launches; 8 sampled tokens against the oracle (a token's output depends on no other token)
    T2 = 2048
    x2 = fill_normal16(state.seed, 9500 + layer, 0, T2 * Hd, 1.0, state.dt, device=state.device).view(T2, Hd)
    lg2 = fill_normal16(state.seed, 9600 + layer, 0, T2 * E, 1.0, state.dt, device=state.device).view(T2, E)
    descs = {}
    for kind, sp in spec.items():
        slabs = {r: (state.slabs[sp.name][r].data_ptr(), state.geom["expert"][r][1], state.geom["expert"][r][0]) for (r, _, _, _) in new}
        descs[kind] = etp.TensorDesc(E, sp.unit_bytes, slabs, state.n_ranks, 0)
    y2, order2, wts2, counts, _ = MU.moe_layer_grouped(ctx, dtn, x2, lg2, m.top_k, F, descs, new)
    assert counts.sum() == T2 * m.top_k and torch.isfinite(y2).all()
    pick = np.unique(np.concatenate([[0, T2 - 1], np.random.default_rng(layer).integers(0, T2, 6)]))
    pk = torch.from_numpy(pick).to(state.device)
    MU.check_against_oracle(y2[pk], order2[pick], wts2[pick], OL.decode16(as_u8(x2[pk]), dtn).reshape(len(pick), Hd),
                            OL.decode16(as_u8(lg2[pk]), dtn).reshape(len(pick), E), Unsharded(spec["gate"]),
                            Unsharded(spec["up"]), Unsharded(spec["down_t"]), m.top_k)
    return err


# ------------------------------------------------------------------------------------------------ the tests
def run_full_config(ctx, key, image, linear_tokens=(), garbage=True, shrink=None, plan_mode=etp.PLAN_CMM, cap_mode="span"):
    cfg = get_config(key)
    if shrink:
        cfg = scaled(cfg, **shrink)
    state = ModelState(cfg, device="cuda:0", image=image, slack_garbage=garbage, plan_mode=plan_mode, cap_mode=cap_mode)
    phases = []
    cs, rs = torch.cuda.Stream(), torch.cuda.Stream()
    m = cfg.model
    for i, st in enumerate(state.steps):
        layer = (7 * i + 3) % m.n_layers
        sample_layers = [layer] + ([-1] if (m.vocab and i == 0) else [])
        snaps = {L: snapshot_layer_params(state, L) for L in sample_layers}
        ksnap = snapshot_layer_kv(state, layer)
        rep = state.reshard(ctx, i, image, cs.cuda_stream, rs.cuda_stream, replan=True)
        cs.synchronize()
        rs.synchronize()
        assert (rep["params"]["n_phases"] == 1 or cap_mode == "tight") and not rep["evicted"]
        phases.append(rep["params"]["n_phases"])
        # the oracle on the sampled layers
        for L in sample_layers:
            compare_layer_params(state, oracle_layer_params(state, i, snaps[L]))
        kexp, kstats = oracle_layer_kv(state, i, layer, ksnap, image)
        compare_layer_kv(state, layer, kexp)
        assert (rep["kv"]["d2d_bytes"], rep["kv"]["h2d_bytes"] + rep["kv"]["reload_dev_bytes"]) == \
               (kstats["d2d_bytes"] * m.n_layers, kstats["h2d_bytes"] * m.n_layers)
        # byte accounting of the parameters from the oracle's plan
        d2d = h2d = 0
        for sp in state.specs:
            M = len(st.new[sp.klass])
            tasks = oracle_tasks(state, st, sp.klass, sp.total_units)
            ps = OP.plan_stats(tasks)
            d2d += ps["transfer_units"] * sp.unit_bytes
            h2d += ps["reload_units"] * sp.unit_bytes
        assert rep["params"]["d2d_bytes"] == d2d and rep["params"]["h2d_bytes"] + rep["params"]["reload_dev_bytes"] == h2d
        # the plain definition over the whole state
        check_params_whole_state(state, i + 1, garbage)
        check_kv_whole_state(state, i + 1, garbage)
        for T in linear_tokens:
            check_linear_sampled(ctx, state, i, layer, T)
        if m.n_experts and linear_tokens:
            check_moe_layer(ctx, state, i, layer)
    state.phases_seen = phases
    return state


@pytest.mark.parametrize("image", ["device", "pinned"])
def test_config2_full_state(ctx, image):
    """BASELINE.json configs[1]: Qwen3-14B shape, 4 -> 3 after rank 1 fails, heads 3/3/2 - the bench workload."""
    run_full_config(ctx, "2", image, linear_tokens=(4, 4096) if image == "device" else ())


def test_config2b_full_state_floor_policy(ctx):
    """same workload under the paper's floor-boundary policy (heads 2/3/3): one KV head and its weights move D2D."""
    run_full_config(ctx, "2b", "pinned", linear_tokens=(4,))


def test_config3_full_state(ctx):
    """configs[2]: Llama-3-8B shape, 8 -> 7 after rank 5 fails, unequal old FFN widths."""
    run_full_config(ctx, "3", "pinned", linear_tokens=(4,))


def test_config3_full_state_migration_aware(ctx):
    """configs[2] under the migration-aware planner (reading M1): owners and wide-shard placement chosen by the library, checked
    against the oracle's exhaustive search; 2.55 GB instead of 5.04 GB move device-to-device; same whole-state and oracle checks."""
    state = run_full_config(ctx, "3", "pinned", linear_tokens=(4,), plan_mode=etp.PLAN_MIGRATION_AWARE)
    st = state.steps[0]
    base = sum(OP.plan_stats(OP.cmm_plan([tuple(s) for s in st.old[k]], len(st.new[k]),
                                         OP.partition(max(e for (_, _, e, _) in st.old[k]), len(st.new[k]), "floor"))[0])["transfer_units"]
               for k in ("head",))
    assert st.plans["head"].stats()["transfer_units"] < base


@pytest.mark.parametrize("budget_kind", ["relocate", "evict"])
def test_config2_kv_block_budget_shrink_full_size(ctx, budget_kind):
    """Reading K5 at full size: config 2's KV cache (8 layers of it; 64 x 2048 tokens = 8192 live blocks in a fragmented pool of
    10240) resharded 4 -> 3 with a block budget below the pool size.  "relocate": budget = 8192 live blocks, every live block
    with id >= 8192 moves to a free id below it (same-rank copies of kept heads, incoming heads written straight to the new id);
    "evict": budget = 6000 < live, the coldest sequences are evicted first.  Table, evicted list and byte counts
    against the oracle's rule; the planes of two layers byte for byte against the oracle."""
    cfg = scaled(get_config("2"), n_layers=8)
    state = ModelState(cfg, device="cuda:0", image="pinned", with_params=False, slack_garbage=True)
    kv, m = state.kv, cfg.model
    bs = cfg.kv.block_size
    live = int(((kv["seq_lens"].astype(np.int64) + bs - 1) // bs).sum())
    budget = live if budget_kind == "relocate" else 6000
    exp_table, exp_evicted, pairs = OS.page_table_rewrite(kv["table"], kv["seq_lens"], kv["last_use"], bs, budget)
    assert (len(exp_evicted) > 0) == (budget_kind == "evict")
    assert sum(1 for p in pairs if p[2] != p[3]) > 500                      # plenty of relocations in a fragmented pool
    layers = [1, 6]
    snaps = {L: snapshot_layer_kv(state, L) for L in layers}
    cs, rs = torch.cuda.Stream(), torch.cuda.Stream()
    rep = state.reshard(ctx, 0, "pinned", cs.cuda_stream, rs.cuda_stream, replan=True, block_budget=budget)
    cs.synchronize()
    rs.synchronize()
    assert sorted(rep["evicted"]) == sorted(exp_evicted)
    assert np.array_equal(rep["table"], exp_table)
    assert rep["table"][rep["table"] >= 0].max() < budget
    for L in layers:
        kexp, kstats = oracle_layer_kv(state, 0, L, snaps[L], "pinned", budget=budget)
        compare_layer_kv(state, L, kexp)
    assert (rep["kv"]["d2d_bytes"], rep["kv"]["h2d_bytes"]) == (kstats["d2d_bytes"] * m.n_layers, kstats["h2d_bytes"] * m.n_layers)


def test_config5a_tight_slabs_multi_phase_full_state(ctx):
    """Reading L5 at full size: config 5a (8 -> 7 -> 6 -> 5) with TIGHT slabs (cap = the widest shard a rank ever holds): shards
    wrap around their slabs and a write may land on a slot another task still reads, so the plans lower to several
    write-after-read hazard phases (one kernel launch each, reloads gated by events).  Same whole-state, oracle and linear checks."""
    state = run_full_config(ctx, "5a", "pinned", linear_tokens=(4,), cap_mode="tight")
    assert max(state.phases_seen) >= 2, state.phases_seen


def test_config4_full_state_moe(ctx):
    """configs[3]: Qwen3-30B-A3B shape (24 layers), 4 -> 3, experts repartitioned unequally (42/43/43)."""
    run_full_config(ctx, "4", "pinned", linear_tokens=(4,))


def test_config5a_sequential_failures_full_state(ctx):
    """configs[4] (a): Llama-3-8B shape, 8 -> 7 -> 6 -> 5, each reshard planned from the previous layout."""
    run_full_config(ctx, "5a", "pinned", linear_tokens=(4,))


# ------------------------------------------------------------------------------------------------ config 5b at its own sizes
@pytest.mark.parametrize("n", [100_000, 1_000_000])
def test_config5b_copy_intervals_full_size_every_byte(ctx, n):
    """configs[4] (b) at the sizes bench.py --microbench times (recipe of workloads/gen.py::microbench_intervals, R-5b):
    10^5 intervals up to 2 MiB (21.7 GiB) and 10^6 intervals up to 128 KiB (19.5 GiB), random 16-byte aligned sources in a
    32-GiB arena, disjoint destinations in random order with random gaps.  EVERY destination byte is checked: the expected
    arena is built on the device from the plain definition - one `dst[b:b+m] = src[a:a+m]` per interval, nothing else - and
    compared whole, gaps and guard bands included (a gap keeps the seeded garbage it held)."""
    from workloads.configs import MICROBENCH_HI, MICROBENCH_LO
    from workloads.gen import SEED0, microbench_intervals
    dev = torch.device("cuda:0")
    src_arena = 32 << 30
    G = 4096
    so, do, sz, dst_arena = microbench_intervals(n, MICROBENCH_LO, MICROBENCH_HI[n], SEED0 + 5000 + n, src_arena)
    src = fill_bytes(SEED0 + 5000, 1, 0, src_arena, device=dev)
    nb = (dst_arena + 2 * G + 7) // 8 * 8
    got = fill_bytes(SEED0 + 5001, 2, 0, nb, device=dev)          # destination arena between two guard bands, all garbage
    exp = got.clone()
    torch.cuda.synchronize()
    st = torch.cuda.Stream()
    rep = etp.etp_copy_intervals(ctx, so + src.data_ptr(), do + got.data_ptr() + G, sz, st.cuda_stream)
    so_l, do_l, sz_l = so.tolist(), (do + G).tolist(), sz.tolist()
    for a, b, m in zip(so_l, do_l, sz_l):                         # the plain definition, interval by interval
        exp[b:b + m] = src[a:a + m]
    st.synchronize()
    torch.cuda.synchronize()
    assert rep["d2d_bytes"] == int(sz.sum()) and rep["n_phases"] == 1
    if not torch.equal(got, exp):
        bad = torch.nonzero(got != exp)[:4].flatten().tolist()
        raise AssertionError(f"n = {n}: destination arena differs from the plain definition at bytes {bad}")
    del got, exp, src
    torch.cuda.empty_cache()


def test_config2_kv_head_major_full_size(ctx):
    """Reading K1's second layout at config-2 size (8 layers of the KV cache): pool[r] = [layer][K|V][block][slot][token][dim],
    so a head of a block is one 4-KiB contiguous run instead of 16 strided 256-byte fragments.  Whole-state plain definition
    on the device, two layers against the oracle's element-by-element applier, pinned backup (zero-copy gather)."""
    cfg = scaled(get_config("2"), n_layers=8)
    state = ModelState(cfg, device="cuda:0", image="pinned", with_params=False, slack_garbage=True, kv_layout=etp.KV_HEAD_MAJOR)
    m = cfg.model
    layers = [0, 5]
    snaps = {L: snapshot_layer_kv(state, L) for L in layers}
    cs, rs = torch.cuda.Stream(), torch.cuda.Stream()
    rep = state.reshard(ctx, 0, "pinned", cs.cuda_stream, rs.cuda_stream, replan=True)
    cs.synchronize()
    rs.synchronize()
    assert not rep["evicted"]
    for L in layers:
        kexp, kstats = oracle_layer_kv(state, 0, L, snaps[L], "pinned")
        compare_layer_kv(state, L, kexp)
    assert (rep["kv"]["d2d_bytes"], rep["kv"]["h2d_bytes"]) == (kstats["d2d_bytes"] * m.n_layers, kstats["h2d_bytes"] * m.n_layers)
    check_kv_whole_state(state, 1, True)
