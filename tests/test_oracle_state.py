"""Pins for the oracle's plan application (parameters, page table, paged KV) and the linear reference:
hand-worked golden images, the plain definitions ("new shard == slice of the unsharded tensor",
"KV_ref readable at its new place") checked through numpy N-d indexing rather than the oracle's own
offset arithmetic, and the textbook triple loop."""
import numpy as np
import pytest

from oracle import linear as OL
from oracle import planning as OP
from oracle import state as OS
from tests import harness as H
from workloads import get_config


# ------------------------------------------------------------------------------------------ golden slab
def load_slab_golden(golden_dir):
    g = {"geom": {}, "before": {}, "after": {}, "shard": [], "host": None}
    for line in open(f"{golden_dir}/slab_tiny.txt"):
        if line.startswith("#") or not line.strip():
            continue
        w = line.split()
        if w[0] == "geom":
            g["geom"][int(w[1])] = (int(w[2]), int(w[3]))
        elif w[0] == "host":
            g["host"] = (int(w[1]), w[2])
        elif w[0] in ("before", "after"):
            g[w[0]][int(w[1])] = w[2]
        elif w[0] == "shard":
            g["shard"].append((int(w[1]), int(w[2]), int(w[3]), w[4]))
    return g


def expand(label: str, unit_bytes: int) -> np.ndarray:
    return np.repeat(np.frombuffer(label.encode(), dtype=np.uint8), unit_bytes).copy()


@pytest.mark.parametrize("unit_bytes", [1, 16, 48])
def test_golden_slab_image(golden_dir, unit_bytes):
    g = load_slab_golden(golden_dir)
    old = [(0, 0, 4, 1), (1, 4, 6, 0), (2, 6, 9, 1), (3, 9, 12, 1)]
    tasks, new = OP.cmm_plan(old, 3)
    snap = {r: expand(s, unit_bytes) for r, s in g["before"].items()}
    host0, host = g["host"]
    out, stats = OS.apply_params(tasks, snap, g["geom"], unit_bytes, expand(host, unit_bytes), host0)
    for r, s in g["after"].items():
        assert out[r].tobytes() == expand(s, unit_bytes).tobytes(), f"rank {r}"
    for (r, b, e, s) in g["shard"]:
        a, c = g["geom"][r]
        assert OS.read_units(out[r], a, c, unit_bytes, b, e).tobytes() == expand(s, unit_bytes).tobytes()
    assert stats == {"d2d_bytes": unit_bytes, "h2d_bytes": 2 * unit_bytes, "kept_bytes": 9 * unit_bytes}
    # snapshot semantics: the inputs were not modified
    for r, s in g["before"].items():
        assert snap[r].tobytes() == expand(s, unit_bytes).tobytes()


def test_slot_addressing():
    assert [OS.slot(u, 6, 4) for u in (6, 7, 8, 4, 5)] == [0, 1, 2, 2, 3]      # golden's r2
    assert [OS.slot(u, 9, 4) for u in (9, 10, 11, 8)] == [0, 1, 2, 3]           # golden's r3
    L = OS._lib()
    for u in range(-20, 40):
        for anchor in (0, 3, 17):
            for cap in (1, 4, 7):
                assert L.oracle_slot(u, anchor, cap) == OS.slot(u, anchor, cap) == ((u - anchor) % cap + cap) % cap


# ------------------------------------------------------------------------------------------ plain definition, params
def check_plain_definition(world, step_idx, out):
    st = world.steps[step_idx]
    for sp in world.specs:
        W = world.unsharded[sp.name].reshape(sp.total_units, sp.unit_bytes)
        for (r, b, e, _) in st.new[sp.klass]:
            anchor, cap = world.geom[sp.name][r]
            S = out[sp.name][r].reshape(cap, sp.unit_bytes)
            idx = [(u - anchor) % cap for u in range(b, e)]
            assert len(set(idx)) == len(idx)
            assert np.array_equal(S[idx], W[b:e]), f"{sp.name} rank {r}: new shard != unsharded slice"


def check_untouched(world, step_idx, before, out):
    st = world.steps[step_idx]
    for sp in world.specs:
        for r, a in out[sp.name].items():
            anchor, cap = world.geom[sp.name][r]
            written = set()
            for (k, src, dst, b, e) in st.tasks[sp.klass]:
                if dst == r and k != OP.KEEP:
                    written |= {(u - anchor) % cap for u in range(b, e)}
            S0 = before[sp.name][r].reshape(cap, sp.unit_bytes)
            S1 = a.reshape(cap, sp.unit_bytes)
            keep = [s for s in range(cap) if s not in written]
            assert np.array_equal(S0[keep], S1[keep]), f"{sp.name} rank {r}: bytes outside the plan changed"


@pytest.mark.parametrize("mode", ["span", "tight", "full"])
@pytest.mark.parametrize("policy", ["floor", "ceil_first"])
@pytest.mark.parametrize("dead", [0, 1, 2, 3])
def test_config1_params_plain_definition(mode, policy, dead):
    cfg = get_config("1")
    world = H.build_param_world(cfg, mode=mode, new_policy=policy, failed=(dead,))
    out, stats = H.oracle_reshard_params(world, 0)
    check_plain_definition(world, 0, out)
    check_untouched(world, 0, world.slabs, out)
    total = sum(sp.total_units * sp.unit_bytes for sp in world.specs)
    assert stats["d2d_bytes"] + stats["h2d_bytes"] + stats["kept_bytes"] == total


def test_config1_byte_counts_match_survey():
    """FFN per tensor keep 435 / P2P 69 / reload 184 units of 512 B; heads: reload
    group 2 -> rank 3, no P2P."""
    world = H.build_param_world(get_config("1"))
    _, stats = H.oracle_reshard_params(world, 0)
    ffn_d2d = 3 * 69 * 512
    ffn_h2d = 3 * 184 * 512
    head_h2d = 32768 + 16384 + 16384 + 32768      # wq, wk, wv, wo_t: one KV group each
    assert stats["d2d_bytes"] == ffn_d2d
    assert stats["h2d_bytes"] == ffn_h2d + head_h2d


def test_sequential_reshards_tiny():
    """Config-5a style chain on the tiny shape: 4 -> 3 -> 2, each plan from the previous layout."""
    cfg = get_config("1")
    for mode in ("span", "tight"):
        world = H.build_param_world(cfg, mode=mode, failed=(2, 0))
        cur = world.slabs
        for i in range(2):
            out, _ = H.oracle_reshard_params(world, i, cur)
            check_plain_definition(world, i, out)
            cur = out


# ------------------------------------------------------------------------------------------ page table
def load_pt_golden(golden_dir):
    d = {"cases": []}
    row = lambda s: [[int(x) for x in r.split()] for r in s.split("|")]
    for line in open(f"{golden_dir}/page_table.txt"):
        if line.startswith("#") or not line.strip():
            continue
        w = line.split(None, 1)
        if w[0] in ("block_size",):
            d[w[0]] = int(w[1])
        elif w[0] in ("seq_lens", "last_use"):
            d[w[0]] = [int(x) for x in w[1].split()]
        elif w[0] == "table":
            d["table"] = np.array(row(w[1]), dtype=np.int32)
        elif w[0] == "case":
            budget, ev, tab = [x.strip() for x in w[1].split(":")]
            ev = [] if ev.split()[1] == "-" else [int(x) for x in ev.split()[1:]]
            d["cases"].append((int(budget), ev, np.array(row(tab), dtype=np.int32)))
    return d


def test_page_table_golden(golden_dir):
    d = load_pt_golden(golden_dir)
    assert len(d["cases"]) == 4
    for budget, ev, tab in d["cases"]:
        new, evicted, pairs = OS.page_table_rewrite(d["table"], d["seq_lens"], d["last_use"], d["block_size"], budget)
        assert evicted == ev, budget
        assert np.array_equal(new, tab), budget


def test_page_table_properties():
    rng = np.random.default_rng(5)
    for _ in range(200):
        n_seqs = int(rng.integers(1, 7))
        bs = int(rng.choice([1, 4, 16]))
        lens = rng.integers(0, 6 * bs, n_seqs)
        from workloads.gen import make_page_table
        table, lens, last_use, n_blocks = make_page_table(n_seqs, lens, bs, 1.5, int(rng.integers(1 << 30)))
        per = [-(-int(x) // bs) for x in lens]
        budget = int(rng.integers(0, n_blocks + 1))
        new, evicted, pairs = OS.page_table_rewrite(table, lens, last_use, bs, budget)
        surv = [s for s in range(n_seqs) if s not in evicted]
        ids = [int(new[s, i]) for s in surv for i in range(per[s])]
        assert len(set(ids)) == len(ids) and all(0 <= b < budget for b in ids)          # injective, in budget
        assert sum(per[s] for s in surv) <= budget
        # LRU order: every evicted sequence is colder than every surviving non-empty sequence
        for v in evicted:
            for s in surv:
                if per[s]:
                    assert (last_use[v], v) < (last_use[s], s)
        # minimal eviction: putting the last evicted one back would exceed the budget
        if evicted:
            assert sum(per[s] for s in surv) + per[evicted[-1]] > budget
        # blocks already below the budget never move
        for (s, i, bo, bn) in pairs:
            assert (bn == bo) if bo < budget else (bn < budget)
        for s in evicted:
            assert (new[s] == -1).all()


# ------------------------------------------------------------------------------------------ KV plain definition
def check_kv_plain_definition(world, st, out, new_table, evicted):
    g, cfg = world.g, world.cfg
    owner = {}
    for (r, b, e, _) in st.new["head"]:
        for h in range(b, e):
            owner[h] = r
    n = 0
    for s in range(cfg.kv.n_seqs):
        if s in evicted:
            continue
        for t in range(int(world.seq_lens[s])):
            b = int(new_table[s, t // g.block_size])
            for l in range(g.n_layers):
                for c in range(2):
                    for h in range(cfg.model.n_kv_heads):
                        r = owner[h]
                        got = H.kv_get(world, out[r], l, c, b, t % g.block_size, (h - world.anchors[r]) % g.head_cap)
                        assert np.array_equal(got, world.kv_ref[s, t, l, c, h]), (s, t, l, c, h)
                        n += 1
    return n


@pytest.mark.parametrize("layout", [0, 1])
@pytest.mark.parametrize("dead", [0, 1, 2, 3])
@pytest.mark.parametrize("budget", [None, 12])
def test_config1_kv_plain_definition(layout, dead, budget):
    """Config 1 KV: 2 seqs x 128 tokens, block 16 (20-block pool); budget 12 of 20 -> one eviction + relocations."""
    cfg = get_config("1")
    world = H.build_kv_world(cfg, layout=layout, failed=(dead,))
    st = world.steps[0]
    bud = world.g.n_blocks if budget is None else budget
    new_table, evicted, pairs = OS.page_table_rewrite(world.table, world.seq_lens, world.last_use,
                                                      world.g.block_size, bud)
    if budget is None:
        assert evicted == [] and np.array_equal(new_table, world.table)
    else:
        assert len(evicted) == 1 and any(bo != bn for (_, _, bo, bn) in pairs)
    snap = {r: p for r, p in world.pools.items() if r != dead}
    out, stats = OS.apply_kv(st.tasks["head"], snap, world.anchors, world.g, world.host_backup,
                             world.host_heads, world.host_head0, pairs)
    n = check_kv_plain_definition(world, st, out, new_table, evicted)
    assert n > 0
    # nothing outside live destination blocks changed
    touched_blocks = {bn for (_, _, _, bn) in pairs}
    for r in out:
        v0, v1 = H.kv_view(world, snap[r]), H.kv_view(world, out[r])
        for b in range(world.g.n_blocks):
            if b not in touched_blocks:
                assert np.array_equal(v0[:, :, b], v1[:, :, b])


def load_kv_golden(golden_dir):
    g = {"plan": [], "anchor": {}, "before": {}, "after": {}, "backup": {}}
    kinds = {"K": OP.KEEP, "T": OP.TRANSFER, "R": OP.RELOAD}
    for line in open(f"{golden_dir}/kv_tiny.txt"):
        if line.startswith("#") or not line.strip():
            continue
        w = line.split()
        if w[0] == "plan":
            g["plan"].append((kinds[w[1]], int(w[2]), int(w[3]), int(w[4]), int(w[5])))
        elif w[0] == "anchor":
            g["anchor"][int(w[1])] = int(w[2])
        elif w[0] in ("before", "after"):
            g[w[0]][(int(w[1]), int(w[2]), int(w[3]))] = w[5:]
        elif w[0] == "backup":
            g["backup"][(int(w[1]), int(w[2]))] = w[4:]
        elif w[0] in ("table", "new_table", "stats"):
            g[w[0]] = [int(x) for x in w[1:]]
        else:
            g[w[0]] = int(w[1])
    return g


def kv_golden_pool(g, rows, heads, layout, frag):
    """Expand the golden's per-plane picture {(block, token): [fragment per slot]} into a pool image through a numpy N-d
    view (never through the oracle's offset arithmetic): fragment "c4" in plane p -> bytes 1 + 4 + 8*2 + 32*p."""
    L, nb, bs = g["n_layers"], g["n_blocks"], g["block_size"]
    shape = (L, 2, nb, bs, heads, frag) if layout == 0 else (L, 2, nb, heads, bs, frag)
    pool = np.zeros(shape, dtype=np.uint8)
    for (b, t), slots in rows.items():
        for sl, name in enumerate(slots):
            for l in range(L):
                for c in range(2):
                    p = 2 * l + c
                    val = 200 + int(name[1:]) + 10 * p if name[0] == "g" else 1 + int(name[1]) + 8 * (ord(name[0]) - ord("a")) + 32 * p
                    if layout == 0:
                        pool[l, c, b, t, sl, :] = val
                    else:
                        pool[l, c, b, sl, t, :] = val
    return pool.reshape(-1)


@pytest.mark.parametrize("layout", [0, 1])
@pytest.mark.parametrize("frag", [1, 16])
def test_golden_kv_image(golden_dir, layout, frag):
    """tests/golden/kv_tiny.txt: a relocated block, a TRANSFER head, a RELOAD head into a wrapped slot, kept heads, a free
    block, both block layouts - the hand-worked picture against page_table_rewrite + apply_kv."""
    g = load_kv_golden(golden_dir)
    old = [(0, 0, 3, 1), (1, 3, 4, 0), (2, 4, 5, 1)]
    tasks, new = OP.cmm_plan(old, 2)
    assert tasks == g["plan"] and new == [(0, 0, 2, 1), (2, 2, 5, 1)]
    table = np.array([g["table"]], dtype=np.int32)
    new_table, evicted, pairs = OS.page_table_rewrite(table, [4], [0], g["block_size"], g["budget"])
    assert new_table.tolist() == [g["new_table"]] and evicted == [] and pairs == [(0, 0, 2, 1), (0, 1, 0, 0)]
    geom = OS.KVGeom(g["n_layers"], g["n_blocks"], g["block_size"], g["head_cap"], frag, 1, layout)
    per_rank = lambda which, r: {(b, t): v for (rr, b, t), v in g[which].items() if rr == r}
    snap = {r: kv_golden_pool(g, per_rank("before", r), g["head_cap"], layout, frag) for r in (0, 2)}
    before = {r: a.copy() for r, a in snap.items()}
    backup = kv_golden_pool(g, g["backup"], 1, layout, frag)
    out, stats = OS.apply_kv(tasks, snap, g["anchor"], geom, backup, 1, 3, pairs)
    for r in (0, 2):
        exp = kv_golden_pool(g, per_rank("after", r), g["head_cap"], layout, frag)
        assert out[r].tobytes() == exp.tobytes(), f"rank {r}, layout {layout}"
        assert snap[r].tobytes() == before[r].tobytes()          # snapshot semantics: the inputs were not modified
    d2d, h2d, kept = g["stats"]
    assert stats == {"d2d_bytes": d2d * frag, "h2d_bytes": h2d * frag, "kept_bytes": kept * frag}
    # a single fragment through the oracle's own accessor: token b (block 1 after the move), head 3 at r2's wrapped slot 2
    assert OS.kv_fragment(out[2], geom, g["anchor"][2], 1, 1, 1, 1, 3)[0] == 1 + 3 + 8 * 1 + 32 * 3


def test_kv_ragged_lengths_and_head_major():
    cfg = get_config("1")
    world = H.build_kv_world(cfg, layout=1, seq_lens=[37, 128])
    st = world.steps[0]
    new_table, evicted, pairs = OS.page_table_rewrite(world.table, world.seq_lens, world.last_use,
                                                      world.g.block_size, world.g.n_blocks)
    snap = {r: p for r, p in world.pools.items() if r != st.dead}
    out, _ = OS.apply_kv(st.tasks["head"], snap, world.anchors, world.g, world.host_backup,
                         world.host_heads, world.host_head0, pairs)
    check_kv_plain_definition(world, st, out, new_table, evicted)


# ------------------------------------------------------------------------------------------ linear reference
def test_linear_ref_is_the_textbook_definition():
    rng = np.random.default_rng(1)
    x = rng.standard_normal((3, 17))
    w = rng.standard_normal((5, 17))
    np.testing.assert_allclose(OL.linear_ref(x, w), OL.linear_triple_loop(x, w), rtol=1e-12, atol=1e-12)
    # a transposed operand or a dropped term fails:
    assert OL.linear_ref(x, w).shape == (3, 5)
    e = np.eye(4)
    assert np.array_equal(OL.linear_ref(e, np.arange(16.0).reshape(4, 4)), np.arange(16.0).reshape(4, 4).T)


def test_decode16_exact():
    import torch
    for name, dt in (("bf16", torch.bfloat16), ("fp16", torch.float16)):
        t = torch.tensor([0.0, 1.0, -2.5, 0.02, 65504.0 if name == "fp16" else 3.0e38, 1e-3], dtype=dt)
        got = OL.decode16(t.view(torch.uint8).numpy(), name)
        assert np.array_equal(got, t.to(torch.float64).numpy())
    assert OL.max_rel_err(np.array([1.0, 2.0]), np.array([1.0, 2.01])) == pytest.approx(0.01 / 2.01)


# ------------------------------------------------------------------------------------------ MoE reference (reading G5)
def test_moe_route_hand_worked():
    """softmax / top-k / renormalisation on a case small enough to do by hand: logits (0, ln 2, ln 4, ln 1) -> p = (1, 2, 4, 1)/8;
    top-2 = experts 2 and 1 with weights 4/6 and 2/6; the tie between experts 0 and 3 goes to the lower index (top-3)."""
    import math
    lg = np.array([[0.0, math.log(2.0), math.log(4.0), 0.0]])
    idx, w = OL.moe_route(lg, 2)
    assert idx.tolist() == [[2, 1]]
    np.testing.assert_allclose(w, [[4 / 6, 2 / 6]], rtol=1e-14)
    idx, w = OL.moe_route(lg, 3)
    assert idx.tolist() == [[2, 1, 0]]
    np.testing.assert_allclose(w, [[4 / 7, 2 / 7, 1 / 7]], rtol=1e-14)
    # shift invariance of softmax and weights summing to one
    idx2, w2 = OL.moe_route(lg + 123.0, 3)
    assert idx2.tolist() == idx.tolist()
    np.testing.assert_allclose(w2, w, rtol=1e-12)


def test_moe_ref_special_cases():
    import math
    rng = np.random.default_rng(7)
    T, Hd, F, E = 5, 6, 4, 3
    x = rng.standard_normal((T, Hd))
    gate, up, down_t = (rng.standard_normal((E, F, Hd)) for _ in range(3))
    lg = rng.standard_normal((T, E))
    # (i) one expert, top-1: the layer is a dense SwiGLU MLP, written out with scalar loops
    y = OL.moe_ref(x, lg[:, :1], gate[:1], up[:1], down_t[:1], 1)
    for t in range(T):
        for o in range(Hd):
            acc = 0.0
            for f in range(F):
                g = sum(gate[0, f, k] * x[t, k] for k in range(Hd))
                u = sum(up[0, f, k] * x[t, k] for k in range(Hd))
                acc += g / (1.0 + math.exp(-g)) * u * down_t[0, f, o]
            assert y[t, o] == pytest.approx(acc, rel=1e-12, abs=1e-12)
    # (ii) identical experts: the renormalised weights sum to one, so any routing gives the single-expert output
    same = lambda a: np.repeat(a[:1], E, axis=0)
    np.testing.assert_allclose(OL.moe_ref(x, lg, same(gate), same(up), same(down_t), 2), y, rtol=1e-12, atol=1e-12)
    # (iii) renaming the experts (and the logit columns with them) changes nothing
    perm = np.array([2, 0, 1])
    np.testing.assert_allclose(OL.moe_ref(x, lg[:, perm], gate[perm], up[perm], down_t[perm], 2),
                               OL.moe_ref(x, lg, gate, up, down_t, 2), rtol=1e-12, atol=1e-12)
    # (iv) top_k = E with equal logits: the plain average of all experts
    avg = sum(OL.moe_ref(x, lg[:, :1], gate[e:e + 1], up[e:e + 1], down_t[e:e + 1], 1) for e in range(E)) / E
    np.testing.assert_allclose(OL.moe_ref(x, np.zeros((T, E)), gate, up, down_t, E), avg, rtol=1e-12, atol=1e-12)
    # (v) a hugely dominant logit with top-1 picks exactly that expert
    big = np.full((T, E), -50.0)
    big[:, 1] = 50.0
    np.testing.assert_allclose(OL.moe_ref(x, big, gate, up, down_t, 1),
                               OL.moe_ref(x, lg[:, :1], gate[1:2], up[1:2], down_t[1:2], 1), rtol=1e-12, atol=1e-12)


# ------------------------------------------------------------------------------------------ all-cores leg == 1-core oracle
def test_parallel_appliers_equal_the_plain_ones():
    """oracle.state.apply_params_parallel / apply_kv_parallel (the OpenMP loop over jobs that bench.py times as the all-cores
    baseline) must produce exactly the images and counters of apply_params / apply_kv, task by task and byte by byte."""
    cfg = get_config("1")
    for mode, dead in (("tight", 2), ("span", 0), ("full", 3)):
        world = H.build_param_world(cfg, mode=mode, failed=(dead,))
        expect, stats = H.oracle_reshard_params(world, 0)
        st = world.steps[0]
        items = [(st.tasks[sp.klass], {r: a for r, a in world.slabs[sp.name].items() if r != st.dead}, world.geom[sp.name],
                  sp.unit_bytes, world.unsharded[sp.name], 0) for sp in world.specs]
        outs, pstats = OS.apply_params_parallel(items, job_bytes=4096)
        assert pstats == stats
        for sp, out in zip(world.specs, outs):
            for r, a in out.items():
                assert a.tobytes() == expect[sp.name][r].tobytes(), (mode, sp.name, r)
    for layout in (0, 1):
        kw = H.build_kv_world(cfg, layout=layout, failed=(1,))
        st, g = kw.steps[0], kw.g
        _, evicted, pairs = OS.page_table_rewrite(kw.table, kw.seq_lens, kw.last_use, g.block_size, 12)
        snap = {r: p for r, p in kw.pools.items() if r != st.dead}
        exp, stats = OS.apply_kv(st.tasks["head"], snap, kw.anchors, g, kw.host_backup, kw.host_heads, kw.host_head0, pairs)
        got, pstats = OS.apply_kv_parallel(st.tasks["head"], snap, kw.anchors, g, kw.host_backup, kw.host_heads, kw.host_head0, pairs,
                                           pairs_per_job=3)
        assert pstats == stats
        for r in exp:
            assert got[r].tobytes() == exp[r].tobytes()
    assert OS.omp_threads() >= 1


def test_swiglu_ref_is_the_inner_term_of_moe_ref():
    """oracle.linear.swiglu_ref (pins the fused gate|up kernel) against scalar loops, and moe_ref with one expert and an
    identity down projection returns exactly it."""
    import math
    rng = np.random.default_rng(9)
    R, Hd, F = 3, 5, 5                       # F = hidden so that an identity down projection exists
    x, g, u = rng.normal(size=(R, Hd)), rng.normal(size=(F, Hd)), rng.normal(size=(F, Hd))
    h = OL.swiglu_ref(x, g, u)
    for r in range(R):
        for f in range(F):
            a = sum(g[f, k] * x[r, k] for k in range(Hd))
            b = sum(u[f, k] * x[r, k] for k in range(Hd))
            assert abs(h[r, f] - a / (1.0 + math.exp(-a)) * b) < 1e-12
    y = OL.moe_ref(x, np.zeros((R, 1)), g[None], u[None], np.eye(F)[None], 1)
    np.testing.assert_allclose(y, h, rtol=1e-13)
