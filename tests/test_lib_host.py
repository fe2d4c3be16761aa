"""Host logic of libetp.so against the oracle (no GPU needed): the library loads and exports every symbol
include/etp.h declares; etp_partition / etp_cmm_plan / etp_plan_create / etp_page_table_rewrite agree with the
oracle exactly (the plan is unique under the readings of DESIGN.md, so task lists are compared verbatim);
status codes of the error paths."""
import os
import re

import numpy as np
import pytest

import paper_2511_11617_b200 as etp
from oracle import planning as OP
from oracle import state as OS
from tests import harness as H
from workloads import get_config

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_symbols():
    src = open(os.path.join(ROOT, "include", "etp.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(etp_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    L = etp.lib()
    syms = header_symbols()
    assert set(syms) == set(etp.EXPORTS), (syms, etp.EXPORTS)
    for s in syms:
        assert getattr(L, s) is not None
    assert "sm_100a" in etp.etp_version()


def test_binding_does_not_import_oracle():
    for f in os.listdir(os.path.join(ROOT, "paper_2511_11617_b200")):
        if f.endswith(".py"):
            txt = open(os.path.join(ROOT, "paper_2511_11617_b200", f)).read()
            assert "oracle" not in txt.replace("``oracle/``", ""), f
    for f in os.listdir(os.path.join(ROOT, "paper_2511_11617_b200", "csrc")):
        assert "oracle" not in open(os.path.join(ROOT, "paper_2511_11617_b200", "csrc", f)).read(), f


def test_fig3_through_the_c_abi(golden_dir):
    """PAPER.md:144 (Fig. 3): 1024 rows, 4 -> 3, GPU:2 (rank 1) fails."""
    assert etp.etp_partition(1024, 3) == [0, 341, 682, 1024]
    old = [(0, 0, 256, 1), (1, 256, 512, 0), (2, 512, 768, 1), (3, 768, 1024, 1)]
    p = etp.etp_cmm_plan(old, 3)
    K, T, R = etp.KEEP, etp.TRANSFER, etp.RELOAD
    assert p.tasks() == [(K, 0, 0, 0, 256), (R, -1, 0, 256, 341), (R, -1, 2, 341, 512), (K, 2, 2, 512, 682),
                         (T, 2, 3, 682, 768), (K, 3, 3, 768, 1024)]
    st = p.stats()
    assert (st["keep_units"], st["transfer_units"], st["reload_units"], st["reload_lower_bound"]) == (682, 86, 256, 256)
    assert p.new_layout() == [(0, 0, 341, 1), (2, 341, 682, 1), (3, 682, 1024, 1)]


@pytest.mark.parametrize("policy", ["floor", "ceil_first"])
def test_partition_matches_oracle(policy):
    rng = np.random.default_rng(7)
    for _ in range(400):
        M = int(rng.integers(1, 17))
        S = int(rng.integers(M, 200000))
        a = int(rng.choice([1, 1, 1, 2, 8, 128]))
        if -(-S // a) < M:
            continue
        assert etp.etp_partition(S, M, policy, a) == OP.partition(S, M, policy, a)
    for S in (8, 17408, 14336, 128, 151936, 128256, 688, 4):
        for M in (1, 2, 3, 4):
            assert etp.etp_partition(S, M, policy) == OP.partition(S, M, policy)


def random_layout(rng, max_n=8, max_h=3000):
    n = int(rng.integers(2, max_n + 1))
    H_ = int(rng.integers(n, max_h))
    cuts = sorted(rng.choice(np.arange(1, H_), size=n - 1, replace=False).tolist()) if n > 1 else []
    b = [0] + cuts + [H_]
    n_dead = int(rng.integers(0, min(3, n - 1) + 1))
    dead = set(rng.choice(n, size=n_dead, replace=False).tolist())
    ranks = sorted(rng.choice(np.arange(0, 2 * n), size=n, replace=False).tolist())
    return [(int(ranks[i]), b[i], b[i + 1], 0 if i in dead else 1) for i in range(n)]


def test_cmm_plan_matches_oracle_random():
    rng = np.random.default_rng(11)
    for it in range(400):
        old = random_layout(rng)
        n_alive = sum(a for (_, _, _, a) in old)
        M = int(rng.integers(1, n_alive + 1))
        Ht = max(e for (_, _, e, _) in old)
        tb = None
        if it % 3 and Ht >= M:
            tb = OP.partition(Ht, M, "ceil_first" if it % 2 else "floor")
        tasks, new = OP.cmm_plan(old, M, tb)
        p = etp.etp_cmm_plan(old, M, tb)
        assert p.tasks() == tasks
        assert p.new_layout() == new
        st, ref = p.stats(), OP.plan_stats(tasks)
        for k in ref:
            assert st[k] == ref[k]
        assert st["reload_lower_bound"] == OP.eq1_reload_lower_bound(old, [b for (_, b, _, _) in new] + [Ht])
        assert st["reload_units"] == st["reload_lower_bound"]          # Eq. 1 attained


def test_comparison_planners_match_oracle():
    """PAPER.md:204 / Table II: Greedy (no P2P for gaps) and Full Reload (no reuse)."""
    rng = np.random.default_rng(13)
    for _ in range(100):
        old = random_layout(rng)
        M = sum(a for (_, _, _, a) in old)
        g_tasks, _ = OP.greedy_plan(old, M)
        f_tasks, _ = OP.full_reload_plan(old, M)
        pg = etp.etp_plan_create(etp.PLAN_GREEDY, old, M)
        pf = etp.etp_plan_create(etp.PLAN_FULL_RELOAD, old, M)
        assert OP._merge_adjacent(pg.tasks()) == g_tasks
        assert pf.tasks() == f_tasks
        pc = etp.etp_cmm_plan(old, M)
        assert pc.stats()["reload_units"] <= pg.stats()["reload_units"] <= pf.stats()["reload_units"]


def test_migration_aware_planner_matches_oracle():
    """Reading M1: the library's subset-DP assignment against the oracle's exhaustive search, task for task (ties included),
    with free bounds (all placements of the wide shards) and with fixed bounds; never more transfers than Algorithm 1's
    in-order owners, the same (minimal) reload."""
    rng = np.random.default_rng(29)
    gained = 0
    for it in range(150):
        old = random_layout(rng)
        n_alive = sum(a for (_, _, _, a) in old)
        M = int(rng.integers(1, n_alive + 1))
        Ht = max(e for (_, _, e, _) in old)
        if Ht < M or M > 5:
            continue
        tb = OP.partition(Ht, M, "ceil_first") if it % 3 == 0 else None
        tasks, new = OP.migration_aware_plan(old, M, tb)
        p = etp.etp_plan_create(etp.PLAN_MIGRATION_AWARE, old, M, tb)
        assert p.new_layout() == new
        assert p.tasks() == tasks
        base = etp.etp_cmm_plan(old, M, tb).stats()
        st = p.stats()
        assert st["reload_units"] == base["reload_units"] == st["reload_lower_bound"]
        assert st["transfer_units"] <= base["transfer_units"]
        gained += st["transfer_units"] < base["transfer_units"]
    assert gained > 10
    with pytest.raises(etp.EtpError) as e:      # search limited to 10 alive ranks
        etp.etp_plan_create(etp.PLAN_MIGRATION_AWARE, [(r, r, r + 1, 1) for r in range(11)], 11)
    assert e.value.status == 5


def test_replicated_sources_reading_c7():
    old = [(0, 0, 6, 1), (1, 4, 10, 1), (2, 8, 12, 0)]
    tasks, new = OP.cmm_plan(old, 2)
    p = etp.etp_cmm_plan(old, 2)
    assert p.tasks() == tasks and p.new_layout() == new


def test_scenario_plans_of_every_config_match():
    class LibSide:
        @staticmethod
        def partition(Hh, M, policy="floor", align=1):
            return etp.etp_partition(Hh, M, policy, align)

        @staticmethod
        def plan(old, M, tb=None):
            p = etp.etp_cmm_plan(old, M, tb)
            return p.tasks(), p.new_layout()

    for key in ("1", "2", "2b", "3", "4", "5a"):
        cfg = get_config(key)
        a = H.plan_scenario(cfg, H.OracleSide)
        b = H.plan_scenario(cfg, LibSide)
        assert len(a) == len(b)
        for sa, sb in zip(a, b):
            assert sa.tasks == sb.tasks and sa.new == sb.new, key


def test_page_table_rewrite_matches_oracle():
    rng = np.random.default_rng(17)
    for _ in range(200):
        n_seqs = int(rng.integers(1, 9))
        bs = int(rng.choice([1, 4, 16]))
        lens = rng.integers(0, 9 * bs, n_seqs).astype(np.int32)
        per = (lens + bs - 1) // bs
        live = int(per.sum())
        n_blocks = live + int(rng.integers(0, 6))
        ids = rng.permutation(max(n_blocks, 1))[:live]
        mb = max(int(per.max()), 1)
        table = np.full((n_seqs, mb), -1, dtype=np.int32)
        k = 0
        for s in range(n_seqs):
            table[s, : per[s]] = ids[k : k + per[s]]
            k += per[s]
        last_use = rng.integers(0, 5, n_seqs).astype(np.int64)        # ties on purpose
        budget = int(rng.integers(0, n_blocks + 1))
        ref_table, ref_ev, ref_pairs = OS.page_table_rewrite(table, lens, last_use, bs, budget)
        t = table.copy()
        ev, pairs = etp.etp_page_table_rewrite(t, lens, last_use, bs, budget)
        assert ev == ref_ev
        assert np.array_equal(t, ref_table)
        assert pairs == [(bo, bn) for (_, _, bo, bn) in ref_pairs]


def test_page_table_golden_through_the_c_abi(golden_dir):
    from tests.test_oracle_state import load_pt_golden
    g = load_pt_golden(golden_dir)
    for budget, evicted, tab in g["cases"]:
        t = np.array(g["table"], dtype=np.int32)
        ev, pairs = etp.etp_page_table_rewrite(t, g["seq_lens"], g["last_use"], g["block_size"], budget)
        assert ev == evicted, budget
        assert np.array_equal(t, tab), budget


def test_error_statuses():
    E = etp.EtpError
    with pytest.raises(E) as e:
        etp.etp_partition(4, 5)
    assert e.value.status == 5                      # UNSUPPORTED: fewer units than shards (reading P4)
    with pytest.raises(E) as e:
        etp.etp_partition(10, 0)
    assert e.value.status == 1
    with pytest.raises(E) as e:
        etp.etp_cmm_plan([(0, 0, 4, 1), (1, 4, 8, 0)], 2)      # M > #alive (reading C6)
    assert e.value.status == 1
    with pytest.raises(E) as e:
        etp.etp_cmm_plan([(0, 0, 4, 1), (0, 4, 8, 1)], 1)      # duplicate rank id
    assert e.value.status == 1
    with pytest.raises(E) as e:
        etp.etp_cmm_plan([(0, 0, 4, 1), (1, 4, 8, 1)], 2, [0, 5, 7])   # bounds do not tile [0,H)
    assert e.value.status == 1
    # an empty interval is a joining rank (reading C6)
    p = etp.etp_cmm_plan([(0, 0, 8, 1), (1, 8, 8, 1)], 2)
    assert p.tasks() == OP.cmm_plan([(0, 0, 8, 1), (1, 8, 8, 1)], 2)[0]


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(etp.EtpError) as e:
        etp.Context(0)
    assert e.value.status == 6                      # ETP_ERR_CUDA


def test_weighted_migration_aware_planner_matches_oracle():
    """etp_plan_create_weighted (reading M2) against oracle.planning.migration_aware_plan(link_cost=...): random layouts (rank
    ids with gaps, several dead ranks), random integer link prices, free and fixed bounds; task for task and layout for
    layout.  Uniform prices give the unweighted plan; link costs with another planner mode are rejected."""
    rng = np.random.default_rng(77)
    done = 0
    while done < 150:
        old = random_layout(rng, max_n=6, max_h=60)
        alive = [s for s in old if s[3]]
        M = int(rng.integers(1, len(alive) + 1))
        Hn = max(e for (_, _, e, _) in old)
        if Hn < M:
            continue
        n_cost = max(r for (r, _, _, _) in old) + 1
        cost = [[0 if a == b else int(rng.integers(1, 10)) for b in range(n_cost)] for a in range(n_cost)]
        tb = OP.partition(Hn, M, ["floor", "ceil_first"][int(rng.integers(0, 2))]) if rng.random() < 0.4 else None
        p = etp.etp_plan_create(etp.PLAN_MIGRATION_AWARE, old, M, tb, link_cost=cost)
        tasks, new = OP.migration_aware_plan(old, M, tb, cost)
        assert p.tasks() == tasks and p.new_layout() == new, (old, M, tb, cost)
        done += 1
    # replicated sources: the cheaper link supplies the unit (C7 -> M2)
    rep = [(0, 0, 4, 1), (1, 0, 4, 1), (2, 4, 8, 1), (3, 8, 8, 1)]
    cost = [[0, 9, 9, 9], [9, 0, 9, 1], [9, 9, 0, 9], [9, 9, 9, 0]]
    p = etp.etp_plan_create(etp.PLAN_MIGRATION_AWARE, rep, 4, [0, 2, 4, 6, 8], link_cost=cost)
    tasks, new = OP.migration_aware_plan(rep, 4, [0, 2, 4, 6, 8], cost)
    assert p.tasks() == tasks and p.new_layout() == new
    old = [(r, 7 * r, 7 * r + 7, 0 if r == 3 else 1) for r in range(8)]
    ones = [[0 if a == b else 1 for b in range(8)] for a in range(8)]
    base = etp.etp_plan_create(etp.PLAN_MIGRATION_AWARE, old, 7)
    same = etp.etp_plan_create(etp.PLAN_MIGRATION_AWARE, old, 7, link_cost=ones)
    assert same.tasks() == base.tasks() and same.new_layout() == base.new_layout()
    with pytest.raises(etp.EtpError) as e:
        etp.etp_plan_create(etp.PLAN_CMM, old, 7, link_cost=ones)
    assert e.value.status == 1
    with pytest.raises(etp.EtpError) as e:
        etp.etp_plan_create(etp.PLAN_MIGRATION_AWARE, old, 7, link_cost=[[0, 1], [1, 0]])
    assert e.value.status == 1


def test_eplb_place_matches_oracle():
    """etp_eplb_place (incremental integer loads, 128-bit cross-multiplication) against oracle/eplb.py (Fractions, recomputed
    from scratch every step): Fig. 4's hand-worked instance and 300 random ones incl. dead ranks, homeless experts, zero loads."""
    from oracle import eplb
    assert etp.etp_eplb_place([60, 20, 20, 10], [0, -1, 2, 3], [2, 0, 2, 3], [2, 0, 2, 2]) == [(1, 3), (0, 3), (1, 2)]
    rng = np.random.default_rng(5)
    for _ in range(300):
        R = int(rng.integers(2, 7))
        E = int(rng.integers(1, 14))
        load = [int(v) for v in rng.integers(0, 2000, E)]
        cap = [int(v) for v in rng.integers(0, 6, R)]
        if not any(cap):
            cap[0] = 1
        usable = [r for r in range(R) if cap[r] > 0]
        home = [int(rng.choice(usable)) if rng.random() > 0.15 else -1 for _ in range(E)]
        slots = [int(v) for v in rng.integers(0, 4, R)]
        if sum(slots[r] for r in usable) < sum(1 for h in home if h < 0):
            with pytest.raises(etp.EtpError) as e:
                etp.etp_eplb_place(load, home, cap, slots)
            assert e.value.status == 3
            continue
        replicas, _ = eplb.place(load, home, cap, slots)
        assert etp.etp_eplb_place(load, home, cap, slots) == replicas, (load, home, cap, slots)
    with pytest.raises(etp.EtpError) as e:
        etp.etp_eplb_place([1], [0], [0], [1])
    assert e.value.status == 1


# ------------------------------------------------------------------------------------------------ interval contract check (host-only)
def _brute_force_verdict(src, dst, sz):
    """The contract of include/etp.h by its plain definition, O(n^2): 'align', 'arg' or None."""
    n = len(sz)
    for i in range(n):
        if sz[i] == 0:
            continue
        if sz[i] < 0 or src[i] == 0 or dst[i] == 0:
            return "arg"
        if (src[i] | dst[i] | sz[i]) & 15:
            return "align"
    live = [i for i in range(n) if sz[i] > 0]
    for a in live:
        for b in live:
            if a < b and dst[a] < dst[b] + sz[b] and dst[b] < dst[a] + sz[a]:
                return "arg"
            if dst[a] < src[b] + sz[b] and src[b] < dst[a] + sz[a]:
                return "arg"
    return None


def _lib_verdict(src, dst, sz):
    try:
        etp.etp_intervals_validate(np.asarray(src, np.int64), np.asarray(dst, np.int64), np.asarray(sz, np.int64))
        return None
    except etp.EtpError as e:
        return {1: "arg", 2: "align"}[e.status]


def test_intervals_validate_against_the_plain_definition():
    """etp_intervals_validate (no device, no context) on 3000 random small plans with planted faults of every kind (overlapping
    destinations, a destination inside a source, its own shifted source, misalignment, negative and zero sizes) against the
    O(n^2) definition of the contract; touching intervals and overlapping SOURCES are legal."""
    rng = np.random.default_rng(11617)
    n_bad = n_ok = 0
    for case in range(3000):
        n = int(rng.integers(1, 12))
        sz = rng.integers(1, 6, n).astype(np.int64) * 16
        dst = 0x10000 + (np.cumsum(sz + rng.integers(0, 2, n) * 16) - sz)           # disjoint, some touching
        dst = dst[rng.permutation(n)]
        src = 0x40000 + rng.integers(0, 64, n).astype(np.int64) * 16                # sources may overlap each other
        kind = int(rng.integers(0, 8))
        k, j = int(rng.integers(0, n)), int(rng.integers(0, n))
        if kind == 1 and n > 1 and k != j:
            dst[k] = dst[j] + 16 * int(rng.integers(-2, 3))                          # destinations overlap (or touch / miss)
        elif kind == 2:
            src[k] = dst[j] + 16 * int(rng.integers(-3, 4))                          # a source on / next to a destination
        elif kind == 3:
            src[k] += 8                                                              # misaligned
        elif kind == 4:
            sz[k] = -16
        elif kind == 5:
            sz[k] = 0                                                                # ignored, whatever its addresses
            dst[k] = dst[j]
        elif kind == 6:
            src[k] = dst[k] + 16                                                     # a shifting copy onto itself
        want, got = _brute_force_verdict(src, dst, sz), _lib_verdict(src, dst, sz)
        assert want == got, (case, kind, src.tolist(), dst.tolist(), sz.tolist(), want, got)
        n_bad += want is not None
        n_ok += want is None
    assert n_bad > 500 and n_ok > 500


@pytest.mark.parametrize("n", [70_000, 300_000])
def test_intervals_validate_threaded_path_finds_one_planted_overlap(n):
    """From 65536 intervals the check runs on several threads (address buckets sorted independently): a valid random plan passes; one
    destination moved 16 bytes into its neighbour, or one source pointed at some destination, is reported with both indices."""
    rng = np.random.default_rng(n)
    sz = rng.integers(1, 9, n).astype(np.int64) * 16
    dst_sorted = 0x1000000 + (np.cumsum(sz + rng.integers(0, 3, n) * 16) - sz)
    perm = rng.permutation(n)
    dst, szp = dst_sorted[perm], sz[perm]
    src = 0x7f0000000000 + rng.integers(0, 1 << 24, n).astype(np.int64) * 16
    etp.etp_intervals_validate(src, dst, szp)
    k = int(np.argmax(dst == dst_sorted[n // 3]))
    pred = int(np.argmax(dst == dst_sorted[n // 3 - 1]))
    bad = dst.copy()
    bad[k] = dst[pred] + szp[pred] - 16
    with pytest.raises(etp.EtpError) as e:
        etp.etp_intervals_validate(src, bad, szp)
    assert e.value.status == 1 and str(pred) in str(e.value) and str(k) in str(e.value)
    bad_s = src.copy()
    bad_s[5] = dst[k] + 16 if szp[k] > 16 else dst[k]
    with pytest.raises(etp.EtpError) as e:
        etp.etp_intervals_validate(bad_s, dst, szp)
    assert e.value.status == 1 and " 5" in str(e.value) and str(k) in str(e.value)


# ------------------------------------------------------------------------------------------------ bench.py's watchdog
@pytest.mark.parametrize("mode,attempts,killed,rc", [("ok", 1, 0, 0), ("hang_once", 2, 1, 0), ("hang_after_result", 1, 1, 0), ("hang", None, 2, 1)])
def test_bench_watchdog_reports_its_retries(tmp_path, mode, attempts, killed, rc):
    """A hang must be visible in the result line: the child's stdout is forwarded, the last JSON object gets
    {"watchdog": {"attempts", "killed"}}; a child that printed its result and then hung is not repeated (exactly one result
    line); two hangs in a row give a non-zero exit code and no result line."""
    import json
    import subprocess
    import sys
    env = dict(os.environ, ETP_WATCHDOG_SELFTEST_MARK=str(tmp_path / "mark"))
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--watchdog-selftest", mode, "--watchdog-s", "6"],
                       stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, env=env, timeout=120)
    assert p.returncode == rc, p.stderr
    results = [json.loads(ln) for ln in p.stdout.splitlines() if ln.startswith("{")]
    if attempts is None:
        assert results == [] and "killed" in p.stderr
        return
    assert len(results) == 1 and results[0]["metric"] == "selftest"
    assert results[0]["watchdog"] == {"attempts": attempts, "killed": killed, "deadline_s": 6.0}
    assert p.stdout.count("a line that is not the result") == 1
