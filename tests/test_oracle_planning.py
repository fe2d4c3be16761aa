"""Pins for the oracle's S1 partition and S2 CMM plan — against the paper's printed values (Fig. 3),
Eq. 1's closed form, exhaustive enumeration, and the invariants of BASELINE.json's north_star.
None of these re-types the oracle's own formula."""
import itertools
import random

import pytest

from oracle import bruteforce
from oracle.planning import (CEIL_FIRST, FLOOR, KEEP, RELOAD, TRANSFER, cmm_plan, eq1_reload_lower_bound,
                             full_reload_plan, greedy_plan, layout_from_bounds, layout_from_widths, migration_aware_plan,
                             partition, plan_stats, weighted_transfer_cost, width_arrangements)

KIND = {"KEEP": KEEP, "TRANSFER": TRANSFER, "RELOAD": RELOAD}


def load_fig3(golden_dir):
    old, tasks, bounds, M, reload_total = [], [], None, None, None
    for line in open(f"{golden_dir}/fig3.txt"):
        line = line.split("#")[0].split()
        if not line:
            continue
        if line[0] == "old":
            old.append(tuple(int(x) for x in line[1:5]))
        elif line[0] == "M":
            M = int(line[1])
        elif line[0] == "bounds":
            bounds = [int(x) for x in line[1:]]
        elif line[0] == "task":
            tasks.append((KIND[line[1]],) + tuple(int(x) for x in line[2:6]))
        elif line[0] == "reload_total":
            reload_total = int(line[1])
    return old, M, bounds, tasks, reload_total


def test_fig3_partition_bounds(golden_dir):
    """PAPER.md:144 prints the target plan [0,341) [341,682) [682,1024) for 1024 rows over 3 GPUs."""
    _, M, bounds, _, _ = load_fig3(golden_dir)
    assert partition(1024, M, FLOOR) == bounds


def test_fig3_task_list(golden_dir):
    """PAPER.md:144 prints every keep / reload / P2P interval of the example."""
    old, M, bounds, tasks, reload_total = load_fig3(golden_dir)
    got, new_layout = cmm_plan(old, M)
    assert got == sorted(tasks, key=lambda t: (t[2], t[3]))
    assert [(s, e) for (_, s, e, _) in new_layout] == list(zip(bounds[:-1], bounds[1:]))
    assert [r for (r, _, _, _) in new_layout] == [0, 2, 3]
    st = plan_stats(got)
    assert st["reload_units"] == reload_total == 256       # "Only 256 rows are reloaded"
    assert st["transfer_units"] == 86 and st["keep_units"] == 682
    assert eq1_reload_lower_bound(old, bounds) == 256


@pytest.mark.parametrize("policy", [FLOOR, CEIL_FIRST])
def test_partition_widths_floor_or_ceil(policy):
    """every shard holds floor(S/g) or ceil(S/g); widths sum to S; any g is valid."""
    for S in list(range(1, 70)) + [688, 1024, 14336, 17408, 128256, 151936]:
        for M in range(1, min(S, 9) + 1):
            b = partition(S, M, policy)
            w = [b[i + 1] - b[i] for i in range(M)]
            assert b[0] == 0 and b[-1] == S and len(b) == M + 1
            assert set(w) <= {S // M, -(-S // M)}
            assert sum(w) == S
            assert w.count(-(-S // M)) == (S % M if S % M else M)


def test_partition_policies_on_baseline_config2():
    """BASELINE.json config 2: '(KV heads split 3/3/2)'; the paper's floor formula gives 2/3/3."""
    w = lambda b: [b[i + 1] - b[i] for i in range(len(b) - 1)]
    assert w(partition(8, 3, CEIL_FIRST)) == [3, 3, 2]
    assert w(partition(8, 3, FLOOR)) == [2, 3, 3]
    assert w(partition(17408, 3, CEIL_FIRST)) == [5803, 5803, 5802]
    assert w(partition(8, 7, FLOOR)) == [1, 1, 1, 1, 1, 1, 2]       # config 3: 8 KV heads over 7 ranks


def test_partition_align_and_errors():
    b = partition(100, 3, FLOOR, align_units=8)
    assert b[0] == 0 and b[-1] == 100 and all(x % 8 == 0 for x in b[:-1])
    with pytest.raises(ValueError):
        partition(2, 3)
    with pytest.raises(ValueError):
        partition(8, 0)


def random_layout(rng, max_n=8, max_h=4000, dead=None):
    n = rng.randint(2, max_n)
    widths = [rng.randint(0 if rng.random() < 0.1 else 1, max(1, max_h // n)) for _ in range(n)]
    if sum(widths) == 0:
        widths[0] = 1
    lay = layout_from_widths(widths)
    k = dead if dead is not None else rng.randint(1, min(2, n - 1))
    dead_ranks = set(rng.sample(range(n), k))
    return [(r, s, e, 0 if r in dead_ranks else 1) for (r, s, e, _) in lay]


def check_invariants(old, M, tasks, new_layout):
    H = max(e for (_, _, e, _) in old)
    holder = {}
    for (r, s, e, a) in old:
        for u in range(s, e):
            holder.setdefault(u, []).append((r, a))
    covered = {}
    for (kind, src, dst, b, e) in tasks:
        assert b < e
        for u in range(b, e):
            assert u not in covered, "I1: unit sourced twice"
            covered[u] = (kind, src, dst)
    owner_of = {}
    for (r, s, e, _) in new_layout:
        for u in range(s, e):
            owner_of[u] = r
    assert sorted(covered) == list(range(H)) == sorted(owner_of), "I1/I5: targets tile [0,H)"
    for u, (kind, src, dst) in covered.items():
        assert dst == owner_of[u]
        alive_holders = [r for (r, a) in holder.get(u, []) if a]
        if dst in alive_holders:
            assert kind == KEEP and src == dst, "I2: retained units never move"
        elif alive_holders:
            assert kind == TRANSFER and src in alive_holders and src != dst, "I4: source alive and holds unit"
        else:
            assert kind == RELOAD and src == -1, "I3: reload only what no survivor holds"


def test_invariants_and_eq1_random():
    """north_star invariants + Eq. 1: reload units == H - sum_i sum_j |src_i ∩ tgt_j|."""
    rng = random.Random(11617)
    for _ in range(300):
        old = random_layout(rng, max_h=300)
        n_alive = sum(a for (_, _, _, a) in old)
        H = max(e for (_, _, e, _) in old)
        M = rng.randint(1, n_alive)
        if H < M:
            continue
        policy = rng.choice([FLOOR, CEIL_FIRST])
        tb = partition(H, M, policy)
        tasks, new_layout = cmm_plan(old, M, tb)
        check_invariants(old, M, tasks, new_layout)
        st = plan_stats(tasks)
        assert st["reload_units"] == eq1_reload_lower_bound(old, tb)
        assert st["total_units"] == H
        assert cmm_plan(old, M, tb)[0] == tasks          # deterministic
        # default targets are the floor formula of Alg. 1 l.2-5
        assert cmm_plan(old, M)[0] == cmm_plan(old, M, partition(H, M, FLOOR))[0]


def test_bruteforce_minimality_tiny():
    """PAPER.md:152/:160 'guarantees a minimal total reload volume' — exhaustive enumeration, H <= 10."""
    rng = random.Random(7)
    n_checked = 0
    for _ in range(120):
        n = rng.randint(2, 5)
        H = rng.randint(n, 10)
        cuts = sorted(rng.sample(range(1, H), n - 1)) if n > 1 else []
        lay = layout_from_bounds([0] + cuts + [H])
        dead = set(rng.sample(range(n), rng.randint(1, min(2, n - 1))))
        old = [(r, s, e, 0 if r in dead else 1) for (r, s, e, _) in lay]
        M = n - len(dead)
        if H < M:
            continue
        tb = partition(H, M, rng.choice([FLOOR, CEIL_FIRST]))
        tasks, new_layout = cmm_plan(old, M, tb)
        st = plan_stats(tasks)
        owners = [r for (r, _, _, _) in new_layout]
        assert (st["reload_units"], st["transfer_units"]) == bruteforce.min_cost_given_owners(old, tb, owners)
        n_checked += 1
    assert n_checked > 80


def test_bruteforce_with_replicated_sources():
    """Reading C7: overlapping (replicated) alive sources — owner first, then ascending rank id."""
    old = [(0, 0, 6, 1), (1, 4, 8, 1), (2, 6, 10, 0), (3, 2, 5, 1)]
    for M in (1, 2, 3):
        tb = partition(10, M)
        tasks, new_layout = cmm_plan(old, M, tb)
        check_invariants(old, M, tasks, new_layout)
        st = plan_stats(tasks)
        owners = [r for (r, _, _, _) in new_layout]
        assert (st["reload_units"], st["transfer_units"]) == bruteforce.min_cost_given_owners(old, tb, owners)


def test_in_order_ownership_is_not_always_transfer_minimal():
    """Reading C11 (reported, not required): N=4, H=4, rank 0 dead — in-order owners transfer 2 units,
    the best owner permutation transfers 1.  'Minimal' in the paper covers reload units only."""
    old = [(0, 0, 1, 0), (1, 1, 2, 1), (2, 2, 3, 1), (3, 3, 4, 1)]
    tb = partition(4, 3)
    tasks, new_layout = cmm_plan(old, 3, tb)
    st = plan_stats(tasks)
    assert (st["reload_units"], st["transfer_units"]) == (1, 2)
    best = bruteforce.best_over_owner_permutations(old, tb)
    assert min(best.values()) == (1, 1)
    assert all(c[0] == 1 for c in best.values())      # reload minimum is permutation-independent (Eq. 1)


def test_migration_aware_plan_against_unit_level_bruteforce():
    """Reading M1: the search over owners and wide-shard placements reaches exactly the minimum that
    oracle/bruteforce.py finds by enumerating a source for every single unit under every owner permutation and every
    bounds vector with widths in {floor, ceil} - no intervals, no Algorithm 1 on that side."""
    import itertools
    from oracle.planning import migration_aware_plan, width_arrangements
    rng = random.Random(17)
    improved = n_checked = 0
    for _ in range(60):
        n = rng.randint(2, 4)
        H = rng.randint(n, 8)
        cuts = sorted(rng.sample(range(1, H), n - 1))
        lay = layout_from_bounds([0] + cuts + [H])
        dead = set(rng.sample(range(n), 1))
        old = [(r, s, e, 0 if r in dead else 1) for (r, s, e, _) in lay]
        M = n - 1
        if H < M:
            continue
        tasks, new = migration_aware_plan(old, M)
        check_invariants(old, M, tasks, new)
        st = plan_stats(tasks)
        got = (st["reload_units"], st["transfer_units"])
        # every bounds vector the definition admits: q/q+1 widths, sum H
        arrs = width_arrangements(H, M)
        q, r = divmod(H, M)
        assert len(arrs) == len(set(map(tuple, arrs))) == len(list(itertools.combinations(range(M), r)))
        assert all(b[0] == 0 and b[-1] == H and all(b[j + 1] - b[j] in (q, q + 1) for j in range(M)) for b in arrs)
        brute = min(min(bruteforce.best_over_owner_permutations(old, tb).values()) for tb in arrs)
        assert got == brute
        base = plan_stats(cmm_plan(old, M)[0])
        assert got[0] == base["reload_units"] and got[1] <= base["transfer_units"]
        improved += got[1] < base["transfer_units"]
        n_checked += 1
    assert n_checked > 40 and improved > 5


def test_migration_aware_plan_worked_example_and_ties():
    from oracle.planning import migration_aware_plan
    # the C11 example: N=4, H=4, rank 0 dead.  In-order floor bounds 0/1/2/4 transfer 2 units; with the bounds fixed the best
    # owners transfer 1; letting the wide shard go first (0/2/3/4) every survivor keeps its unit and rank 1 reloads unit 0.
    old = [(0, 0, 1, 0), (1, 1, 2, 1), (2, 2, 3, 1), (3, 3, 4, 1)]
    tasks, new = migration_aware_plan(old, 3, partition(4, 3))
    assert plan_stats(tasks)["transfer_units"] == 1
    tasks, new = migration_aware_plan(old, 3)
    assert new == [(1, 0, 2, 1), (2, 2, 3, 1), (3, 3, 4, 1)]
    assert tasks == [(RELOAD, -1, 1, 0, 1), (KEEP, 1, 1, 1, 2), (KEEP, 2, 2, 2, 3), (KEEP, 3, 3, 3, 4)]
    # nothing to gain: an intact formula layout keeps everything and the tie goes to the smallest (bounds, owners)
    lay = layout_from_bounds(partition(10, 3))
    tasks, new = migration_aware_plan(lay, 3)
    assert new == lay and all(k == KEEP for (k, _, _, _, _) in tasks)
    # fixed bounds: only the owners move
    old = [(0, 0, 4, 1), (1, 4, 8, 0), (2, 8, 12, 1), (3, 12, 16, 1)]
    tasks, new = migration_aware_plan(old, 3, [0, 5, 11, 16])
    assert [b for (_, b, _, _) in new] == [0, 5, 11]


def test_table2_ordering_in_units():
    """PAPER.md:204 / Table II: reload(Full) >= reload(Greedy) >= reload(CM); P2P only in CM."""
    rng = random.Random(3)
    strict = 0
    for _ in range(100):
        old = random_layout(rng, max_h=500, dead=1)
        M = sum(a for (_, _, _, a) in old)
        H = max(e for (_, _, e, _) in old)
        if H < M:
            continue
        cm = plan_stats(cmm_plan(old, M)[0])
        gr = plan_stats(greedy_plan(old, M)[0])
        fu = plan_stats(full_reload_plan(old, M)[0])
        assert fu["reload_units"] == H and fu["transfer_units"] == 0 and fu["keep_units"] == 0
        assert gr["transfer_units"] == 0 and gr["keep_units"] == cm["keep_units"]
        assert fu["reload_units"] >= gr["reload_units"] >= cm["reload_units"]
        assert gr["reload_units"] == cm["reload_units"] + cm["transfer_units"]
        strict += cm["transfer_units"] > 0
    assert strict > 50


def test_survey_config1_ffn_numbers():
    """Config 1 (BASELINE.json): explicit unequal old FFN widths 160/176/184/168, rank 2 dies, 3 ranks.
    Worked independently in SURVEY.md §8(d): keep 435, P2P 69 (rank 1->0 [160,229)), reload 184
    ([336,458)->rank 1, [458,520)->rank 3)."""
    old = [(r, s, e, 0 if r == 2 else 1) for (r, s, e, _) in layout_from_widths([160, 176, 184, 168])]
    tasks, new_layout = cmm_plan(old, 3)
    assert [(s, e) for (_, s, e, _) in new_layout] == [(0, 229), (229, 458), (458, 688)]
    st = plan_stats(tasks)
    assert (st["keep_units"], st["transfer_units"], st["reload_units"]) == (435, 69, 184)
    assert (TRANSFER, 1, 0, 160, 229) in tasks
    assert (RELOAD, -1, 1, 336, 458) in tasks and (RELOAD, -1, 3, 458, 520) in tasks


def test_sequential_failures_config5_units():
    """Config 5a: Llama-3-8B FFN 14336, equal widths, failures 5 then 0 then 7;
    per step keep/P2P/reload = 9728/2816/1792; 7166/5122/2048; 7168/4778/2390."""
    lay = layout_from_bounds(partition(14336, 8))
    expect = [(9728, 2816, 1792), (7166, 5122, 2048), (7168, 4778, 2390)]
    for dead, exp in zip((5, 0, 7), expect):
        old = [(r, s, e, 0 if r == dead else 1) for (r, s, e, _) in lay]
        tasks, lay = cmm_plan(old, len(lay) - 1)
        st = plan_stats(tasks)
        assert (st["keep_units"], st["transfer_units"], st["reload_units"]) == exp


def test_errors_and_edge_cases():
    old = layout_from_widths([4, 4, 4])
    with pytest.raises(ValueError):
        cmm_plan([(0, 0, 4, 1), (1, 4, 8, 0)], 2)        # M > #alive (reading C6)
    with pytest.raises(ValueError):
        cmm_plan(old, 3, [0, 4, 8, 11])                    # bounds must end at H
    # no failure, same M: everything is kept
    tasks, _ = cmm_plan(old, 3)
    assert all(k == KEEP for (k, *_r) in tasks)
    # a joining (repaired) GPU appears as an alive rank with an empty interval (reading C6): scale-up 2 -> 3
    old = [(0, 0, 6, 1), (1, 6, 12, 1), (2, 12, 12, 1)]
    tasks, new_layout = cmm_plan(old, 3)
    st = plan_stats(tasks)
    assert st["reload_units"] == 0 and st["transfer_units"] == 2 + 4 and [r for (r, *_x) in new_layout] == [0, 1, 2]
    # two dead, non-adjacent ranks -> a target can have two reload gaps (reading C5)
    old = [(0, 0, 2, 0), (1, 2, 4, 1), (2, 4, 6, 0), (3, 6, 8, 1)]
    tasks, _ = cmm_plan(old, 1)
    assert [(k, b, e) for (k, _, _, b, e) in tasks] == [(RELOAD, 0, 2), (KEEP, 2, 4), (RELOAD, 4, 6), (TRANSFER, 6, 8)]


# ------------------------------------------------------------------------------------------ link-cost weights (reading M2)
def two_island_cost(n, island, far):
    """link_cost[src][dst]: 1 inside an island of `island` consecutive ranks, `far` across islands."""
    return [[0 if a == b else (1 if a // island == b // island else far) for b in range(n)] for a in range(n)]


def test_weighted_migration_aware_plan_against_unit_level_bruteforce():
    """Reading M2 ("incorporating link reachability and cost weighting into planning"): the weighted planner's
    (reload, weighted transfer cost) equals the minimum, over every owner permutation and every {floor, ceil} bounds vector, of
    the UNIT-LEVEL brute force that prices every unit's source by its link - no intervals, no Algorithm 1."""
    import itertools
    from oracle import bruteforce as BF
    rng = random.Random(20)
    checked = 0
    while checked < 25:
        n = rng.randint(3, 4)
        Hn = rng.randint(n, 8)
        cuts = sorted(rng.sample(range(1, Hn), n - 1)) if Hn > n else list(range(1, n))
        b = [0] + cuts + [Hn]
        dead = rng.randrange(n)
        old = [(r, b[r], b[r + 1], 0 if r == dead else 1) for r in range(n)]
        M = n - 1
        if Hn < M:
            continue
        cost = [[0 if a == c else rng.randint(1, 5) for c in range(n)] for a in range(n)]
        tasks, new = migration_aware_plan(old, M, None, cost)
        st = plan_stats(tasks)
        got = (st["reload_units"], weighted_transfer_cost(tasks, cost))
        alive = [r for (r, _, _, a) in old if a]
        best = min(BF.min_weighted_cost_given_owners(old, tb, owners, cost)
                   for tb in width_arrangements(Hn, M) for owners in itertools.permutations(alive, M))
        assert got == best, (old, cost, got, best)
        checked += 1


def test_weighted_plan_prefers_cheap_links_and_uniform_costs_change_nothing():
    # two NVLink islands {0,1,2,3} and {4,5,6,7}; rank 3 dies; 7 targets over 56 units
    old = [(r, 7 * r, 7 * r + 7, 0 if r == 3 else 1) for r in range(8)]
    uniform = two_island_cost(8, 8, 1)
    islands = two_island_cost(8, 4, 16)
    base = migration_aware_plan(old, 7)
    assert migration_aware_plan(old, 7, None, uniform) == base                      # one NVSwitch node: the result to state
    tasks, new = migration_aware_plan(old, 7, None, islands)
    assert plan_stats(tasks)["reload_units"] == plan_stats(base[0])["reload_units"] == 7
    assert weighted_transfer_cost(tasks, islands) <= weighted_transfer_cost(base[0], islands)
    # replicated sources (C7 -> M2): the cheaper holder supplies the unit
    rep = [(0, 0, 4, 1), (1, 0, 4, 1), (2, 4, 8, 1), (3, 8, 8, 1)]
    cost = [[0, 9, 9, 9], [9, 0, 9, 1], [9, 9, 0, 9], [9, 9, 9, 0]]
    t, _ = cmm_plan(rep, 4, [0, 2, 4, 6, 8], owners=[0, 3, 2, 1], link_cost=cost)
    assert (TRANSFER, 1, 3, 2, 4) in t                                              # rank 3 pulls [2,4) from rank 1 (cost 1), not rank 0 (9)
