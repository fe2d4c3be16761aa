"""ORACLE (test infrastructure) — S1 partition and S2 Continuous Minimal Migration plan.

Written from PAPER.md §III-B (:92-94), Algorithm 1 (:98-140), the prose of §III-C (:152),
Fig. 3 (:144) and Eq. 1 (:154-160).  Pure Python integers; no numpy, no blocking, no reordering.
Ranks are 0-based here (Fig. 3 is 1-based: "GPU:2" = rank 1).

Readings of garbled / silent passages are those of DESIGN.md ("Readings"):
  C1  Alg.1 l.11 prints AddTransferPlan(inter, gpu_i, gpu_i); read (inter, src=gpu_i, dst=gpu_j)  [Fig. 3]
  C2  Alg.1 l.18 prints AddReloadPlan(tar_range, gpu_i);      read dst=gpu_j                      [Fig. 3]
  C3  target j is owned by the j-th ALIVE rank in ascending rank id                               [Fig. 3]
  C4  a "transfer" whose source is the owner itself is a KEEP (no byte moves)                     [Fig. 3 "keeps"]
  C5  tar_range after subtraction may be several gaps -> one RELOAD per maximal gap, ascending
  C7  replicated sources: the owner itself first, then ascending rank id
"""
from __future__ import annotations

from typing import List, Optional, Sequence, Tuple

FLOOR = "floor"            # Alg.1 l.2-5: boundary_j = floor(j*H/M)           (the paper's definition)
CEIL_FIRST = "ceil_first"  # first (H mod M) shards get ceil(H/M)             (BASELINE.json config 2: 3/3/2)

KEEP, TRANSFER, RELOAD = 0, 1, 2

Shard = Tuple[int, int, int, int]        # (rank, begin, end, alive)    = (gpu_i, s_i, e_i, alive_i)
Task = Tuple[int, int, int, int, int]    # (kind, src_rank, dst_rank, begin, end); src_rank = -1 for RELOAD


def partition(total_units: int, parts: int, policy: str = FLOOR, align_units: int = 1) -> List[int]:
    """Bounds b_0..b_M of an unequal-width split of S units over g_t = M shards.

    PAPER.md:94 — "some GPUs hold shard size floor(S/g_t) while others hold ceil(S/g_t)".
    FLOOR      : b_j = floor(j*S/M)                       (Alg. 1 l.3-4; Fig. 3 0/341/682/1024)
    CEIL_FIRST : widths ceil(S/M) for the first S mod M shards, floor(S/M) after
    align_units > 1 (paper silent; reading P5): split ceil(S/align) super-units, scale, clip the end to S.
    """
    S, M, a = int(total_units), int(parts), int(align_units)
    if M < 1 or S < 0 or a < 1:
        raise ValueError("bad partition arguments")
    n = -(-S // a)   # super-units
    if n < M:
        raise ValueError("fewer units than shards (replication is out of scope, reading P4)")
    if policy == FLOOR:
        b = [(j * n) // M for j in range(M + 1)]
    elif policy == CEIL_FIRST:
        q, r = divmod(n, M)
        b = [0]
        for j in range(M):
            b.append(b[-1] + q + (1 if j < r else 0))
    else:
        raise ValueError("unknown policy")
    return [min(x * a, S) for x in b]


def layout_from_bounds(bounds: Sequence[int], ranks: Optional[Sequence[int]] = None,
                       alive: Optional[Sequence[int]] = None) -> List[Shard]:
    n = len(bounds) - 1
    ranks = list(range(n)) if ranks is None else list(ranks)
    alive = [1] * n if alive is None else list(alive)
    return [(ranks[i], bounds[i], bounds[i + 1], int(alive[i])) for i in range(n)]


def layout_from_widths(widths: Sequence[int]) -> List[Shard]:
    b = [0]
    for w in widths:
        b.append(b[-1] + int(w))
    return layout_from_bounds(b)


def _subtract(rest: List[Tuple[int, int]], a: int, b: int) -> List[Tuple[int, int]]:
    """rest \\ [a,b) for a sorted list of disjoint half-open intervals."""
    out = []
    for (x, y) in rest:
        if b <= x or y <= a:
            out.append((x, y))
            continue
        if x < a:
            out.append((x, a))
        if b < y:
            out.append((b, y))
    return out


def cmm_plan(old_layout: Sequence[Shard], M: int, target_bounds: Optional[Sequence[int]] = None,
             owners: Optional[Sequence[int]] = None, link_cost=None) -> Tuple[List[Task], List[Shard]]:
    """Algorithm 1 with readings C1-C7.  Returns (tasks sorted by (dst, begin), new layout).
    ``owners`` (reading M1, not in the paper): owners[j] = the alive rank that will hold target j, instead of the
    j-th alive rank of reading C3.  ``link_cost`` (reading M2): link_cost[src][dst] = integer cost of moving one unit from
    rank src to rank dst; replicated sources are then tried in ascending (cost to the owner, rank id) instead of rank id."""
    old = [tuple(int(v) for v in s) for s in old_layout]
    if not old:
        raise ValueError("empty layout")
    for (_, s, e, _) in old:
        if s > e or s < 0:
            raise ValueError("bad interval")
    H = max(e for (_, _, e, _) in old)                                   # l.1  H <- max(e_i) for all i
    if target_bounds is None:
        target_bounds = [(j * H) // M for j in range(M + 1)]             # l.2-5
    tb = [int(x) for x in target_bounds]
    if len(tb) != M + 1 or tb[0] != 0 or tb[-1] != H or any(tb[j] > tb[j + 1] for j in range(M)):
        raise ValueError("target bounds must tile [0,H)")
    G = sorted(r for (r, _, _, a) in old if a)                           # C3: alive ranks, ascending id
    if len(set(r for (r, _, _, _) in old)) != len(old):
        raise ValueError("duplicate rank id")
    if M > len(G) or M < 1:
        raise ValueError("M must be in 1..#alive (reading C6)")
    if owners is not None:
        G = [int(r) for r in owners]
        alive_ids = {r for (r, _, _, a) in old if a}
        if len(G) != M or len(set(G)) != M or any(r not in alive_ids for r in G):
            raise ValueError("owners must be M distinct alive ranks")
    alive_sorted = sorted((s for s in old if s[3]), key=lambda s: s[0])
    tasks: List[Task] = []
    for j in range(M):                                                   # l.6
        dst = G[j]
        rest = [(tb[j], tb[j + 1])] if tb[j] < tb[j + 1] else []         # l.7 tar_range
        others = [s for s in alive_sorted if s[0] != dst]
        if link_cost is not None:
            others.sort(key=lambda s: (link_cost[s[0]][dst], s[0]))                                  # M2
        order = [s for s in alive_sorted if s[0] == dst] + others                                    # C7
        for (rank_i, s_i, e_i, _) in order:                              # l.8-9, alive only
            for (x, y) in list(rest):
                a, b = max(x, s_i), min(y, e_i)                          # l.10 inter
                if a < b:                                                # l.11
                    kind = KEEP if rank_i == dst else TRANSFER           # C4
                    tasks.append((kind, rank_i, dst, a, b))              # l.12 (C1: dst = gpu_j)
                    rest = _subtract(rest, a, b)                         # l.13
        for (x, y) in rest:                                              # l.17-18 (C2, C5)
            tasks.append((RELOAD, -1, dst, x, y))
    tasks.sort(key=lambda t: (t[2], t[3]))
    new_layout = [(G[j], tb[j], tb[j + 1], 1) for j in range(M)]
    return tasks, new_layout


MAX_ALIVE_MIGRATION_AWARE = 10


def width_arrangements(H: int, M: int) -> List[List[int]]:
    """Every bounds vector whose widths are floor(H/M) or ceil(H/M) (PAPER.md:94 fixes the widths, not which ranks are
    wide), in lexicographic order."""
    import itertools
    q, r = divmod(H, M)
    out = []
    for wide in itertools.combinations(range(M), r):
        b = [0]
        for j in range(M):
            b.append(b[-1] + q + (1 if j in wide else 0))
        out.append(b)
    return sorted(out)


def weighted_transfer_cost(tasks: Sequence[Task], link_cost) -> int:
    """Sum over TRANSFER tasks of units x link_cost[src][dst] (reading M2; "link reachability and cost weighting")."""
    return sum((e - b) * (1 if link_cost is None else link_cost[s][d]) for (k, s, d, b, e) in tasks if k == TRANSFER)


def migration_aware_plan(old_layout: Sequence[Shard], M: int, target_bounds: Optional[Sequence[int]] = None, link_cost=None):
    """SURVEY.md 8(f) #2 / DESIGN.md reading M1 (an extension; PAPER.md:160 makes only the reload volume minimal and
    :247/:257 leave transfer cost to future work).  Plain definition by exhaustion: over every admissible bounds vector
    (all placements of the wide shards, or the given bounds) and every injective assignment of targets to alive ranks,
    run Algorithm 1 with those owners and take the lexicographic minimum of
        (reload units, transfer units, bounds vector, owners vector).
    With ``link_cost`` (reading M2: PAPER.md:247, :257 leave "link reachability and cost weighting" of the planner to future
    work) the second component is the WEIGHTED transfer cost sum(units x link_cost[src][dst]); uniform costs change nothing.
    Returns (tasks, new layout) like cmm_plan."""
    import itertools
    old = [tuple(int(v) for v in s) for s in old_layout]
    H = max(e for (_, _, e, _) in old)
    alive = sorted(r for (r, _, _, a) in old if a)
    if M < 1 or M > len(alive):
        raise ValueError("M must be in 1..#alive (reading C6)")
    if len(alive) > MAX_ALIVE_MIGRATION_AWARE:
        raise ValueError("migration-aware search is limited to 10 alive ranks")
    if target_bounds is None and H < M:
        raise ValueError("fewer units than shards")
    cands = [list(int(x) for x in target_bounds)] if target_bounds is not None else width_arrangements(H, M)
    best = None
    for tb in cands:
        for owners in itertools.permutations(alive, M):
            tasks, new = cmm_plan(old, M, tb, owners, link_cost)
            st = plan_stats(tasks)
            key = (st["reload_units"], weighted_transfer_cost(tasks, link_cost), tuple(tb), tuple(owners))
            if best is None or key < best[0]:
                best = (key, tasks, new)
    return best[1], best[2]


def greedy_plan(old_layout: Sequence[Shard], M: int, target_bounds: Optional[Sequence[int]] = None):
    """'Greedy' of PAPER.md:204: keep the local overlap; "missing bytes are reloaded from host memory on the
    target GPU and we do not schedule cross-device transfers for those gaps"."""
    tasks, new_layout = cmm_plan(old_layout, M, target_bounds)
    out = [(RELOAD, -1, d, b, e) if k == TRANSFER else (k, s, d, b, e) for (k, s, d, b, e) in tasks]
    return _merge_adjacent(out), new_layout


def full_reload_plan(old_layout: Sequence[Shard], M: int, target_bounds: Optional[Sequence[int]] = None):
    """'Full Reload' of PAPER.md:204: "without data reuse" — every target unit is reloaded."""
    _, new_layout = cmm_plan(old_layout, M, target_bounds)
    return [(RELOAD, -1, r, s, e) for (r, s, e, _) in new_layout if s < e], new_layout


def _merge_adjacent(tasks: List[Task]) -> List[Task]:
    tasks = sorted(tasks, key=lambda t: (t[2], t[3]))
    out: List[Task] = []
    for t in tasks:
        if out and out[-1][0] == t[0] and out[-1][1] == t[1] and out[-1][2] == t[2] and out[-1][4] == t[3]:
            out[-1] = (t[0], t[1], t[2], out[-1][3], t[4])
        else:
            out.append(t)
    return out


def plan_stats(tasks: Sequence[Task]):
    keep = sum(e - b for (k, _, _, b, e) in tasks if k == KEEP)
    xfer = sum(e - b for (k, _, _, b, e) in tasks if k == TRANSFER)
    rel = sum(e - b for (k, _, _, b, e) in tasks if k == RELOAD)
    return {"keep_units": keep, "transfer_units": xfer, "reload_units": rel, "total_units": keep + xfer + rel,
            "n_tasks": len(tasks)}


def eq1_reload_lower_bound(old_layout: Sequence[Shard], target_bounds: Sequence[int]) -> int:
    """Eq. 1, literally: Reload* = H - sum_{i in S} sum_j |[s_i,e_i) ∩ [u_j,v_j)|,
    S = surviving sources (disjoint, as the equation assumes)."""
    H = max(e for (_, _, e, _) in old_layout)
    tot = 0
    for (_, s, e, alive) in old_layout:
        if not alive:
            continue
        for j in range(len(target_bounds) - 1):
            u, v = target_bounds[j], target_bounds[j + 1]
            tot += max(0, min(e, v) - max(s, u))
    return H - tot
