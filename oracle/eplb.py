"""ORACLE (test infrastructure) — EPLB-style expert replica placement after an elastic reshard.

PAPER.md:172-174 (Fig. 4 and the paragraph under it): "the system applies an EPLB-like dynamic load balancing strategy
... replicating hot-spot experts and adjusting routing ... the new parameter sharding might leave one GPU with a smaller
shard and thus more idle compute capacity ... an intelligent EPLB planner detects this heterogeneity and schedules more
expert replicas to the under-utilized GPU. This results in a new state that, while not arithmetically balanced in terms of
request count, is performance-optimal"; Fig. 4(c): "places the recovered Expert 1 and new replicas of the hotspot Expert 0
onto the most idle GPU (GPU 3)".  The paper gives no algorithm; what follows is DESIGN.md reading E1, step by step, in exact
integer arithmetic (plain Python ints and Fractions, no numpy):

  inputs   load[e]      tokens routed to expert e (>= 0)
           home[e]      the rank that holds expert e after the reshard (the expert-granularity plan), or -1 for an expert
                        that has no holder yet (Fig. 4's "recovered" expert)
           capacity[r]  compute available for expert work on rank r (> 0 for a usable rank, 0 for a dead one); unequal
                        after an unequal-width reshard
           slots[r]     spare expert slots of rank r (slab slack)
  notion   an expert with k instances sends load[e] / k to each of them (routing is adjusted evenly);
           L(r) = (sum over instances on r of load[e] / k_e) / capacity[r]   - the normalised load of rank r
  step 1   homeless experts, in descending load (tie: lower id): to the usable rank with a spare slot whose normalised load
           AFTER taking the expert is smallest (tie: lower rank id).
  step 2   repeat: let cur = max_r L(r) and hot = the lowest rank attaining it.  Over every expert e with an instance on
           hot (k_e < MAX_INSTANCES) and every usable rank d with a spare slot that does not hold e yet, evaluate the
           maximum normalised load after adding an instance of e on d; take the smallest (tie: lower e, then lower d).
           If it is not strictly below cur, stop; else create that replica.
  output   the replicas in creation order [(expert, rank)], and instances[e] = [home, replica ranks in creation order].

Routing convention used by the kernels' harness: an expert with n routed rows and k instances gives instance j the rows
[floor(j * n / k), floor((j + 1) * n / k)) of its row block.
"""
from __future__ import annotations

from fractions import Fraction
from typing import Dict, List, Sequence, Tuple

MAX_INSTANCES = 8      # per expert, home included


def rank_loads(load: Sequence[int], instances: Sequence[Sequence[int]], n_ranks: int) -> List[Fraction]:
    """Un-normalised load per rank: sum over the instances it hosts of load[e] / k_e."""
    out = [Fraction(0)] * n_ranks
    for e, ranks in enumerate(instances):
        for r in ranks:
            out[r] += Fraction(load[e], len(ranks))
    return out


def max_normalised(load, instances, capacity) -> Fraction:
    S = rank_loads(load, instances, len(capacity))
    return max((S[r] / capacity[r] for r in range(len(capacity)) if capacity[r] > 0), default=Fraction(0))


def place(load: Sequence[int], home: Sequence[int], capacity: Sequence[int], slots: Sequence[int]
          ) -> Tuple[List[Tuple[int, int]], List[List[int]]]:
    E, R = len(load), len(capacity)
    if len(home) != E or len(slots) != R:
        raise ValueError("length mismatch")
    if any(v < 0 for v in load) or any(c < 0 for c in capacity) or any(s < 0 for s in slots):
        raise ValueError("negative input")
    for e in range(E):
        if home[e] != -1 and not (0 <= home[e] < R and capacity[home[e]] > 0):
            raise ValueError("home must be a usable rank or -1")
    free = list(slots)
    instances: List[List[int]] = [[home[e]] if home[e] >= 0 else [] for e in range(E)]
    replicas: List[Tuple[int, int]] = []
    # step 1: homeless experts to the most idle rank
    for e in sorted((e for e in range(E) if home[e] < 0), key=lambda e: (-load[e], e)):
        S = rank_loads(load, instances, R)
        cands = [d for d in range(R) if capacity[d] > 0 and free[d] > 0]
        if not cands:
            raise ValueError("no spare slot for a homeless expert")
        d = min(cands, key=lambda d: ((S[d] + load[e]) / capacity[d], d))
        instances[e].append(d)
        free[d] -= 1
        replicas.append((e, d))
    # step 2: replicate what sits on the hottest rank while that lowers the maximum
    while True:
        S = rank_loads(load, instances, R)
        usable = [r for r in range(R) if capacity[r] > 0]
        cur = max(S[r] / capacity[r] for r in usable)
        hot = min(r for r in usable if S[r] / capacity[r] == cur)
        best = None
        for e in range(E):
            if hot not in instances[e] or len(instances[e]) >= MAX_INSTANCES:
                continue
            for d in usable:
                if free[d] <= 0 or d in instances[e]:
                    continue
                trial = [list(x) for x in instances]
                trial[e].append(d)
                key = (max_normalised(load, trial, capacity), e, d)
                if best is None or key < best:
                    best = key
        if best is None or best[0] >= cur:
            break
        _, e, d = best
        instances[e].append(d)
        free[d] -= 1
        replicas.append((e, d))
    return replicas, instances


def split_rows(n_rows: int, k: int) -> List[Tuple[int, int]]:
    """Rows of one expert's block over its k instances (even routing): instance j gets [floor(j n / k), floor((j+1) n / k))."""
    return [((j * n_rows) // k, ((j + 1) * n_rows) // k) for j in range(k)]


def replica_slots(shards: Sequence[Tuple[int, int, int, int]], geom: Dict[int, Tuple[int, int]], replicas: Sequence[Tuple[int, int]]) -> List[int]:
    """Where a replica lives (reading E1, memory side): rank d keeps unit u of its shard at slot (u - anchor) mod cap (reading
    L3); a replica takes the LOWEST slot of d's slab that holds no unit of d's current shard and no earlier replica.
    shards: [(rank, begin, end, alive)] of the expert class; geom[rank] = (anchor, cap)."""
    taken = {r: set() for r in geom}
    for (r, b, e, alive) in shards:
        if alive:
            for u in range(b, e):
                taken[r].add((u - geom[r][0]) % geom[r][1])
    out = []
    for (e, d) in replicas:
        s = next(s for s in range(geom[d][1]) if s not in taken[d])
        taken[d].add(s)
        out.append(s)
    return out
