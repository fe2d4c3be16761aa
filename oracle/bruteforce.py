"""ORACLE (test infrastructure) — exhaustive check of "minimal" on tiny instances.

PAPER.md:152/:160 claim the CMM plan "guarantees a minimal total reload volume".  This module makes no
use of intervals or of Algorithm 1: it enumerates EVERY assignment of a source to every unit of every
target — source in {each alive rank that holds the unit} ∪ {host} — and returns the lexicographic
minimum of (reloaded units, transferred units).  Exponential; for H <= ~12 only.
"""
from __future__ import annotations

import itertools
from typing import Dict, List, Sequence, Tuple

HOST = -1


def _holders(old_layout, u) -> List[int]:
    return [r for (r, s, e, alive) in old_layout if alive and s <= u < e]


def min_cost_given_owners(old_layout, target_bounds: Sequence[int], owners: Sequence[int]) -> Tuple[int, int]:
    """Enumerate all source assignments; owners[j] = rank that will hold target j."""
    units = []   # (owner, [feasible sources])
    for j in range(len(target_bounds) - 1):
        for u in range(target_bounds[j], target_bounds[j + 1]):
            units.append((owners[j], _holders(old_layout, u) + [HOST]))
    best = None
    for choice in itertools.product(*[srcs for (_, srcs) in units]):
        reload_units = sum(1 for c in choice if c == HOST)
        transfer_units = sum(1 for (own, _), c in zip(units, choice) if c != HOST and c != own)
        cost = (reload_units, transfer_units)
        if best is None or cost < best:
            best = cost
    return best


def min_weighted_cost_given_owners(old_layout, target_bounds: Sequence[int], owners: Sequence[int], link_cost) -> Tuple[int, int]:
    """Same enumeration with a per-link price (reading M2): minimum of (reloaded units, sum over transferred units of
    link_cost[source][owner]).  No intervals, no Algorithm 1."""
    units = []
    for j in range(len(target_bounds) - 1):
        for u in range(target_bounds[j], target_bounds[j + 1]):
            units.append((owners[j], _holders(old_layout, u) + [HOST]))
    best = None
    for choice in itertools.product(*[srcs for (_, srcs) in units]):
        reload_units = sum(1 for c in choice if c == HOST)
        cost = sum(link_cost[c][own] for (own, _), c in zip(units, choice) if c != HOST and c != own)
        if best is None or (reload_units, cost) < best:
            best = (reload_units, cost)
    return best


def best_over_owner_permutations(old_layout, target_bounds: Sequence[int]) -> Dict[Tuple[int, ...], Tuple[int, int]]:
    """Same, for every injective choice of owners among the alive ranks (reading C11: reported, not required)."""
    alive = sorted(r for (r, _, _, a) in old_layout if a)
    M = len(target_bounds) - 1
    out = {}
    for owners in itertools.permutations(alive, M):
        out[owners] = min_cost_given_owners(old_layout, target_bounds, owners)
    return out
