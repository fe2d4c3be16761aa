"""Pins for oracle/eplb.py (reading E1 of PAPER.md:172-174 / Fig. 4): the figure's qualitative outcome on a hand-worked
instance, exhaustive search for the best SINGLE replica on tiny instances, and the invariants of every result."""
import itertools
import random
from fractions import Fraction

import pytest

from oracle import eplb


def test_fig4_recovered_expert_and_hot_replicas_go_to_the_most_idle_gpu():
    """Fig. 4: 4 GPUs, GPU 1 fails; the re-shard leaves GPU 3 with the smaller dense shard = more free compute;
    "EPLB ... places the recovered Expert 1 and new replicas of the hotspot Expert 0 onto the most idle GPU (GPU 3)".
    Hand-worked: loads 60 / 20 / 20 / 10, capacities 2 / 0 / 2 / 3 (GPU 1 dead, GPU 3 has the idle share), two spare slots each.
      step 1  Expert 1 (homeless, load 20): (60+20)/2 = 40 on GPU 0, (20+20)/2 = 20 on GPU 2, (10+20)/3 = 10 on GPU 3 -> GPU 3.
      step 2  L = 30, -, 10, 10: hot = GPU 0 holds only Expert 0; a second instance makes its share 30:
              on GPU 2 -> max(15, 25, 10) = 25; on GPU 3 -> max(15, 10, 20) = 20 -> GPU 3.          [the figure's two placements]
              L = 15, -, 10, 20: hot = GPU 3 (experts 0, 1, 3).  Expert 0 -> GPU 2 (shares 20): max(10, 20, 50/3) = 20;
              Expert 1 -> GPU 0 (shares 10): max(20, 10, 50/3) = 20; Expert 1 -> GPU 2: max(15, 15, 50/3) = 50/3;
              Expert 3 -> GPU 0 (shares 5): max(35/2, 10, 55/3) = 55/3; Expert 3 -> GPU 2: max(15, 25/2, 55/3) = 55/3
              -> Expert 1 -> GPU 2 (50/3 < 20).
              L = 15, -, 15, 50/3: hot = GPU 3.  Expert 0 -> GPU 2: GPU 2 = (20+10+20)/2 = 25; Expert 1 -> GPU 0 (shares 20/3):
              GPU 0 = (30+20/3)/2 = 55/3; Expert 3 -> GPU 0: 35/2; Expert 3 -> GPU 2: (20+10+5)/2 = 35/2 - none below 50/3 -> stop."""
    load, capacity = [60, 20, 20, 10], [2, 0, 2, 3]
    replicas, instances = eplb.place(load, [0, -1, 2, 3], capacity, [2, 0, 2, 2])
    assert replicas[:2] == [(1, 3), (0, 3)]                      # Fig. 4(c)
    assert replicas == [(1, 3), (0, 3), (1, 2)]
    assert instances == [[0, 3], [3, 2], [2], [3]]
    assert eplb.max_normalised(load, instances, capacity) == Fraction(50, 3)
    # "not arithmetically balanced in terms of request count": GPU 3 serves 50 of the 110 tokens, GPU 0 and 2 30 each
    assert eplb.rank_loads(load, instances, 4) == [30, 0, 30, 50]


def brute_best_single_replica(load, home, capacity, slots):
    """Every way of adding ONE instance (any expert, any rank with a slot that lacks it) -> smallest max normalised load."""
    base = [[h] for h in home]
    best = eplb.max_normalised(load, base, capacity)
    for e in range(len(load)):
        for d in range(len(capacity)):
            if capacity[d] > 0 and slots[d] > 0 and d != home[e]:
                trial = [list(x) for x in base]
                trial[e].append(d)
                best = min(best, eplb.max_normalised(load, trial, capacity))
    return best


def test_one_slot_greedy_is_the_exhaustive_optimum():
    rng = random.Random(4)
    for _ in range(300):
        R = rng.randint(2, 4)
        E = rng.randint(R, 7)
        load = [rng.randint(0, 50) for _ in range(E)]
        home = [rng.randrange(R) for _ in range(E)]
        capacity = [rng.randint(1, 4) for _ in range(R)]
        d = rng.randrange(R)
        slots = [1 if r == d else 0 for r in range(R)]
        replicas, instances = eplb.place(load, home, capacity, slots)
        assert len(replicas) <= 1
        assert eplb.max_normalised(load, instances, capacity) == brute_best_single_replica(load, home, capacity, slots)


def test_invariants_random():
    rng = random.Random(5)
    for _ in range(200):
        R = rng.randint(2, 6)
        E = rng.randint(1, 12)
        load = [rng.randint(0, 1000) for _ in range(E)]
        capacity = [rng.randint(0, 5) for _ in range(R)]
        if not any(capacity):
            capacity[0] = 1
        usable = [r for r in range(R) if capacity[r] > 0]
        home = [rng.choice(usable) for _ in range(E)]
        slots = [rng.randint(0, 3) for _ in range(R)]
        replicas, instances = eplb.place(load, home, capacity, slots)
        before = eplb.max_normalised(load, [[h] for h in home], capacity)
        after = eplb.max_normalised(load, instances, capacity)
        assert after <= before                                     # replication never hurts; every step strictly lowers the maximum
        used = [0] * R
        for (e, d) in replicas:
            used[d] += 1
            assert capacity[d] > 0
        assert all(used[r] <= slots[r] for r in range(R))          # spare slots respected
        for e, ranks in enumerate(instances):
            assert ranks[0] == home[e] and len(set(ranks)) == len(ranks) <= eplb.MAX_INSTANCES   # home first, no rank twice
        assert sum(eplb.rank_loads(load, instances, R)) == sum(load)                              # every token is served once
        # prefix property: each replica was an improvement when it was made
        inst = [[h] for h in home]
        cur = before
        for (e, d) in replicas:
            inst[e].append(d)
            nxt = eplb.max_normalised(load, inst, capacity)
            assert nxt < cur
            cur = nxt


def test_split_rows_and_errors():
    assert eplb.split_rows(10, 3) == [(0, 3), (3, 6), (6, 10)]
    assert eplb.split_rows(2, 4) == [(0, 0), (0, 1), (1, 1), (1, 2)]
    assert eplb.split_rows(0, 2) == [(0, 0), (0, 0)]
    with pytest.raises(ValueError):
        eplb.place([1], [0], [0], [1])            # home on a dead rank
    with pytest.raises(ValueError):
        eplb.place([1], [-1], [1], [0])           # homeless expert, no slot
    assert eplb.place([5, 5], [0, 1], [1, 1], [4, 4]) == ([], [[0], [1]])      # balanced: nothing to do


def test_replica_slots_hand_worked():
    # rank 0: anchor 0, cap 5, shard [0,3) -> slots 0 1 2 taken; rank 1: anchor 3, cap 4, shard [2,5): slots (2-3)%4=3, 0, 1 taken
    geom = {0: (0, 5), 1: (3, 4)}
    shards = [(0, 0, 3, 1), (1, 2, 5, 1)]
    assert eplb.replica_slots(shards, geom, [(4, 0), (0, 1), (3, 0)]) == [3, 2, 4]
    with pytest.raises(StopIteration):
        eplb.replica_slots(shards, geom, [(0, 1), (1, 1)])            # rank 1 has one spare slot only
