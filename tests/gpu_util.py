"""GPU-side test plumbing: device buffers with guard bands, pinned host images, the C-ABI "side" of the harness.
No method arithmetic here."""
from __future__ import annotations

from typing import Dict, Optional

import numpy as np
import torch

import paper_2511_11617_b200 as etp

GUARD = 256
GUARD_BYTE = 0xA5


class LibSide:
    """partition / plan through the C ABI (same interface as harness.OracleSide).  Every answer of the library is compared
    with the oracle's on the spot, so a world built with this side proves S1 / S2 on the GPU box too (`-m gpu` deselects the
    host-only parity tests of tests/test_lib_host.py): a wrong library plan fails here, not silently in the expected image."""
    name = "libetp"

    @staticmethod
    def partition(H, M, policy="floor", align=1):
        from oracle import planning as OP
        got = etp.etp_partition(H, M, policy, align)
        assert got == OP.partition(H, M, policy, align), f"etp_partition({H}, {M}, {policy}) differs from the oracle"
        return got

    @staticmethod
    def plan(old, M, tb=None):
        from oracle import planning as OP
        p = etp.etp_cmm_plan(old, M, tb)
        tasks, new = p.tasks(), p.new_layout()
        o_tasks, o_new = OP.cmm_plan(old, M, tb)
        assert [tuple(t) for t in tasks] == [tuple(t) for t in o_tasks], "etp_cmm_plan: task list differs from oracle.planning.cmm_plan"
        assert [tuple(s) for s in new] == [tuple(s) for s in o_new], "etp_cmm_plan: new layout differs from oracle.planning.cmm_plan"
        return tasks, new


class DevBuf:
    """uint8 device buffer [GUARD | payload | GUARD]; payload pointer is 256-B aligned."""

    def __init__(self, payload: np.ndarray):
        n = int(payload.size)
        self.n = n
        self.t = torch.full((GUARD + n + GUARD,), GUARD_BYTE, dtype=torch.uint8, device="cuda")
        if n:
            self.t[GUARD:GUARD + n] = torch.from_numpy(np.ascontiguousarray(payload)).cuda()

    @property
    def ptr(self) -> int:
        return self.t.data_ptr() + GUARD

    def payload(self) -> np.ndarray:
        return self.t[GUARD:GUARD + self.n].cpu().numpy()

    def guards_intact(self) -> bool:
        g = self.t.cpu().numpy()
        return bool((g[:GUARD] == GUARD_BYTE).all() and (g[GUARD + self.n:] == GUARD_BYTE).all())


def pinned(a: np.ndarray) -> torch.Tensor:
    t = torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    assert t.data_ptr() % 16 == 0
    return t


class Streams:
    def __init__(self):
        self.copy = torch.cuda.Stream()
        self.reload = torch.cuda.Stream()

    def sync(self):
        self.copy.synchronize()
        self.reload.synchronize()


def make_plans(step, mode: int = 0) -> Dict[str, "etp.Plan"]:
    """One plan handle per granularity class, from the step's old layout and new bounds (mode: etp.PLAN_*)."""
    plans = {}
    for klass, old in step.old.items():
        new = step.new[klass]
        tb = [b for (_, b, _, _) in new] + [new[-1][2]]
        plans[klass] = etp.etp_plan_create(mode, old, len(new), tb)
    return plans
