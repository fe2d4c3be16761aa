"""Race and stale-state hunting without a sanitizer (compute-sanitizer is closed on this pool, profiles/r2_sanitizer.md):
the kernels that hand-roll synchronisation - mbarrier rings, cluster barriers, multicast commits, ticketed split-K and
tail-split reductions, atomic work queues, cross-stream hazard phases - are run many times back to back on one context,
with a disturbing kernel in between so that SM residency and timing differ from run to run, and every run must reproduce
the first one bit for bit (all of these paths are deterministic by construction: fixed summation orders, disjoint writes).
The first run of each case is checked against the oracle, so "all equal" cannot mean "all equally wrong".  Outputs are
pre-filled with NaN patterns: an element a run failed to write differs from the first run's."""
import os

import numpy as np
import pytest
import torch

import paper_2511_11617_b200 as etp
from oracle import linear as OL
from tests import harness as H
from tests import test_gpu_linear as TL
from tests import test_gpu_reshard as TR
from tests.gpu_util import DevBuf, LibSide, Streams
from workloads import get_config
from workloads.gen import as_u8, fill_normal16, torch_dtype

pytestmark = pytest.mark.gpu
REPEATS = int(os.environ.get("ETP_STRESS_REPEATS", "25"))   # the soak run of profiles/r2_sanitizer.md sets 400


@pytest.fixture(scope="module")
def ctx():
    c = etp.Context(0)
    yield c
    c.close()


def disturb(i):
    """occupy a varying number of SMs for a varying time right before the next launch"""
    n = (1 + (i * 37) % 23) << 16
    a = torch.empty(n, dtype=torch.float32, device="cuda")
    a.normal_()
    return a.sum()


@pytest.mark.parametrize("mode,T,K,N,widths,pair_opt", [
    ("row", 2560, 1000, 2040, (300, 400, 300), 1),      # CTA pairs + tail split (ticketed fp32 partials)
    ("col", 1000, 1024, 3000, (1000, 1001, 999), 1),    # CTA pairs, two accumulator stages, odd tile counts
    ("row", 512, 2312, 2048, (770, 771, 771), 0),       # single-CTA tiles, several items per CTA
    ("col", 4, 5120, 5120, (1707, 1707, 1706), 1),      # 4 tokens: split-K through the prepared-group kernel
])
def test_shard_linear_repeats_bit_for_bit(ctx, mode, T, K, N, widths, pair_opt):
    dt = "bf16"
    cut = N if mode == "col" else K
    layout = TL.widths_to_layout(widths)
    geom = {r: (b - 1 - r, (e - b) + 3 + r) for (r, b, e, _) in layout}
    row_bytes = (K if mode == "col" else N) * 2
    w_u8 = as_u8(fill_normal16(TL.SEED, 2100 + T, 0, N * K, 0.02, torch_dtype(dt))).copy()
    x_u8 = as_u8(fill_normal16(TL.SEED, 2101 + T, 0, T * K, 1.0, torch_dtype(dt))).copy()
    slabs = TL.shard_into_slabs(w_u8, row_bytes, layout, geom)
    bufs = {r: DevBuf(a) for r, a in slabs.items()}
    desc = etp.TensorDesc(cut, row_bytes, {r: (bufs[r].ptr, geom[r][1], geom[r][0]) for r in bufs}, len(widths), 0)
    xb = DevBuf(x_u8)
    ys = [torch.full((T * N,), float("nan"), dtype=torch.bfloat16, device="cuda") for _ in range(REPEATS)]
    ctx.set_option(etp.OPT_LINEAR_CTA_PAIR, pair_opt)
    try:
        for i, y in enumerate(ys):
            disturb(i)
            etp.etp_shard_linear(ctx, etp.COL_PARALLEL if mode == "col" else etp.ROW_PARALLEL, dt, xb.ptr, T, K, N, desc, layout, 1, y.data_ptr(), 0)
    finally:
        ctx.set_option(etp.OPT_LINEAR_CTA_PAIR, 1)
    torch.cuda.synchronize()
    ref = TL.reference(dt, x_u8, w_u8, T, K, N, transposed=(mode == "row"))
    TL.check(as_u8(ys[0].cpu()), ref, dt, T, N)
    for i in range(1, REPEATS):
        assert torch.equal(ys[0].view(torch.int16), ys[i].view(torch.int16)), f"run {i} differs from run 0"


@pytest.mark.parametrize("moe_pair", [0, 2])
def test_moe_fused_layer_repeats_bit_for_bit(ctx, moe_pair):
    """gate|up fused + down through the grouped kernels (single-CTA and CTA-pair), many items per CTA / cluster."""
    E, F, Hd, widths = 6, 384, 256, (2, 1, 3)
    rows = (300, 17, 0, 520, 256, 64)
    ws, descs, layout, geom, bufs = TL._moe_world(E, F, Hd, widths, 1, 31)
    offs = np.concatenate([[0], np.cumsum(rows)]).astype(np.int64)
    R = int(offs[-1])
    dt = torch_dtype("bf16")
    x_u8 = as_u8(fill_normal16(TL.SEED, 2200, 0, R * Hd, 1.0, dt)).copy()
    xb = DevBuf(x_u8)
    hs = [torch.full((R * F,), float("nan"), dtype=dt, device="cuda") for _ in range(REPEATS)]
    ys = [torch.full((R * Hd,), float("nan"), dtype=dt, device="cuda") for _ in range(REPEATS)]
    ctx.set_option(etp.OPT_MOE_CTA_PAIR, moe_pair)
    try:
        for i in range(REPEATS):
            disturb(i)
            etp.etp_moe_gate_up(ctx, "bf16", xb.ptr, Hd, F, descs["gate"], descs["up"], hs[i].data_ptr(), row_offsets=offs, layout=layout)
            etp.etp_moe_linear(ctx, etp.ROW_PARALLEL, "bf16", hs[i].data_ptr(), offs, F, Hd, descs["down_t"], layout, ys[i].data_ptr())
    finally:
        ctx.set_option(etp.OPT_MOE_CTA_PAIR, 1)
    torch.cuda.synchronize()
    x64 = OL.decode16(x_u8, "bf16").reshape(R, Hd)
    g64, u64 = (OL.decode16(ws[k], "bf16").reshape(E, F, Hd) for k in ("gate", "up"))
    ref = np.concatenate([OL.swiglu_ref(x64[offs[e]:offs[e + 1]], g64[e], u64[e]) for e in range(E) if rows[e]])
    TL.check(as_u8(hs[0].cpu()), ref, "bf16", R, F)
    for i in range(1, REPEATS):
        assert torch.equal(hs[0].view(torch.int16), hs[i].view(torch.int16)), f"gate|up run {i} differs from run 0"
        assert torch.equal(ys[0].view(torch.int16), ys[i].view(torch.int16)), f"down run {i} differs from run 0"


@pytest.mark.parametrize("image", ["pinned", "device"])
def test_multi_phase_reshard_repeats_bit_for_bit(ctx, image):
    """Config 1 with tight (wrapping) slabs: several hazard phases ordered by events across the copy and reload streams, the
    atomic work queues of kernel (a), the zero-copy gather.  Every repeat starts from a fresh upload of the same world and is
    compared with the oracle's image (so each run is checked, not only run 0)."""
    cfg = get_config("1")
    world = H.build_param_world(cfg, side=LibSide, mode="tight")
    expect, stats = H.oracle_reshard_params(world, 0)
    streams = Streams()
    for i in range(REPEATS):
        bufs, images = TR.upload_param_world(world, image=image)
        disturb(i)
        rep = TR.run_param_step(ctx, world, bufs, images, 0, streams)
        TR.compare_params(world, bufs, expect, {world.steps[0].dead})
        assert rep["d2d_bytes"] == stats["d2d_bytes"] and rep["n_phases"] >= 2


# ------------------------------------------------------------------------------------------------ liveness of the hand-rolled waits
def test_starved_barrier_fails_loudly_within_seconds():
    """Every spin wait of the kernels is an mbarrier wait with a 10-s deadline (csrc/etp_wait.cuh).  etp_debug_starved_wait launches a
    kernel that waits - with the copy kernel's own wait routine - on a barrier nobody arrives on: the call must come back with
    ETP_ERR_CUDA and a record naming the kernel family, block, thread and barrier within seconds (not hang until the pool is reset),
    and every later call must fail as well.  The CUDA context is lost afterwards, so the whole thing runs in a throw-away process."""
    import json
    import subprocess
    import sys
    code = r'''
import json, os, sys, time
import paper_2511_11617_b200 as etp
c = etp.Context(0)
out = {}
t0 = time.time()
try:
    etp.etp_debug_starved_wait(c)
    out["first"] = "no error"
except etp.EtpError as e:
    out["first"] = [e.status, str(e)]
out["seconds"] = time.time() - t0
try:
    etp.Context(0)
    out["later"] = "no error"
except etp.EtpError as e:
    out["later"] = [e.status, str(e)]
print("RESULT " + json.dumps(out), flush=True)
os._exit(0)          # no teardown on a dead context
'''
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    p = subprocess.run([sys.executable, "-c", code], cwd=root, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, timeout=120)
    lines = [ln for ln in p.stdout.splitlines() if ln.startswith("RESULT ")]
    assert lines, (p.stdout, p.stderr)
    out = json.loads(lines[-1][7:])
    status, msg = out["first"]
    assert status == 6, out                                         # ETP_ERR_CUDA
    assert "device wait starved" in msg and "interval copy" in msg and "thread 0 " in msg and "parity 0" in msg, msg
    assert 9.0 <= out["seconds"] <= 40.0, out
    assert out["later"] != "no error" and out["later"][0] == 6, out   # the error is sticky: nothing hangs, nothing pretends to work
