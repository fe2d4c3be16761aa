"""etp_copy_intervals_static: the interval copy for callers that are not allowed to allocate device memory.

Who needs it: a reshard runs right after a GPU failure, when the surviving GPUs' HBM is full of weights and KV blocks and the
serving engine's memory pool owns whatever is left, so a cudaMalloc from inside this library can fail or take memory the engine
counted on; cudaMalloc / cudaFree also stall every stream of the device; and code hosted inside another component's CUDA context
is often forbidden to create memory.  The normal entry points need an etp_ctx (whose creation allocates arenas, events, streams);
this one keeps the copy kernel's scratch (descriptors, item table, queue heads) in a 0.4-MiB static device array of the library
and takes no ctx.

What is checked: on the same seeded intervals the static entry point leaves every destination byte (gaps and guard bands
included) exactly as the existing etp_copy_intervals does, and as the plain definition computed on the host says, on TWO calls in
a row (the second with fewer, differently sized intervals, so stale descriptors and non-zero queue heads of the first call would
show); the limits are rejected with ETP_ERR_CAPACITY and nothing written; the device's free memory does not change across the
calls.  Byte work: the tolerance is equality, as in the other copy tests.

This file is named to be collected last: pytest -x stops at the first failure, and a failure here must not hide the parity tests.
It passes alone in a fresh process (the first call does the per-device set-up) and after the other GPU tests."""
import numpy as np
import pytest
import torch

import paper_2511_11617_b200 as etp
from tests.gpu_util import DevBuf
from workloads.gen import microbench_intervals

pytestmark = pytest.mark.gpu

MAX_INTERVALS = 4096      # include/etp.h: limits of etp_copy_intervals_static
MAX_BULK_PIECES = 32768


def _case(n, hi, seed, src, max_total):
    """config-5b recipe (workloads.gen): log-uniform sizes from 16 B, overlapping sources, disjoint destinations with gaps"""
    so, do, sz, dst_arena = microbench_intervals(n, 16, hi, seed, src.size, max_total=max_total)
    dst0 = np.random.default_rng(seed).integers(0, 256, dst_arena, dtype=np.uint8)
    expect = dst0.copy()
    for a, b, m in zip(so, do, sz):
        expect[b:b + m] = src[a:a + m]
    return so, do, sz, dst0, expect


def test_static_entry_matches_ctx_path_two_calls_in_a_row():
    src = np.random.default_rng(11).integers(0, 256, 48 << 20, dtype=np.uint8)
    S = DevBuf(src)
    stream = torch.cuda.Stream()
    ctx = etp.Context(0)
    try:
        # call 1: the most intervals the entry point takes, 16 B .. 2 MiB (bulk pieces, ragged tails, batches of small ones);
        # call 2: fewer intervals, all below 32 KiB (no bulk queue at all -> the staged small-batch instantiation), so anything
        # left over from call 1 in the static array (bulk descriptors, item table, advanced queue heads) would be visible
        cases = [_case(MAX_INTERVALS, 2 << 20, 101, src, 192 << 20), _case(1500, 8 << 10, 202, src, 64 << 20)]
        bufs = []
        for so, do, sz, dst0, expect in cases:
            D_ctx, D_static = DevBuf(dst0), DevBuf(dst0)
            etp.etp_copy_intervals(ctx, so + S.ptr, do + D_ctx.ptr, sz, stream.cuda_stream)
            bufs.append((D_ctx, D_static, so, do, sz, expect))
        stream.synchronize()
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        for D_ctx, D_static, so, do, sz, expect in bufs:      # the two static calls back to back on one stream, no sync in between
            etp.etp_copy_intervals_static(so + S.ptr, do + D_static.ptr, sz, stream.cuda_stream)
        stream.synchronize()
        assert torch.cuda.mem_get_info()[0] == free_before, "the no-allocation entry point changed the device's free memory"
        for k, (D_ctx, D_static, so, do, sz, expect) in enumerate(bufs):
            assert D_static.guards_intact() and D_ctx.guards_intact(), k
            got = D_static.payload().tobytes()
            assert got == D_ctx.payload().tobytes(), f"call {k + 1}: static entry point differs from etp_copy_intervals"
            assert got == expect.tobytes(), f"call {k + 1}: differs from the plain definition"
        assert S.guards_intact() and S.payload().tobytes() == src.tobytes()
    finally:
        ctx.close()


def test_static_entry_same_buffers_twice():
    """The same call repeated (second time over different source bytes): the array's contents from the first call are exactly the
    descriptors of the second, the queue heads are not; the result must follow the second source."""
    rng = np.random.default_rng(5)
    n = 700
    size = rng.choice([16, 256, 4096, 48 << 10, 300 << 10], n).astype(np.int64)
    do = np.cumsum(size + 16 * rng.integers(0, 3, n)) - size
    so = (rng.integers(0, (8 << 20) // 16, n) * 16).astype(np.int64)
    total = int(do[-1] + size[-1])
    stream = torch.cuda.Stream()
    D = DevBuf(np.zeros(total, np.uint8))
    for rep in range(2):
        src = rng.integers(0, 256, (8 << 20) + (300 << 10), dtype=np.uint8)
        S = DevBuf(src)
        expect = D.payload().copy()
        for a, b, m in zip(so, do, size):
            expect[b:b + m] = src[a:a + m]
        etp.etp_copy_intervals_static(so + S.ptr, do + D.ptr, size, stream.cuda_stream)
        stream.synchronize()
        assert D.guards_intact() and D.payload().tobytes() == expect.tobytes(), rep


def test_static_entry_rejects_what_it_cannot_hold():
    S, D = DevBuf(np.zeros(1 << 20, np.uint8)), DevBuf(np.full(1 << 20, 7, np.uint8))
    n = MAX_INTERVALS + 1
    i = np.arange(n, dtype=np.int64)
    with pytest.raises(etp.EtpError) as e:      # too many intervals
        etp.etp_copy_intervals_static(S.ptr + 16 * i, D.ptr + 16 * i, np.full(n, 16, np.int64))
    assert e.value.status == 3 and "4096" in str(e.value)
    # too many 256-KiB pieces: one more than the limit, described but never touched (the check comes before any enqueue, and the
    # addresses are beyond the buffers, so an enqueued copy would fault)
    big = np.array([(MAX_BULK_PIECES + 1) * (256 << 10)], dtype=np.int64)
    with pytest.raises(etp.EtpError) as e:
        etp.etp_copy_intervals_static(np.array([S.ptr]), np.array([S.ptr + (1 << 40)]), big)
    assert e.value.status == 3 and "32768" in str(e.value)
    with pytest.raises(etp.EtpError) as e:      # the contract of etp_copy_intervals: overlapping destinations
        etp.etp_copy_intervals_static(np.array([S.ptr, S.ptr + 64]), np.array([D.ptr, D.ptr + 32]), np.array([64, 64]))
    assert e.value.status == 1
    with pytest.raises(etp.EtpError) as e:      # misaligned
        etp.etp_copy_intervals_static(np.array([S.ptr + 8]), np.array([D.ptr]), np.array([64]))
    assert e.value.status == 2
    etp.etp_copy_intervals_static(np.zeros(0, np.int64), np.zeros(0, np.int64), np.zeros(0, np.int64))   # empty: a no-op
    torch.cuda.synchronize()
    assert D.guards_intact() and (D.payload() == 7).all()
