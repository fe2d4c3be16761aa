"""The N > 1 path of bench.py on CPU (gloo, world_size 2).  The hot path does not shard ("replicas only"):
every rank reshards its own replica, there is no data-path collective, and the only cross-rank step is the max-over-ranks
of the device times; `value` = bytes of ALL ranks / that time.  `--impl reference` runs on rank 0 alone."""
import json
import os
import subprocess
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, torch.device("cpu"))     # rank 1 is the slow replica
        out[rank] = (ms, bench.whole_job_gbps(3e9, world, ms))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_gloo_world2():
    world, port = 2, 29500 + os.getpid() % 2000
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]                                  # every rank sees the same aggregate
    ms, gbps = res[0]
    assert ms == 15.0                                        # the MAX over ranks, not the mean or rank 0's
    assert gbps == pytest.approx(2 * 3e9 / 15e-3 / 1e9)      # bytes of all ranks / max time


def _shard_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    owners = bench.split_ranks(8, world)
    mine = {r: ("handle-of", rank, r) for r in owners[rank]}        # what ModelState._open_remote exchanges (picklable handles)
    got = [None] * world
    dist.all_gather_object(got, mine)
    seen = sorted(r for h in got for r in h)
    moved = torch.tensor([float(100 * (rank + 1))], dtype=torch.float64)
    dist.all_reduce(moved, op=dist.ReduceOp.SUM)
    ms = torch.tensor([float(3 + rank)], dtype=torch.float64)
    dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    out.put((rank, owners, seen, moved.item(), ms.item(), [got[p][r][1] for p in range(world) for r in got[p]]))
    dist.destroy_process_group()


def test_sharded_partition_by_destination_rank_gloo_world2():
    """--sharded bookkeeping on CPU: simulated rank r belongs to process r mod N, every rank has exactly one owner, the handle
    exchange reaches everybody, the job's bytes are the SUM and its time the MAX over processes."""
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, 29713, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
    for rank, owners, seen, moved, ms, owner_of_handle in res:
        assert owners == [[0, 2, 4, 6], [1, 3, 5, 7]] and seen == list(range(8))
        assert moved == 300.0 and ms == 4.0
        assert owner_of_handle == [0, 0, 0, 0, 1, 1, 1, 1]


def _run_reference(rank):
    env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank), CUDA_VISIBLE_DEVICES="")
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1", "--gpus", "2",
                           "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=600)


def test_reference_arm_runs_on_rank0_only():
    r1 = _run_reference(1)
    assert r1.returncode == 0 and r1.stdout.strip() == ""   # other ranks exit 0 without work
    r0 = _run_reference(0)
    assert r0.returncode == 0, r0.stderr[-2000:]
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["gpu_launches"] == 0 and line["higher_is_better"] is True


def test_ours_fails_loudly_without_a_gpu():
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1", "--warmup", "0"], env=env,
                       capture_output=True, text=True, timeout=600)
    assert r.returncode != 0 and "no CPU fallback" in (r.stderr + r.stdout)


def test_roofline_traffic_is_read_from_the_committed_ncu_capture():
    """bench.py's roofline.traffic comes from profiles/r3_copy_kernel_full.csv (one parameter launch + one KV launch of config 2):
    the file must stay in the layout the parser reads, and the DRAM bytes must stay near the algorithmic 2 B per moved byte."""
    import bench
    t = bench.ncu_traffic_per_launch()
    assert t is not None, "profiles/r3_copy_kernel_full.csv is missing or not in the 'metric,unit,launch1,launch2,...' layout"
    algorithmic = 2.0 * (9.425e9 + 5.369e9) / 2.0          # config 2, device-resident images: bytes moved by the two launches
    assert 0.95 < t / algorithmic < 1.10


def test_ncu_capture_describes_the_kernel_that_is_built():
    """A stale capture must not be quoted: profiles/r3_copy_kernel_full.md records the commit and the SASS hash of
    etp_interval_copy_kernel it profiled; the hash is recomputed here from the built libetp.so (cuobjdump -sass).  After any
    change to the copy kernel this test fails until the capture is taken again."""
    import bench
    from paper_2511_11617_b200 import _build
    stamp = bench.ncu_capture_stamp()
    assert stamp is not None, "profiles/r3_copy_kernel_full.md must carry 'commit: <sha>' and 'kernel_sass_sha: <hash>' lines"
    _build.build()
    built = _build.kernel_sass_sha("etp_interval_copy_kernel")
    assert stamp["kernel_sass_sha"] == built, (
        f"the committed ncu capture profiled kernel {stamp['kernel_sass_sha']} (commit {stamp['commit']}), the built one is {built}: re-capture")
    src = bench.traffic_source()
    assert src["matches_built_kernel"] is True and src["commit"] == stamp["commit"]
