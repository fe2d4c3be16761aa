"""Run under torchrun by tests/test_gpu_multidevice.py (never collected by pytest): N processes, every one on cuda:0
(ETP_BENCH_ALIAS_GPU0=1, gloo plumbing), build the SHARDED ModelState of a config - each process owns the slabs and pools of
the simulated ranks r with r mod N == its rank and maps the others through CUDA IPC -, run one reshard in which each process
writes only its own ranks, then check the WHOLE state (every rank, local and mapped) against the plain definition evaluated
from the seeded generator, and the per-process byte counts against the oracle's plan."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import torch
import torch.distributed as dist


def main():
    key, n_layers, n_seqs = sys.argv[1], int(sys.argv[2]), int(sys.argv[3])
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    torch.cuda.set_device(0)
    dist.init_process_group("gloo")
    import paper_2511_11617_b200 as etp
    from oracle import planning as OP
    from paper_2511_11617_b200.state import ModelState
    from tests import test_gpu_fullsize as F
    from workloads import get_config
    from workloads.configs import scaled

    def exchange(mine):
        out = [None] * world
        dist.all_gather_object(out, mine)
        return out

    cfg = scaled(get_config(key), n_layers=n_layers, n_seqs=n_seqs)
    state = ModelState(cfg, device="cuda:0", image="pinned", slack_garbage=True, shard=(rank, world), exchange=exchange)
    torch.cuda.synchronize()
    dist.barrier()
    ctx = etp.Context(0)
    ctx.set_rank_devices(state.rank_devices())
    cs, rs = torch.cuda.Stream(), torch.cuda.Stream()
    rep = state.reshard(ctx, 0, "pinned", cs.cuda_stream, rs.cuda_stream, replan=True)
    cs.synchronize(), rs.synchronize()
    dist.barrier()
    torch.cuda.synchronize()
    F.check_params_whole_state(state, 1, True)
    F.check_kv_whole_state(state, 1, True)
    # bytes this process moved = the oracle's tasks whose destination it owns
    st = state.steps[0]
    d2d = rel = 0
    for sp in state.specs:
        for (kind, src, dst, b, e) in F.oracle_tasks(state, st, sp.klass, sp.total_units):
            if state.is_local(dst):
                d2d += (e - b) * sp.unit_bytes if kind == OP.TRANSFER else 0
                rel += (e - b) * sp.unit_bytes if kind == OP.RELOAD else 0
    assert rep["params"]["d2d_bytes"] == d2d and rep["params"]["h2d_bytes"] == rel, (rank, rep["params"], d2d, rel)
    tot = torch.tensor([float(rep["params"]["d2d_bytes"] + rep["params"]["h2d_bytes"] + rep["params"]["remote_bytes"])], dtype=torch.float64)
    lo, hi = tot.clone(), tot.clone()
    dist.all_reduce(lo, op=dist.ReduceOp.MIN)
    dist.all_reduce(hi, op=dist.ReduceOp.MAX)
    assert lo.item() == hi.item() == tot.item()          # every process sees the same plan: local + remote = everything
    dist.barrier()
    ctx.close()
    print(f"SHARDED_OK rank {rank}/{world} d2d={d2d} reload={rel}")
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
