"""Multi-GPU host logic on CPU (world_size 2, gloo): the path does not shard ("replicas only"), so
N > 1 means N independent replicas whose whole-job figure is sum(applications) / max(time)."""
import os
import subprocess
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, cnt = bench.reduce_over_ranks(dist, 100.0 + 50.0 * rank, 32 + rank, "cpu")
    w = bench.make_workload(2, rank)  # rank-specific seed: replicas are independent problems
    pos = torch.from_numpy(w.x[w.N_bead:w.N_bead + 4].copy())
    gathered = [torch.zeros_like(pos) for _ in range(world)]
    dist.all_gather(gathered, pos)
    if rank == 0:
        out.put((ms, cnt, bool(torch.equal(gathered[0], gathered[1]))))
    dist.destroy_process_group()


def test_replica_aggregation_world2_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    ms, cnt, same = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert ms == 150.0 and cnt == 65.0   # max over ranks, sum over ranks
    assert not same                      # different seeds per rank


def test_single_rank_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks(None, 12.5, 7, "cpu") == (12.5, 7.0)


def test_reference_arm_other_ranks_exit_silently():
    """Under torchrun only rank 0 runs and prints the reference arm; the other ranks exit 0 without work."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--config", "1"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
