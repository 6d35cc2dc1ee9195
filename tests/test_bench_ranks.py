"""The N > 1 path of bench.py on CPU (gloo, world size 2).  The path does not shard (north_star: one GPU), so N ranks are N
independent replicas: the only cross-rank logic is the contract's max-over-ranks timing and the whole-job value, plus the
rule that the reference arm runs on rank 0 only."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, torch.device("cpu"))     # rank 1 is the slow one
    dist.barrier()
    out[rank] = (ms, bench.job_value(world, 1000.0, ms))
    dist.destroy_process_group()


def test_max_over_ranks_and_job_value_gloo_world2():
    import torch.multiprocessing as mp
    mgr = mp.Manager()
    out = mgr.dict()
    port = _free_port()
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    assert out[0] == out[1]                                  # every rank sees the slowest rank's time
    ms, value = out[0]
    assert ms == 15.0
    assert value == pytest.approx(2 * 1000.0 / 15e-3)        # whole-job aggregate of two replicas


def test_single_process_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, None, None) == 3.5
    assert bench.job_value(1, 2.0e9, 10.0) == pytest.approx(2.0e11)


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
