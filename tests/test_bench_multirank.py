"""Host logic of bench.py's N > 1 path on CPU (gloo, world_size 2): replicas only -- every rank times an independent
plan, times are reduced with MAX and histories with SUM; the reference arm runs on rank 0
alone.  No GPU and no compute call is involved."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r pretends it needed (100 + 50 r) ms / (1 + r) s for (10 + r) * 1e6 histories
    res = bench.reduce_over_ranks(100.0 + 50.0 * rank, 1.0 + rank, (10 + rank) * 1e6, (20 + rank) * 1e6, world,
                                  torch.device("cpu"))
    out[rank] = res
    dist.barrier()
    dist.destroy_process_group()


def test_times_max_histories_sum_over_two_ranks():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, 29731, out), nprocs=world, join=True)
        for r in range(world):
            assert out[r] == (150.0, 2.0, 21e6, 41e6)


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks(1.0, 2.0, 3.0, 4.0, 1, torch.device("cpu")) == (1.0, 2.0, 3.0, 4.0)


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
