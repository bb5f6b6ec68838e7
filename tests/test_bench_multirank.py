"""Host logic of bench.py's N > 1 path on CPU (gloo, world_size 2).  The N ranks share ONE plan (strong scaling: each
transports its slice of every phase's histories); times are reduced with MAX and histories with
SUM; `python bench.py --gpus N` outside a launcher starts the N ranks itself; the reference arm runs on rank 0 alone.
No GPU and no compute call is involved."""
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


def test_gpus_2_without_a_launcher_starts_two_ranks():
    # what the driver's N = 1 style command line does for N > 1: no WORLD_SIZE in the environment
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--dry-ranks"],
                       env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(x) for x in r.stdout.splitlines() if x.startswith("{")]
    assert lines == [{"dry": True, "n_gpus": 2, "ranks_seen": 2, "requested": 2}]


def test_rank_count_must_match_gpus():
    env = dict(os.environ, RANK="0", LOCAL_RANK="0", WORLD_SIZE="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--dry-ranks"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode != 0 and "--gpus 2" in r.stderr


def test_roofline_figures_are_tied_to_the_kernel_source(tmp_path, monkeypatch):
    # the lane-instruction counts bench.py multiplies with come from ncu captures under profiles/; the metrics file
    # carries the git blob hash of each kernel's source at capture time, and an edited source must show as STALE
    import hashlib
    sys.path.insert(0, ROOT)
    import bench
    src = tmp_path / "kernel.cu"
    src.write_text("__global__ void k() {}\n")
    data = src.read_bytes()
    blob = hashlib.sha1(b"blob %d\0" % len(data) + data).hexdigest()
    git = subprocess.run(["git", "hash-object", str(src)], capture_output=True, text=True).stdout.strip()
    assert not git or git == blob                                          # the same hash `git hash-object` prints
    csv = tmp_path / "metrics.csv"
    csv.write_text(f"# header\n#source,transport_kernel,{src},{blob}\nkernel,workload,metric,value,source\n"
                   "transport_kernel,config5,thread_inst_per_step,217.89,x.ncu-rep\n")
    monkeypatch.setattr(bench, "PROFILE_CSV", str(csv))
    assert bench.profile_source_state() == {"transport_kernel": "current"}
    assert bench.profile_metrics()[("transport_kernel", "config5", "thread_inst_per_step")] == 217.89
    src.write_text("__global__ void k() {}  // a comment\n")
    assert bench.profile_source_state()["transport_kernel"].startswith("STALE")
