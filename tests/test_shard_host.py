"""Host logic of the multi-GPU path on CPU: the partition arithmetic of pbs4d_shard_window (device-free entry of the
library) and bench.py's exchange helpers under torch.distributed with the gloo backend, world_size 2 -- every history
exactly once, empty shards, integer sums reproduce the unsharded grids, source-phase ownership."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1809_03927_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("n,world", [(0, 1), (1, 1), (5, 8), (7, 2), (100, 3), (10 ** 8, 8), (2 ** 62, 7), (12345, 148)])
def test_shard_windows_partition_the_history_range(n, world):
    edge = 0
    for r in range(world):
        b, c = binding.shard_window(n, r, world)
        assert b == edge and c >= 0                             # contiguous, in rank order, no gap, no overlap
        assert b == (n * r) // world and b + c == (n * (r + 1)) // world
        assert c in (n // world, n // world + 1)                # balanced to within one history
        edge = b + c
    assert edge == n                                            # every history exactly once


def test_shard_window_bad_arguments():
    for args in [(-1, 0, 1), (10, 0, 0), (10, 2, 2), (10, -1, 2)]:
        with pytest.raises(RuntimeError):
            binding.shard_window(*args)


def test_source_phase_ownership():
    sys.path.insert(0, ROOT)
    import bench
    owners = bench.source_owners([7, 3, 4, 6], 3)
    assert owners == {3: 0, 4: 1, 6: 2, 7: 0}
    masks = [bench.owner_mask(owners, r) for r in range(3)]
    assert masks == [(1 << 3) | (1 << 7), 1 << 4, 1 << 6]
    assert sum(masks) == sum(1 << p for p in owners)            # every source phase pushed exactly once
    assert bench.source_owners([1, 2], 8) == {1: 0, 2: 1}       # more ranks than source phases: the rest push nothing


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # "transport": history h of phase p deposits the integer (h + 1) * (p + 3) at voxel (h * 7 + p) % 50
    n_hist = {0: 11, 1: 0, 2: 5}
    grids, full = [], []
    for p, n in n_hist.items():
        b, c = binding.shard_window(n, rank, world)
        q = torch.zeros(50, dtype=torch.int64); f = torch.zeros(50, dtype=torch.int64)
        for h in range(n):
            v = (h + 1) * (p + 3) * (2 ** 40 + 1)               # beyond fp64-exact float sums: integer adds only
            f[(h * 7 + p) % 50] += v
            if b <= h < b + c:
                q[(h * 7 + p) % 50] += v
        grids.append(q); full.append(f)
    bench.sum_energy_grids(grids, world)
    ok = all(torch.equal(a, b) for a, b in zip(grids, full))
    # "accumulation": the owner holds the sums, the others zeros; after the exchange everyone holds everything
    owners = bench.source_owners([2, 5, 9], world)
    pairs = {}
    for p, r in owners.items():
        val = torch.full((6,), p * 1000 + 1, dtype=torch.int64)
        pairs[p] = (val.clone() if r == rank else torch.zeros(6, dtype=torch.int64),
                    (val * 2).clone() if r == rank else torch.zeros(6, dtype=torch.int64))
    bench.share_accumulators(pairs, owners, world)
    ok2 = all(int(pairs[p][0][0]) == p * 1000 + 1 and int(pairs[p][1][5]) == 2 * (p * 1000 + 1) for p in owners)
    out[rank] = (ok, ok2)
    dist.barrier()
    dist.destroy_process_group()


def test_exchange_helpers_two_ranks_gloo():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, 29741, out), nprocs=world, join=True)
        assert all(out[r] == (True, True) for r in range(world))
