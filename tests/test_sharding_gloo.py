"""World-size-2 gloo tests (CPU) of the multi-rank bookkeeping used by bench.py --gpus N: direction
slices partition the job, step time is the max over ranks, units are summed, and gathered force
slices land in global direction order."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2602_10712_b200 import sharding
from paper_2602_10712_b200 import workloads as W


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        S_total, D = 11, 3                                        # ragged split: 6 + 5 directions
        mine = sharding.direction_slice(S_total, rank, world)
        # stand-in for the per-rank srp_forces result: F[k, j] = (k, global j, rank)
        local = torch.zeros((D, len(mine), 3))
        for k in range(D):
            local[k, :, 0] = k
            local[k, :, 1] = torch.from_numpy(mine.astype(np.float32))
            local[k, :, 2] = rank
        full = sharding.gather_forces(local, S_total)
        t, u = sharding.combine_timing(1.0 + rank, 100 * (rank + 1))
        dirs = sharding.weak_scaling_directions(4, rank, world)
        if rank == 0:
            torch.save({"full": full, "t": t, "u": u, "dirs0": dirs}, out)
        else:
            torch.save({"dirs1": dirs}, out + ".1")
    finally:
        dist.destroy_process_group()


def test_two_rank_sharding(tmp_path):
    out = str(tmp_path / "r0.pt")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    r = torch.load(out, weights_only=False)
    full = r["full"].numpy()
    assert full.shape == (3, 11, 3)
    assert np.array_equal(full[1, :, 1], np.arange(11))           # global direction order restored
    assert np.array_equal(full[2, :, 2], np.arange(11) % 2)       # interleaved ownership
    assert r["t"] == 2.0 and r["u"] == 300.0                      # max of times, sum of units
    d0, d1 = r["dirs0"], torch.load(out + ".1", weights_only=False)["dirs1"]
    allv = W.fibonacci_sphere(8)
    assert np.array_equal(d0, allv[0::2]) and np.array_equal(d1, allv[1::2])   # weak scaling: disjoint shares


def test_slices_partition_and_single_process_passthrough():
    for S, world in ((4096, 8), (11, 2), (5, 4)):
        parts = [sharding.direction_slice(S, r, world) for r in range(world)]
        assert sorted(np.concatenate(parts).tolist()) == list(range(S))
    assert sharding.combine_timing(1.5, 7) == (1.5, 7.0)
    x = torch.ones((2, 3, 3))
    assert sharding.gather_forces(x, 3) is x
