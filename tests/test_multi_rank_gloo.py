"""World-size-2 test of the multi-GPU plumbing on CPU (gloo): frame sharding
covers the batch exactly once, timing is the max over ranks, gathering restores
frame order.  The data path itself has no collective (frames are independent)."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, n_frames, out_dir):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_1607_07624_b200 import sharding
        lo, hi = sharding.my_frames(n_frames)
        # stand-in for the per-rank sensor: each "frame" result is its global index
        local = torch.arange(lo, hi, dtype=torch.float32).reshape(-1, 1, 1).repeat(1, 2, 2)
        slow = sharding.max_over_ranks(1.0 + rank)
        parts = sharding.gather_frames(local, n_frames)
        np.save(os.path.join(out_dir, f"r{rank}.npy"), np.array([lo, hi, slow]))
        if rank == 0:
            np.save(os.path.join(out_dir, "gathered.npy"), torch.cat(parts).numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_frames", [100, 7])
def test_two_ranks_shard_time_and_gather(tmp_path, n_frames):
    world, port = 2, 29500 + (os.getpid() % 2000) + n_frames
    mp.spawn(_worker, args=(world, port, n_frames, str(tmp_path)), nprocs=world, join=True)
    r0, r1 = np.load(tmp_path / "r0.npy"), np.load(tmp_path / "r1.npy")
    assert r0[0] == 0 and r0[1] == r1[0] and r1[1] == n_frames          # exact cover, in order
    assert abs((r0[1] - r0[0]) - (r1[1] - r1[0])) <= 1                  # balanced
    assert r0[2] == r1[2] == 2.0                                        # max over ranks
    g = np.load(tmp_path / "gathered.npy")
    assert g.shape == (n_frames, 2, 2) and np.array_equal(g[:, 0, 0], np.arange(n_frames))


def test_single_process_helpers_are_identity():
    from paper_1607_07624_b200 import sharding
    assert sharding.my_frames(10) == (0, 10)
    assert sharding.max_over_ranks(3.5) == 3.5
    t = torch.ones(3, 2)
    assert sharding.gather_frames(t, 3)[0] is t
