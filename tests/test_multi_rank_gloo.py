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
        from paper_1607_07624_b200 import sharding, workloads as wl
        lo, hi = sharding.my_frames(n_frames)
        # the rank's block of frames as bench.py builds it: whole steps of the config, starting at step lo
        cfg = wl.CONFIGS["cfg1_tiny"]
        mine = wl.phase_batch(cfg, steps=hi - lo, first_step=lo)
        whole = wl.phase_batch(cfg, steps=n_frames)
        assert np.array_equal(mine, whole[lo:hi])                       # the shards tile the unsharded batch
        # stand-in for the per-rank sensor: each "frame" result is its global index
        local = torch.arange(lo, hi, dtype=torch.float32).reshape(-1, 1, 1).repeat(1, 2, 2)
        slow = sharding.max_over_ranks(1.0 + rank)
        parts = sharding.gather_frames(local, n_frames)
        np.save(os.path.join(out_dir, f"r{rank}.npy"), np.array([lo, hi, slow]))
        if rank == 0:
            np.save(os.path.join(out_dir, "gathered.npy"), torch.cat(parts).numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_frames", [12, 7])
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


# ---- bench.py's own multi-rank entry point ---------------------------------------------------
def _bench(*argv, timeout=300):
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_PORT")}
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *argv], capture_output=True, text=True,
                          timeout=timeout, env=env, cwd=ROOT)


def test_bench_gpus_2_starts_two_ranks_and_reports_the_whole_job():
    """`python bench.py --gpus 2` with no launcher must start two ranks itself (PAPER.md:L346
    "multiple GPUs ... in the same system").  --dry-run swaps the CUDA sensor for a CPU stand-in on gloo, so the
    spawn, the frame sharding (sharding.my_frames over world x batch), the barrier / max-over-ranks timing and the
    one-line report are the code the GPU run uses."""
    import json
    p = _bench("--gpus", "2", "--dry-run", "--steps", "2", "--warmup", "1", "--config", "cfg1_tiny")
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [ln for ln in p.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, p.stdout                                   # rank 0 alone prints
    line = json.loads(lines[0])
    assert line["n_gpus"] == 2 and line["dry_run"] is True and line["scaling"] == "weak"
    assert line["config"]["frames_per_step"] == 20 and line["config"]["frames_per_rank"] == 10
    assert len(line["per_rank_frames_per_s"]) == 2
    # whole-job value = all ranks' frames / the slowest rank's time: never above the sum of the ranks' own rates
    assert 0 < line["value"] <= sum(line["per_rank_frames_per_s"]) * (1 + 1e-9)
    assert line["value"] <= 2 * min(line["per_rank_frames_per_s"]) * (1 + 1e-9)


def test_bench_refuses_more_gpus_than_the_node_has():
    n_dev = torch.cuda.device_count() if torch.cuda.is_available() else 0
    if n_dev >= 2:
        pytest.skip("this node has two devices")
    p = _bench("--gpus", "2", "--steps", "1", "--warmup", "0")
    assert p.returncode != 0 and "needs 2 CUDA devices" in (p.stderr + p.stdout)


def test_bench_under_a_launcher_checks_world_size():
    import subprocess
    env = dict(os.environ, WORLD_SIZE="2", RANK="0", LOCAL_RANK="0")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "1", "--dry-run"], capture_output=True,
                       text=True, timeout=120, env=env, cwd=ROOT)
    assert p.returncode != 0 and "WORLD_SIZE=2" in (p.stderr + p.stdout)
