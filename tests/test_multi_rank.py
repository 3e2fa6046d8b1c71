"""N > 1 path of bench.py on CPU: world_size 2 over gloo (replicas only - every rank runs its
own seeded trajectory, the ranks meet only in a barrier and a MAX reduction of their timings)."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        dist.barrier()
        ms = 1.0 + 0.5 * rank                       # rank 1 is the slower replica
        got = bench.max_over_ranks([ms, 10.0 - rank], dist, torch.device("cpu"))
        rate = bench.whole_job_rate(world, 98304, 1000, got[0])
        with open(os.path.join(out, "r%d.json" % rank), "w") as f:
            json.dump({"max": got, "rate": rate, "seed": bench.replica_seed(100, rank)}, f)
    finally:
        dist.destroy_process_group()


def test_timings_are_maxed_and_rate_is_whole_job(tmp_path):
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    res = [json.load(open(tmp_path / ("r%d.json" % r))) for r in range(2)]
    for r in res:
        assert r["max"] == [1.5, 10.0]                                   # the slowest rank on every rank
        assert abs(r["rate"] - 2 * 98304 * 1000 / 1.5e-3) < 1e-3       # both replicas' atom-steps over that time
    assert res[0]["seed"] != res[1]["seed"]                              # independent trajectories


def test_single_process_needs_no_process_group():
    import bench
    assert bench.max_over_ranks([2.0, 3.0], None, torch.device("cpu")) == [2.0, 3.0]
    assert bench.whole_job_rate(1, 10, 5, 1.0) == 50000.0


def test_reference_arm_runs_on_rank_0_only():
    """Under torchrun the oracle arm is printed by rank 0; the other ranks exit 0 without work or output."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "3"], env=env, capture_output=True, text=True, timeout=120)
    assert p.returncode == 0 and p.stdout.strip() == ""
