"""N > 1 host logic on CPU (gloo, world_size 2), replica mode (the default of bench.py --gpus N): ranks run
independent replicas and the only exchange is bench.py's max-over-ranks timing reduction; the reference arm runs on
rank 0 alone.  The point-sharded mode is covered by tests/test_sharding_host.py and tests/test_gpu_sharding.py."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = [120.0, 150.0][rank]                       # rank 1 is the slow one
    got = bench.max_over_ranks(ms)
    seed = bench.replica_seed(3, rank)
    dist.barrier()
    dist.destroy_process_group()
    with open(f"{out}.{rank}", "w") as fh:
        json.dump({"max": got, "seed": seed, "rate": bench.whole_job_rate(world, 10, got)}, fh)


def test_timing_is_the_max_over_ranks_and_replicas_get_their_own_seed(tmp_path):
    out = str(tmp_path / "r")
    mp.spawn(_worker, args=(2, 29631, out), nprocs=2, join=True)
    res = [json.load(open(f"{out}.{r}")) for r in range(2)]
    assert res[0]["max"] == res[1]["max"] == 150.0
    assert [r["seed"] for r in res] == [3, 1003]
    assert res[0]["rate"] == 2 * 10 / 0.150           # whole-job units / slowest rank's time


def test_without_a_process_group_the_reduction_is_the_identity():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.max_over_ranks(7.5) == 7.5
    assert bench.whole_job_rate(1, 10, 100.0) == 100.0


def test_reference_arm_runs_on_rank_0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert p.returncode == 0 and p.stdout.strip() == ""
