"""The N > 1 path of bench.py on CPU: two gloo ranks (replicas only, no data-path
collective; the only communication is the max-over-ranks of the timed region)."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _rank(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r's timed region took (1 + r) seconds for 1000 units
    seconds, value = bench.replicas_aggregate(1.0 + rank, 1000, world)
    dist.barrier()
    dist.destroy_process_group()
    with open(f"{out}.{rank}", "w") as f:
        json.dump({"seconds": seconds, "value": value}, f)


def test_two_ranks_take_the_slowest_and_count_every_replica(tmp_path):
    world, out = 2, str(tmp_path / "r")
    mp.spawn(_rank, args=(world, 29500 + os.getpid() % 2000, out), nprocs=world, join=True)
    got = [json.load(open(f"{out}.{r}")) for r in range(world)]
    for g in got:
        assert g["seconds"] == 2.0                      # the max over ranks, on every rank
        assert g["value"] == 2 * 1000 / 2.0             # units of ALL replicas over the job's time


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.replicas_aggregate(0.5, 100, 1) == (0.5, 200.0)


def test_reference_arm_runs_on_rank_zero_only():
    """Under torchrun the other ranks of --impl reference exit 0 without work or output."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
