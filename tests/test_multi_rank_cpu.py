"""N > 1 path on CPU (`-m "not gpu"`): the hot path does not shard ("replicas only"),
so the only multi-rank logic is bench.py's aggregation -- max over ranks of the device time, whole-job
value = all ranks' units / that time -- and the reference arm's "rank 0 only" rule.  Covered with
world_size 2 over gloo at 127.0.0.1."""
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
    sec = [0.010, 0.025][rank]  # rank 1 is the slow replica
    dist.barrier()
    sec_max = bench.max_over_ranks(torch, sec, dist, torch.device("cpu"))
    value = bench.replicas_value(world, 1000, 7, sec_max)
    dist.barrier()
    with open(f"{out}.{rank}", "w") as f:
        json.dump({"sec_max": sec_max, "value": value}, f)
    dist.destroy_process_group()


def test_replicas_aggregate_over_two_ranks(tmp_path):
    port = 29500 + os.getpid() % 2000
    out = str(tmp_path / "r")
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    for rank in range(2):
        with open(f"{out}.{rank}") as f:
            r = json.load(f)
        assert r["sec_max"] == 0.025  # every rank sees the slowest replica's time
        assert r["value"] == 2 * 1000 * 4 * 7 / 0.025  # units of all ranks over that time


def test_reference_arm_runs_on_rank_zero_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--workload", "config0", "--steps", "1", "--warmup", "3"],
                       env=env, capture_output=True, text=True, timeout=300)
    assert p.returncode == 0 and p.stdout.strip() == ""
    env["RANK"] = "0"
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--workload", "config0", "--steps", "1", "--warmup", "3"],
                       env=env, capture_output=True, text=True, timeout=300)
    assert p.returncode == 0
    line = json.loads(p.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["n_gpus"] == 2
