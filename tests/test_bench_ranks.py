"""bench.py's multi-rank bookkeeping on CPU (gloo, world_size 2): the path has no collective -- `--gpus N` runs N independent
replicas -- so what N > 1 adds is the barrier, the max over ranks of the device time, the whole-job
value and "rank 0 alone prints".  These run without a GPU."""
import json
import os
import subprocess
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(dist, 100.0 + 50.0 * rank, torch.device("cpu"))    # rank 1 is the slow replica
    dist.barrier()
    if rank == 0:
        with open(out, "w") as f:
            json.dump({"ms": ms, "value": bench.whole_job_value(world, 1024, 13, ms)}, f)
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_gloo(tmp_path):
    out = str(tmp_path / "r0.json")
    mp.spawn(_worker, args=(2, 29631, out), nprocs=2, join=True)
    got = json.load(open(out))
    assert got["ms"] == 150.0                                   # the slowest replica sets the time
    assert got["value"] == pytest.approx(2 * 1024 * 13 / 0.150)   # both replicas' work over that time


def test_single_process_needs_no_process_group():
    assert bench.max_over_ranks(None, 12.5, None) == 12.5
    assert bench.whole_job_value(1, 512, 11, 100.0) == pytest.approx(56320.0)


def test_reference_arm_prints_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--cfg", "1", "--steps", "1",
                        "--warmup", "0", "--gpus", "2"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--cfg", "1", "--steps", "1",
                        "--warmup", "0", "--gpus", "2"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
