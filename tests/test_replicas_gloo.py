"""N > 1 is "replicas only": no data-path collective, the only cross-rank step is the max over
ranks of the device time and the sum of the work.  world_size-2 gloo run of exactly the helpers bench.py uses, and
the reference arm's rank-0-only rule."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
torch = pytest.importorskip("torch")


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(100.0 + 50.0 * rank, world, "cpu")   # rank 1 is the slow one
    val = bench.job_value(world, 1000, 10, 2, ms)
    dist.barrier()
    dist.destroy_process_group()
    with open(f"{out}.{rank}", "w") as f:
        json.dump({"ms": ms, "value": val}, f)


def test_max_over_ranks_and_job_value_world2(tmp_path):
    import torch.multiprocessing as mp
    out = str(tmp_path / "res")
    mp.spawn(_worker, args=(2, 29533, out), nprocs=2, join=True)
    for rank in range(2):
        r = json.load(open(f"{out}.{rank}"))
        assert r["ms"] == 150.0                              # the slowest replica sets the time on every rank
        assert r["value"] == pytest.approx(2 * 1000 * 10 * 2 / 0.150)


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
