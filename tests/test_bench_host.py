"""Host-side logic of bench.py on CPU: the N>1 aggregation (gloo, world_size 2) and the
reference arm's contract (rank 0 prints one JSON line, other ranks exit 0 silently)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    res = bench.reduce_over_ranks(dist, torch.device("cpu"), 10.0 + rank, 1.0 + 2 * rank, 1000 + rank, 500 * (rank + 1), 7)
    dist.barrier()
    dist.destroy_process_group()
    if rank == 0:
        with open(out, "w") as f:
            json.dump(res, f)


def test_reduce_over_ranks_gloo_world2(tmp_path):
    import torch.multiprocessing as mp
    out = str(tmp_path / "res.json")
    mp.spawn(_worker, args=(2, 29741, out), nprocs=2, join=True)
    ms, e2e_s, n_total, pairs_total, launches = json.load(open(out))
    assert ms == 11.0 and e2e_s == 3.0            # max over ranks
    assert n_total == 2001.0 and pairs_total == 1500.0 and launches == 14   # summed work


def test_reduce_over_ranks_single():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks(None, None, 3.0, 4.0, 10, 5, 2) == (3.0, 4.0, 10.0, 5.0, 2)


def test_reference_arm_contract():
    env = dict(os.environ, RANK="0", WORLD_SIZE="2")
    r0 = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0",
                         "--steps", "3", "--warmup", "1", "--gpus", "2"], capture_output=True, text=True, env=env)
    assert r0.returncode == 0, r0.stderr
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "particle_updates_per_s"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] == 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 1e5
    env["RANK"] = "1"
    r1 = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0",
                         "--steps", "3", "--warmup", "1", "--gpus", "2"], capture_output=True, text=True, env=env)
    assert r1.returncode == 0 and r1.stdout.strip() == ""


def test_bench_refuses_to_run_the_product_on_cpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--config", "0", "--steps", "1"],
                       capture_output=True, text=True)
    assert r.returncode != 0 and "no CPU fallback" in (r.stderr + r.stdout)
