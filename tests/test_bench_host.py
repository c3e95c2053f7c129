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


def test_ncu_export_is_keyed_by_the_kernel_sources(tmp_path, monkeypatch):
    """bench.py takes `traffic` and the instruction counts from a tracked ncu export; one step = the last launch
    of every kernel instantiation; an export measured on other kernel sources reads as (None, 'stale...')."""
    sys.path.insert(0, ROOT)
    import bench
    head = '"ID","Process ID","Process Name","Host Name","Kernel Name","Context","Stream","Block Size","Grid Size","Device","CC","Section Name","Metric Name","Metric Unit","Metric Value"'

    def row(i, name, metric, unit, value):
        return '"%d","1","python","h","%s","1","7","(256, 1, 1)","(444, 1, 1)","0","10.0","Command line profiler metrics","%s","%s","%s"' % (
            i, name, metric, unit, value)
    raw = tmp_path / "raw.csv"
    raw.write_text("\n".join([
        "==PROF== noise", head,
        row(0, "void cuba::k_collide<256, 6, 1536, 3, 0, 0, 0>(cuba::CollideParams)", "dram__bytes_read.sum", "Gbyte", "9.0"),     # an earlier step
        row(1, "void cuba::k_collide<64, 4, 256, 12, 0, 0, 0>(cuba::CollideParams)", "dram__bytes_read.sum", "Mbyte", "100"),
        row(2, "void cuba::k_collide<256, 6, 1536, 3, 0, 0, 0>(cuba::CollideParams)", "dram__bytes_read.sum", "Gbyte", "1.5"),
        row(2, "void cuba::k_collide<256, 6, 1536, 3, 0, 0, 0>(cuba::CollideParams)", "smsp__inst_executed.sum", "inst", "549,000,000"),
        row(2, "void cuba::k_collide<256, 6, 1536, 3, 0, 0, 0>(cuba::CollideParams)", "launch__registers_per_thread", "register/thread", "80"),
        row(3, "void cuba::k_scatter<0>(cuba::Geom)", "dram__bytes_write.sum", "Gbyte", "1.25"),
    ]) + "\n")
    monkeypatch.setattr(bench, "NCU_EXPORT", str(tmp_path / "export_c%d.csv"))
    bench.import_ncu(str(raw), 2)
    d, src = bench.ncu_export(2)
    assert d["k_collide"]["dram__bytes_read.sum"] == 1.5e9 + 100e6          # the last launch of each of the two instantiations
    assert d["k_collide"]["smsp__inst_executed.sum"] == 549e6 and d["k_collide"]["launch__registers_per_thread"] == 80
    assert d["k_scatter"]["dram__bytes_write.sum"] == 1.25e9
    monkeypatch.setattr(bench, "kernel_source_hash", lambda: "0" * 64)
    d, why = bench.ncu_export(2)
    assert d is None and why.startswith("stale")
    d, why = bench.ncu_export(7)
    assert d is None and "no tracked" in why
    r = bench.fp64_roofline(86e6, 1.0, 18.56e12, "x")
    assert abs(r["frac"] - (86e6 / 1e-3) / (18.56e12 / 32)) < 1e-12 and abs(r["peak_tflops"] - 37.12) < 1e-9
