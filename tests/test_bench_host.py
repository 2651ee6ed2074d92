"""Host logic of bench.py without a GPU: the N > 1 aggregation (replicas only) over gloo, world_size 2,
and the reference arm's JSON contract on a tiny sample."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _rank(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms, value = bench.aggregate_replicas(10.0 * (rank + 1), 5, world, torch.device("cpu"), torch, dist)
    dist.barrier()
    if rank == 0:
        json.dump({"ms": ms, "value": value}, open(out, "w"))
    dist.destroy_process_group()


def test_replica_aggregation_gloo_world2(tmp_path):
    out = str(tmp_path / "agg.json")
    mp.spawn(_rank, args=(2, 29500 + os.getpid() % 2000, out), nprocs=2, join=True)
    r = json.load(open(out))
    assert r["ms"] == 20.0                       # max over ranks (10 ms, 20 ms)
    assert abs(r["value"] - 2 * 5 / 20e-3) < 1e-9   # both ranks' iterations over the slowest rank's time


def test_single_rank_aggregation():
    import bench
    ms, value = bench.aggregate_replicas(8.0, 4, 1, torch.device("cpu"), torch, dist)
    assert ms == 8.0 and abs(value - 500.0) < 1e-9


def test_reference_arm_json_contract():
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "tiny",
                        "--steps", "2", "--warmup", "1"], capture_output=True, text=True, timeout=600)
    assert p.returncode == 0, p.stderr
    line = json.loads(p.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "lsqr_iterations_per_s" and line["unit"] == "it/s"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0
