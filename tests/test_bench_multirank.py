"""Host logic of bench.py for N > 1 ("replicas only"), on CPU with the gloo backend, world_size 2:
the whole-job rate is the sum of the ranks' units over the MAX of the ranks' times, and the reference arm runs on rank 0
only."""
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
    ms_local = 10.0 if rank == 0 else 25.0          # rank 1 is the slow one
    units = 1000 * (rank + 1)                        # 1000 + 2000 units
    rate, ms = bench.whole_job_rate(ms_local, units, dist, torch.device("cpu"))
    out[rank] = (rate, ms)
    dist.destroy_process_group()


def test_whole_job_rate_is_sum_of_units_over_max_time():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, 29591, out), nprocs=world, join=True)
        res = dict(out)
    for r in range(world):
        rate, ms = res[r]
        assert ms == 25.0
        assert abs(rate - 3000 / 25e-3) < 1e-6


def test_single_process_rate_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    rate, ms = bench.whole_job_rate(4.0, 8, None, torch.device("cpu"))
    assert ms == 4.0 and abs(rate - 2000.0) < 1e-9


def test_reference_arm_runs_on_rank_zero_only():
    """`bench.py --impl reference` under a 2-rank launch: rank 1 exits 0 without work or output; rank 0 prints the line."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1", MASTER_ADDR="127.0.0.1", MASTER_PORT="29592")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                        "--workload", "cfg1"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"] = "0"; env["LOCAL_RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "2", "--warmup", "1",
                        "--workload", "cfg1"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0


def test_plain_start_with_gpus_2_launches_its_own_ranks():
    """`python bench.py --gpus 2 --impl reference` with no launcher around it (the shape of the driver's N = 1 command): bench.py
    re-executes itself under torch.distributed.run with two ranks; exactly one JSON line comes out, from rank 0, with n_gpus = 2."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "reference", "--steps", "2", "--warmup", "1",
                        "--workload", "cfg1"], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    assert lines[0]["impl"] == "reference" and lines[0]["n_gpus"] == 2 and lines[0]["value"] > 0
