"""Host-side logic of bench.py for N > 1 (replicas only, no data-path collective), exercised on CPU
with the gloo backend and world_size 2: the max-over-ranks timing rule, the whole-job aggregate, and the rule that
only rank 0 runs and prints the reference arm."""
import json
import os
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    t_local = 0.010 * (rank + 1)                  # rank 1 is the slow one
    t = bench.max_over_ranks(t_local, world)
    dist.barrier()
    out[rank] = (t, bench.aggregate_value(world, 1000, 5, t))
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_gloo():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, 29641, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1], "every rank must see the same (max) time"
    t, v = res[0]
    assert abs(t - 0.020) < 1e-12
    assert abs(v - 2 * 1000 * 5 / 0.020) < 1e-6


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(0.5, 1) == 0.5
    assert bench.aggregate_value(1, 10, 2, 4.0) == 5.0


def test_reference_arm_rank0_only():
    """--impl reference under torchrun: rank 0 prints the JSON line, the other ranks exit 0 without work."""
    env = dict(os.environ, WORLD_SIZE="2", LOCAL_RANK="0")
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--workload", "c1",
           "--steps", "1", "--warmup", "0", "--cpu-sample", "256"]
    r1 = subprocess.run(cmd, env=dict(env, RANK="1"), capture_output=True, text=True, timeout=300)
    assert r1.returncode == 0 and r1.stdout.strip() == ""
    r0 = subprocess.run(cmd, env=dict(env, RANK="0"), capture_output=True, text=True, timeout=300)
    assert r0.returncode == 0, r0.stderr
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["n_gpus"] == 2
