"""Multi-GPU is "replicas only": N independent replicas with different seeds, no
data-path collective.  What the N > 1 path adds on the host -- per-rank seeds, max-over-ranks timing,
summed launch counts, rank 0 alone running the reference arm -- is covered here with two gloo
processes on the CPU."""
import json
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    times, counts = bench.reduce_over_ranks([10.0 + rank, 5.0 - rank, 1.0], [7 + rank], world, "cpu")
    cfg = bench.build_workload("C1", (32, 32), rank)
    q.put((rank, times, counts, int(cfg["params"]["seed"]), int(cfg["ids"].sum())))
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_over_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    (r0, t0, c0, s0, l0), (r1, t1, c1, s1, l1) = out
    assert t0 == t1 == [11.0, 5.0, 1.0]      # max over ranks
    assert c0 == c1 == [15]                  # sum over ranks
    assert s0 != s1 and l0 == l1             # independent replicas of the same workload


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks([1.5, 2.5], [3], 1, "cpu") == ([1.5, 2.5], [3])


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--dims", "32x32x32"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env = dict(os.environ, RANK="0", WORLD_SIZE="2", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--dims", "32x32x32"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
