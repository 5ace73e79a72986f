"""N > 1 host logic of bench.py on CPU: world_size 2 over gloo (no GPU).

The path runs on one GPU (north_star); bench.py --gpus N runs N independent replicas: per-rank
seeds, time = max over ranks, value = units of all ranks / that time, rank 0 alone prints; the reference arm
runs on rank 0 only and the other ranks exit 0 without work.
"""
import json
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = bench.WORKLOADS["su3_48"]
    ms_local = 100.0 + 50.0 * rank                      # rank 1 is the slow one
    ms = bench.max_over_ranks(dist, ms_local, "cpu")
    updates = (bench.N_HB + bench.N_OR) * 4 * wl["L"] ** 4
    q.put((rank, bench.rank_seed(wl, rank), ms, bench.whole_job_rate(world, updates, ms, 10)))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_aggregation_over_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, ms0, v0), (r1, s1, ms1, v1) = out
    assert (s0, s1) == (7, 8)                           # independent chains
    assert ms0 == ms1 == 150.0                          # both ranks see the max
    updates = 5 * 4 * 48 ** 4
    assert v0 == v1 == 2 * updates / (150.0 / 10 * 1e-3)


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(None, 12.5, "cpu") == 12.5
    assert bench.whole_job_rate(1, 1000, 10.0, 10) == 1000 / 1e-3


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env = dict(os.environ, RANK="0", WORLD_SIZE="2", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "2", "--warmup", "1", "--workload", "su2_8"], env=env, capture_output=True,
                       text=True, timeout=300)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["metric"] == "link_updates_per_s"
