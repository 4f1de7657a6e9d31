"""N > 1 host logic on CPU (world_size 2, gloo): `bench.py --gpus N` runs independent replicas (DESIGN.md 8,
"replicas only"): the only cross-rank steps are the barrier and the max-over-ranks of the device time, and
the reference arm runs on rank 0 alone."""
import json
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms_local = 3.0 + 2.0 * rank                      # rank 1 is the slow replica
    dist.barrier()
    ms = bench.max_over_ranks(ms_local, world, "cpu")
    value = bench.job_throughput(1536 * 32 * 10, world, ms)
    q.put((rank, ms, value))
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, value in res:
        assert ms == 5.0                             # both ranks see the slowest rank's time
        assert abs(value - 2 * 1536 * 32 * 10 / 5.0e-3) < 1e-6 * value
    import bench
    assert bench.max_over_ranks(4.25, 1, "cpu") == 4.25


def test_reference_arm_runs_on_rank0_only():
    # rank 1 of a 2-rank launch exits 0 without work and prints nothing
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
