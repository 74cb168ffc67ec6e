"""N > 1 is "replicas only": one process per GPU, no data-path collective; the ranks
exchange exactly one number per timed region (the max of the device-timed interval) and rank 0 prints the
line.  The host-side logic runs here under gloo with world_size 2 on the CPU."""
from __future__ import annotations

import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank: int, world: int, port: int, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 3.0 * rank, world, "cpu")        # rank 1 is the slow one
    dist.barrier()
    q.put((rank, ms, bench.replica_us_per_layer_step(ms, 2, 32, world)))
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_metric_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [g[1] for g in got] == [13.0, 13.0]                        # every rank sees the max
    assert abs(got[0][2] - 13.0 * 1e3 / 64 / 2) < 1e-9                # two replicas: twice the layer-steps


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(7.5, 1, "cpu") == 7.5
    assert bench.replica_us_per_layer_step(3.2, 1, 32, 1) == 100.0


def test_reference_arm_only_rank0_works():
    """bench.py --impl reference under torchrun: ranks other than 0 exit 0 without work or output."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
