"""N > 1 path of bench.py on CPU: world_size 2, gloo.  The hot path does not shard ("replicas only"):
each rank runs the same workload and the job's number is Σ tokens ÷ max-over-ranks device time."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    seconds = [0.010, 0.025][rank]              # rank 1 is the slow replica
    t = bench.max_over_ranks(seconds)
    dist.barrier()
    out.put((rank, t, bench.job_throughput(2048 * 10, t, world)))
    dist.destroy_process_group()


def test_max_over_ranks_and_job_throughput_gloo_world2():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, t, val in res:
        assert t == pytest.approx(0.025)                       # every rank sees the slowest rank's time
        assert val == pytest.approx(2 * 2048 * 10 / 0.025)     # whole-job tokens/s, not per GPU


def test_single_process_identity():
    import bench
    assert bench.max_over_ranks(0.5) == 0.5
    assert bench.job_throughput(100, 0.5, 1) == 200.0
