"""The N > 1 path of bench.py on CPU: the path does not shard (replicas only), so the only cross-rank
logic is the max-over-ranks time and the whole-job sum.  Two gloo processes on 127.0.0.1."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms = 10.0 + 5.0 * rank                      # rank 1 is the slow replica
        worst = bench.max_over_ranks(dist, ms, torch.device("cpu"))
        out.put((rank, worst, bench.job_tcups(world, 2.0e12, worst * 1e-3)))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_replicas_max_time_and_job_sum():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, worst, value in got:
        assert worst == 15.0                                     # both ranks agree on the slowest replica's time
        assert abs(value - 2 * 2.0e12 / 15.0e-3 / 1e12) < 1e-9   # two replicas' cell updates over that time


def test_single_process_is_identity():
    import bench
    assert bench.max_over_ranks(None, 3.5, None) == 3.5
    assert bench.job_tcups(1, 1.0e12, 1.0) == 1.0
