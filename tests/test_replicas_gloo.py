"""The N > 1 path of bench.py ("replicas only") with world_size 2 over gloo on CPU:
barrier, max over ranks of the per-rank time, whole-job throughput."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2205_00856_b200 import replicas as R


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert R.dist_env() == (rank, world, rank)
        R.barrier(world)
        ms = R.max_over_ranks(10.0 + 5.0 * rank, world)       # rank 1 is the slow one
        q.put((rank, ms, R.whole_job_throughput(1 << 20, 100, ms, world)))
    finally:
        dist.destroy_process_group()


def test_two_replicas_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, val in res:
        assert ms == 15.0                                       # the max over ranks, on every rank
        assert val == pytest.approx(2 * (1 << 20) * 100 / 15e-3 / 1e9)


def test_single_process_is_identity():
    assert R.max_over_ranks(3.5, 1) == 3.5
    assert R.whole_job_throughput(1000, 10, 1.0, 1) == pytest.approx(1e-2)
