"""Host protocol of the sharded mode (paper_2205_00856_b200/sharded.py) on CPU: the SAME generators and the same
`DistributedStepper` that drive `cn_shard_*` on GPUs, here with world_size 2 (and 3) over gloo and a numpy stand-in
for the per-shard plan (tests/shard_stub.py: the paper's scheme with one process per block, written densely).
Checked against the oracle's plain Thomas stepper on the WHOLE system: the exchange order (edge values, then one
record per step), the rank-ordered all-gather and the in-place update of the local rows.  Also the in-process driver
`LocalShards` (what the GPU parity tests use) on the same stand-in."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import cn_oracle as O
from paper_2205_00856_b200 import sharded as SH
from paper_2205_00856_b200 import workloads as W

from shard_stub import NumpyShard

CFG = W.scaled(W.CONFIGS["C1"], N=384, dx=0.05, dt=0.01)  # s = 1: strong coupling between neighbouring rows
NSTEPS = (3, 1, 2)                                        # three runs on the same vector, 6 steps in all


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n = CFG.N // world
        V, psi = W.potential(CFG), W.psi0(CFG)
        plan = NumpyShard(n, CFG.dx, CFG.dt, V[rank * n:(rank + 1) * n], rank, world)
        mine = torch.from_numpy(psi[rank * n:(rank + 1) * n].copy())
        st = SH.DistributedStepper(plan, device=torch.device("cpu"))
        st.factorize()
        for k in NSTEPS:
            st.step(mine, k)
        q.put((rank, mine.numpy().copy()))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_distributed_stepper_gloo(world):
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    parts = dict(q.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    out = np.concatenate([parts[r] for r in range(world)])
    ref = O.step(CFG.dx, CFG.dt, W.potential(CFG), W.psi0(CFG), sum(NSTEPS))
    assert np.max(np.abs(out - ref)) <= 1e-11


@pytest.mark.parametrize("S", [1, 2, 4, 6])
def test_local_shards_driver(S):
    n = CFG.N // S
    V, psi = W.potential(CFG), W.psi0(CFG)
    plans = [NumpyShard(n, CFG.dx, CFG.dt, V[r * n:(r + 1) * n], r, S) for r in range(S)]
    parts = [torch.from_numpy(psi[r * n:(r + 1) * n].copy()) for r in range(S)]
    grp = SH.LocalShards(plans, lambda c: torch.zeros(c, dtype=torch.complex128), torch.cat)
    grp.factorize()
    for k in NSTEPS:
        grp.step(parts, k)
    grp.step(parts, 0)  # no-op
    out = np.concatenate([x.numpy() for x in parts])
    ref = O.step(CFG.dx, CFG.dt, V, psi, sum(NSTEPS))
    assert np.max(np.abs(out - ref)) <= 1e-11


def test_protocol_exchange_count():
    """n steps = n + 1 exchanges (edge values + one record per step) of the sizes the plan states."""
    plan = NumpyShard(CFG.N, CFG.dx, CFG.dt, W.potential(CFG), 0, 1)
    alloc = lambda c: torch.zeros(c, dtype=torch.complex128)  # noqa: E731
    g = SH.factorize_protocol(plan, alloc)
    rec = next(g)
    assert rec.numel() == plan.counts()[0]
    with pytest.raises(StopIteration):
        g.send(rec.clone())
    psi = torch.from_numpy(W.psi0(CFG).copy())
    g = SH.run_protocol(plan, psi, 4, alloc)
    sizes, rec = [], next(g)
    try:
        while True:
            sizes.append(rec.numel())
            rec = g.send(rec.clone())
    except StopIteration:
        pass
    assert sizes == [1] + [plan.counts()[1]] * 4
