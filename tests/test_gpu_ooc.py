"""Out-of-core mode: psi in pinned host memory, the library's device memory capped,
partitions streamed H2D / solved / D2H.  Parity with the oracle element by element."""
import numpy as np
import pytest

from oracle import cn_oracle as O
from paper_2205_00856_b200 import binding as B
from paper_2205_00856_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL_PSI = 1e-10


def torch_():
    import torch
    return torch


OOC_CASES = [
    # (N, P, budget bytes, steps)
    (1 << 16, 1 << 8, 1 << 20, 3),      # 11 parts, ragged last part
    (1 << 16, 1 << 8, 1 << 20, 1),      # prologue + epilogue only
    (1 << 17, 1 << 14, 6 << 20, 4),     # m = 8, nested RS (16384 joint lines)
    (1 << 18, 1 << 6, 3 << 20, 3),      # m = 4096: tile = block = 4096 points
    (1 << 15, 1 << 7, 400000, 5),       # parts of a single tile
    (3 << 15, 3 << 7, 1 << 20, 3),      # N not a power of two
    ((1 << 15) + 256, 129, 1000000, 3), # the last part (256 points) is not a whole tile: its tail reads the zeroed / stale buffer rows
]


@pytest.mark.parametrize("N,P,budget,steps", OOC_CASES)
def test_ooc_parity(N, P, budget, steps):
    torch = torch_()
    cfg = W.scaled(W.CONFIGS["C5"], N=N, P=P)
    V, psi = W.potential(cfg), W.psi0(cfg)
    dx, dt = 0.05, 0.01  # C5's dx = 0.01 at these sizes would put the whole packet in a few rows
    ref = O.step(dx, dt, V, psi, steps)
    h = torch.from_numpy(psi.copy()).pin_memory()
    with B.Plan(N, P, dx, dt, V, device_budget=budget) as plan:
        plan.factorize()
        info = plan.info()
        assert info["out_of_core"] == 1 and info["device_bytes"] <= budget, info
        assert info["tile_points"] < N
        plan.step(h, steps)
        torch.cuda.synchronize()
        # a second call continues from the host array
        plan.step(h, 2)
        torch.cuda.synchronize()
    ref2 = O.step(dx, dt, V, ref, 2)
    err = np.max(np.abs(h.numpy() - ref2))
    assert err <= TOL_PSI, err


def test_ooc_needs_pinned_host_memory():
    torch = torch_()
    N, P = 1 << 15, 1 << 7
    V, psi = W.random_system(N, seed=3)
    with B.Plan(N, P, 0.1, 0.01, V, device_budget=400000) as plan:
        plan.factorize()
        with pytest.raises(B.CnError) as ei:
            plan.step(torch.from_numpy(psi).cuda(), 1)      # a device pointer
        assert ei.value.status == B.CN_EINVAL
        with pytest.raises(B.CnError) as ei:
            plan.step(psi.copy(), 1)                        # pageable host memory
        assert ei.value.status == B.CN_EINVAL
    # a budget that cannot hold even one part
    with B.Plan(N, P, 0.1, 0.01, V, device_budget=50000) as plan:
        with pytest.raises(B.CnError) as ei:
            plan.factorize()
        assert ei.value.status == B.CN_ENOMEM


def test_budget_large_enough_stays_in_core():
    torch = torch_()
    N, P = 1 << 14, 1 << 6
    V, psi = W.random_system(N, seed=4)
    ref = O.step(0.1, 0.01, V, psi, 2)
    d = torch.from_numpy(psi).cuda()
    with B.Plan(N, P, 0.1, 0.01, V, device_budget=1 << 30) as plan:
        plan.factorize()
        assert plan.info()["out_of_core"] == 0
        plan.step(d, 2)
        torch.cuda.synchronize()
    assert np.max(np.abs(d.cpu().numpy() - ref)) <= TOL_PSI
