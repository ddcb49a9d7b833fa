"""Many systems with a potential of their own each (cn_plan_set_systems / cn_batched_sweep_v; SURVEY 8f-3,
PAPER.md:74, 209-211: with a non-separable V(x, y) every line of a sweep has its own tridiagonal matrix).
Every system against the oracle's plain Thomas stepper with that system's potential, element by element."""
import numpy as np
import pytest

from oracle import cn_oracle as O
from paper_2205_00856_b200 import binding as B
from paper_2205_00856_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL_PSI = 1e-10


def problem(n, nsys, seed, dx=0.05, dt=0.004):
    """nsys systems of n rows: seeded smooth potentials that differ from system to system, dense complex states"""
    rng = np.random.default_rng(seed)
    x = (np.arange(n) - 0.5 * (n - 1)) * dx
    amp, wid, cen = rng.uniform(-2, 2, (nsys, 1)), rng.uniform(0.5, 5, (nsys, 1)), rng.uniform(x[0], x[-1], (nsys, 1))
    V = amp * np.exp(-((x[None, :] - cen) / wid) ** 2) + 0.5 * rng.uniform(0, 1, (nsys, 1)) * x[None, :] ** 2 / max(1.0, x[-1] ** 2)
    psi = rng.standard_normal((nsys, n)) + 1j * rng.standard_normal((nsys, n))
    return dx, dt, np.ascontiguousarray(V), np.ascontiguousarray(psi)


def oracle_all(dx, dt, V, psi, nsteps):
    return np.stack([O.step(dx, dt, V[k], psi[k], nsteps) for k in range(V.shape[0])])


@pytest.mark.parametrize("n,nsys,fast", [
    (8, 128, True), (64, 64, True), (256, 32, True), (512, 16, True), (8192, 4, True), (1024, 1, True),
    (2048, 37, True),
    (8, 3, False),       # N / 8 is not a multiple of 32 -> one thread per system
    (24, 32, False),     # 3 blocks of 8 rows per system: not a power of two -> one thread per system
    (100, 7, False),
])
def test_contiguous_systems(n, nsys, fast):
    import torch
    dx, dt, V, psi = problem(n, nsys, seed=n + nsys)
    nsteps = 5
    ref = oracle_all(dx, dt, V, psi, nsteps)
    d = torch.from_numpy(psi.reshape(-1).copy()).cuda()
    with B.Plan(n * nsys, nsys, dx, dt, V.reshape(-1)) as plan:
        plan.set_systems(nsys, 1, n).factorize()
        assert plan.info()["path"] == (B.PATH_TILED if fast else B.PATH_GENERIC)
        plan.batched_sweep_v(d, 2)
        plan.batched_sweep_v(d, nsteps - 2)
        torch.cuda.synchronize()
        out = d.cpu().numpy().reshape(nsys, n)
        assert np.max(np.abs(out - ref)) <= TOL_PSI
        with pytest.raises(B.CnError):  # systems with matrices of their own: not the shared-matrix sweep
            plan.batched_sweep(d, nsys, 1, n, 1)


@pytest.mark.parametrize("n,nsys", [(64, 8), (300, 100), (1024, 512)])
def test_interleaved_systems(n, nsys):
    """Column layout psi[row][system] (the y-sweep of a 2-D grid with a non-separable potential)."""
    import torch
    dx, dt, V, psi = problem(n, nsys, seed=7 * n + nsys)
    nsteps = 3
    ref = oracle_all(dx, dt, V, psi, nsteps)
    d = torch.from_numpy(np.ascontiguousarray(psi.T).reshape(-1)).cuda()
    with B.Plan(n * nsys, nsys, dx, dt, np.ascontiguousarray(V.T).reshape(-1)) as plan:
        plan.set_systems(nsys, nsys, 1).factorize()
        plan.batched_sweep_v(d, nsteps)
        torch.cuda.synchronize()
        out = d.cpu().numpy().reshape(n, nsys).T
        assert np.max(np.abs(out - ref)) <= TOL_PSI


def test_2d_nonseparable_potential():
    """A 2-D Lie-split step with V(x, y) that does NOT separate: the x sweep uses V/2 along rows, the y sweep V/2 along
    columns, every line with its own matrix.  Oracle: the same two sweeps line by line with the plain 1-D stepper."""
    import torch
    ny = nx = 256
    dx, dt = 0.1, 0.01
    x = (np.arange(nx) - 0.5 * (nx - 1)) * dx
    V2 = 0.5 * (x[None, :] ** 2 + x[:, None] ** 2) + 0.3 * x[None, :] * x[:, None] + np.cos(x[None, :] * x[:, None])
    rng = np.random.default_rng(11)
    psi = rng.standard_normal((ny, nx)) + 1j * rng.standard_normal((ny, nx))
    ref = psi.copy()
    for _ in range(3):
        ref = np.stack([O.step(dx, dt, 0.5 * V2[y], ref[y], 1) for y in range(ny)])
        ref = np.stack([O.step(dx, dt, 0.5 * V2[:, c], ref[:, c], 1) for c in range(nx)], axis=1)
    d = torch.from_numpy(psi.reshape(-1).copy()).cuda()
    half = np.ascontiguousarray(0.5 * V2).reshape(-1)
    with B.Plan(nx * ny, ny, dx, dt, half) as px, B.Plan(nx * ny, nx, dx, dt, half) as py:
        px.set_systems(ny, 1, nx).factorize()
        py.set_systems(nx, nx, 1).factorize()
        for _ in range(3):
            px.batched_sweep_v(d, 1)
            py.batched_sweep_v(d, 1)
        torch.cuda.synchronize()
    assert np.max(np.abs(d.cpu().numpy().reshape(ny, nx) - ref)) <= TOL_PSI


def test_systems_errors():
    dx, dt, V, psi = problem(64, 8, 1)
    with B.Plan(512, 8, dx, dt, V.reshape(-1)) as plan:
        for args in ((3, 1, 64), (8, 1, 65), (8, 2, 1), (0, 1, 64)):
            with pytest.raises(B.CnError) as e:
                plan.set_systems(*args)
            assert e.value.status == B.CN_EINVAL
        with pytest.raises(B.CnError) as e:
            plan.batched_sweep_v(0x10, 1)   # no systems declared
        assert e.value.status == B.CN_EINVAL
