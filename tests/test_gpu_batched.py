"""Parity of cn_batched_sweep with the oracle: every system of a sweep against the
serial Thomas CN stepper, and the 2-D Lie split psi <- CN_y CN_x psi (reading R18) against the oracle's 2-D stepper."""
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


def rand_batch(N, nsys, seed):
    rng = np.random.default_rng([seed, N, nsys])
    V = rng.uniform(-1.0, 1.0, N)
    z = rng.standard_normal((nsys, N, 2))
    return V, (z[..., 0] + 1j * z[..., 1]).astype(np.complex128)


def oracle_batch(dx, dt, V, psi, nsteps):
    return np.stack([O.step(dx, dt, V, psi[k], nsteps) for k in range(psi.shape[0])])


X_CASES = [
    # (N, nsys, pad): N = 8 * 2^k -> in-CTA (N <= 2048) or cluster of 2 / 4 / 8 CTAs; ragged last tile; padded rows
    (64, 1, 0), (64, 37, 0), (128, 33, 8), (256, 9, 0), (512, 5, 0), (1024, 7, 3), (2048, 3, 0), (2048, 1, 0),
    (4096, 5, 0), (8192, 3, 0), (8192, 300, 0), (16384, 2, 16), (16384, 19, 0),
    # generic path: N is not 8 * 2^k
    (100, 13, 0), (9, 4, 2), (2, 3, 0), (24576, 2, 0),
]


@pytest.mark.parametrize("N,nsys,pad", X_CASES)
def test_x_sweep(N, nsys, pad):
    torch = torch_()
    V, psi = rand_batch(N, nsys, 5)
    dx, dt = 0.1, 0.02
    for nsteps in (1, 2):
        ref = oracle_batch(dx, dt, V, psi, nsteps)
        buf = np.full((nsys, N + pad), 7.0 + 7.0j)
        buf[:, :N] = psi
        d = torch.from_numpy(buf).cuda()
        with B.Plan(N, 1 if N < 16 else 2, dx, dt, V) as plan:
            plan.factorize()
            plan.batched_sweep(d, nsys, 1, N + pad, nsteps)
            torch.cuda.synchronize()
        out = d.cpu().numpy()
        err = np.max(np.abs(out[:, :N] - ref))
        assert err <= TOL_PSI, (N, nsys, pad, nsteps, err)
        assert np.all(out[:, N:] == 7.0 + 7.0j)  # padding untouched


Y_CASES = [
    # (N, nsys, pad): N = 16 * 2^k -> one CTA (N <= 1024) or cluster of 2 / 4 / 8 CTAs; ragged last strip
    (64, 8, 0), (64, 13, 0), (128, 40, 3), (256, 9, 0), (512, 24, 0), (1024, 17, 1), (2048, 16, 0), (4096, 11, 0),
    (8192, 8, 0), (8192, 100, 4), (8192, 1200, 0),
    # generic path
    (100, 13, 0), (64, 5, 0), (16384, 9, 0),
]


@pytest.mark.parametrize("N,nsys,pad", Y_CASES)
def test_y_sweep(N, nsys, pad):
    torch = torch_()
    V, psi = rand_batch(N, nsys, 6)
    dx, dt = 0.1, 0.02
    for nsteps in (1, 2):
        ref = oracle_batch(dx, dt, V, psi, nsteps)     # [nsys][N]
        buf = np.full((N, nsys + pad), 7.0 + 7.0j)     # row j of every system is contiguous: buf[j][k]
        buf[:, :nsys] = psi.T
        d = torch.from_numpy(buf).cuda()
        with B.Plan(N, 2, dx, dt, V) as plan:
            plan.factorize()
            plan.batched_sweep(d, nsys, nsys + pad, 1, nsteps)
            torch.cuda.synchronize()
        out = d.cpu().numpy()
        err = np.max(np.abs(out[:, :nsys].T - ref))
        assert err <= TOL_PSI, (N, nsys, pad, nsteps, err)
        assert np.all(out[:, nsys:] == 7.0 + 7.0j)


@pytest.mark.parametrize("kind,N,nsys,opts", [
    ("x", 64, 40, {}), ("x", 2048, 5, {}), ("x", 4096, 3, {}), ("x", 8192, 3, {}), ("x", 16384, 2, {}),
    ("y", 64, 40, {}), ("y", 1024, 11, {}), ("y", 2048, 9, {}), ("y", 8192, 10, {}),
    # strips of 4 columns (CN_OPT_BY_COLS = 4): in-CTA up to 2048 rows, clusters of 2 / 4 CTAs above
    ("y", 128, 13, {"by_cols": 4}), ("y", 1024, 6, {"by_cols": 4}), ("y", 2048, 9, {"by_cols": 4}),
    ("y", 4096, 5, {"by_cols": 4}), ("y", 8192, 7, {"by_cols": 4}),
])
def test_sweeps_strong_coupling(kind, N, nsys, opts):
    """s = dt / (4 dx^2) = 12.5: |q| is close to 1, so the map of a chunk does not decay and the inflow of a chunk
    carries information from the whole system -- every level of the scans (lanes, warps, CTAs of a cluster) with its
    multipliers computed once per kernel matters at the 1e-10 bar.  Also the 4-column strips of the y kernel."""
    torch = torch_()
    V, psi = rand_batch(N, nsys, 8)
    dx, dt = 0.01, 0.005
    for nsteps in (1, 3):
        ref = oracle_batch(dx, dt, V, psi, nsteps)
        d = torch.from_numpy(psi.copy() if kind == "x" else np.ascontiguousarray(psi.T)).cuda()
        with B.Plan(N, 2, dx, dt, V, **opts) as plan:
            plan.factorize()
            if kind == "x":
                plan.batched_sweep(d, nsys, 1, N, nsteps)
            else:
                plan.batched_sweep(d, nsys, nsys, 1, nsteps)
            torch.cuda.synchronize()
        out = d.cpu().numpy()
        err = np.max(np.abs((out if kind == "x" else out.T) - ref))
        assert err <= TOL_PSI, (kind, N, nsys, opts, nsteps, err)


@pytest.mark.parametrize("n", [256, 1024, 2048])
def test_c4_lie_split_scaled(n):
    """Config C4's recipe at n x n: x-sweep then y-sweep per step, one plan per direction, against the oracle."""
    torch = torch_()
    cfg = W.scaled(W.CONFIGS["C4"], N=n, nsys=n)
    psi = W.psi0_2d(cfg)
    Vx, Vy = W.potential(cfg), W.potential_y(cfg)
    steps = 4
    ref = O.step_2d(cfg.dx, cfg.dt, Vx, Vy, psi, steps)
    d = torch.from_numpy(psi).cuda()
    with B.Plan(n, 8, cfg.dx, cfg.dt, Vx) as px, B.Plan(n, 8, cfg.dx, cfg.dt, Vy) as py:
        px.factorize()
        py.factorize()
        for _ in range(steps):
            px.batched_sweep(d, n, 1, n, 1)
            py.batched_sweep(d, n, n, 1, 1)
        torch.cuda.synchronize()
    out = d.cpu().numpy()
    assert np.max(np.abs(out - ref)) <= TOL_PSI
    assert abs(np.vdot(out, out).real * cfg.dx * cfg.dx - 1.0) <= 1e-12


def test_batched_argument_errors():
    torch = torch_()
    V = np.zeros(64)
    psi = torch.zeros((4, 64), dtype=torch.complex128, device="cuda")
    with B.Plan(64, 8, 0.1, 0.01, V) as plan:
        with pytest.raises(B.CnError) as ei:
            plan.batched_sweep(psi, 4, 1, 64, 1)
        assert ei.value.status == B.CN_ENOTFACTORIZED
        plan.factorize()
        for args in [(0, 1, 64), (4, 2, 3), (4, 1, 32), (4, 2, 1)]:   # nsys < 1, no unit stride, overlapping systems
            with pytest.raises(B.CnError) as ei:
                plan.batched_sweep(psi, *args, 1)
            assert ei.value.status == B.CN_EINVAL, args
        plan.batched_sweep(psi, 4, 1, 64, 0)


@pytest.mark.parametrize("kind,N,nsys", [("x", 512, 6000), ("x", 8192, 600), ("y", 1024, 2048), ("y", 8192, 512)])
def test_batched_refill_stress(kind, N, nsys):
    """Many tiles per persistent CTA on L2-resident grids, repeated: the shapes on which a TMA refill can overtake
    shared-memory loads that are still queued when the CTA barrier opens (hazard 1).  The first
    64 systems against the oracle, all systems by norm conservation (the matrix is shared, CN is unitary)."""
    torch = torch_()
    V, sysm = rand_batch(N, nsys, 11)
    dx, dt = 0.1, 0.02
    ref = oracle_batch(dx, dt, V, sysm[:64], 2)
    host = sysm if kind == "x" else np.ascontiguousarray(sysm.T)
    n0 = np.sum(np.abs(sysm) ** 2, 1)
    with B.Plan(N, 2, dx, dt, V) as plan:
        plan.factorize()
        for _ in range(15):
            d = torch.from_numpy(host).cuda()
            if kind == "x":
                plan.batched_sweep(d, nsys, 1, N, 2)
            else:
                plan.batched_sweep(d, nsys, nsys, 1, 2)
            torch.cuda.synchronize()
            out = d.cpu().numpy()
            out = out if kind == "x" else out.T
            assert np.max(np.abs(out[:64] - ref)) <= TOL_PSI
            assert np.max(np.abs(np.sum(np.abs(out) ** 2, 1) / n0 - 1.0)) <= 1e-11
