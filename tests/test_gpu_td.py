"""Time-dependent Hamiltonian H(t) = H0 + f(t) g(x): cn_step_td through the C-ABI
against the oracle's step_td (one plain Thomas solve with its own diagonals per step), same tolerances as the static
path: max |dpsi| <= 1e-10, relative residual of a solve <= 1e-12."""
import numpy as np
import pytest

from oracle import cn_oracle as O
from paper_2205_00856_b200 import binding as B
from paper_2205_00856_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL_PSI = 1e-10
TOL_RES = 1e-12


def gpu_td(N, P, dx, dt, V, g, field, psi, **opts):
    import torch
    d = torch.from_numpy(np.ascontiguousarray(psi)).cuda()
    with B.Plan(N, P, dx, dt, np.ascontiguousarray(V), **opts) as plan:
        plan.factorize()
        plan.set_td_shape(np.ascontiguousarray(g))
        plan.step_td(d, field)
        torch.cuda.synchronize()
        out = d.cpu().numpy()
        # the plan holds the static factors again: a static step after the driven ones must match the oracle too
        plan.step(d, 2)
        torch.cuda.synchronize()
        info = plan.info()
    return out, d.cpu().numpy(), info


def laser(nsteps, dt, E0=0.05, omega=0.3):
    t = (np.arange(nsteps) + 0.5) * dt          # midpoint of every step
    return E0 * np.sin(omega * t) * np.sin(np.pi * t / (nsteps * dt)) ** 2


CASES = [
    # (N, P, opts)
    (4096, 64, dict(path=B.PATH_TILED)),
    (4096, 64, dict(path=B.PATH_GENERIC)),
    (4096, 64, dict()),                              # auto: the on-chip stepper is NOT used for driven steps
    (5000, 123, dict()),                             # ragged blocks -> generic kernels
    (1 << 16, 1 << 13, dict()),                      # nested RS
    (1 << 16, 1 << 13, dict(pdl=0)),
    (1 << 18, 1 << 10, dict()),
]


@pytest.mark.parametrize("N,P,opts", CASES)
def test_td_parity(N, P, opts):
    cfg = W.scaled(W.CONFIGS["C1"], N=N)
    dx, dt = 0.05, 0.01
    V, psi = W.potential(cfg), W.psi0(cfg)
    x = W.grid(cfg)
    nsteps = 12
    field = laser(nsteps, dt, E0=0.5)               # strong enough to move gamma in the 3rd digit
    ref = O.step_td(dx, dt, V, x, field, psi)
    out, out2, info = gpu_td(N, P, dx, dt, V, x, field, psi, **opts)
    err = float(np.max(np.abs(out - ref)))
    assert err <= TOL_PSI, (N, P, opts, err)
    assert float(np.max(np.abs(out2 - O.step(dx, dt, V, ref, 2)))) <= TOL_PSI
    assert abs(np.vdot(out, out).real / np.vdot(psi, psi).real - 1.0) <= 1e-12


def test_td_zero_field_is_static_and_one_solve_residual():
    cfg = W.scaled(W.CONFIGS["C1"], N=1 << 14)
    dx, dt = cfg.dx, cfg.dt
    V, psi, x = W.potential(cfg), W.psi0(cfg), W.grid(cfg)
    out, _, _ = gpu_td(cfg.N, 1 << 8, dx, dt, V, x, np.zeros(3), psi)
    assert float(np.max(np.abs(out - O.step(dx, dt, V, psi, 3)))) <= TOL_PSI
    # one driven solve: residual with the stencil typed here
    f = 0.37
    one, _, _ = gpu_td(cfg.N, 1 << 8, dx, dt, V, x, np.array([f]), psi)
    s = dt / (4 * dx * dx)
    a = 1 + 1j * (2 * s + 0.5 * dt * (V + f * x))

    def apply(diag, off, v):
        y = diag * v
        y[1:] += off * v[:-1]
        y[:-1] += off * v[1:]
        return y
    d = apply(np.conj(a), 1j * s, psi)
    r = apply(a, -1j * s, one) - d
    assert np.linalg.norm(r) / np.linalg.norm(d) <= TOL_RES


def test_td_errors():
    import torch
    V = np.zeros(64)
    d = torch.zeros(64, dtype=torch.complex128, device="cuda")
    with B.Plan(64, 8, 0.1, 0.01, V) as plan:
        plan.factorize()
        with pytest.raises(B.CnError):              # no shape set
            plan.step_td(d, np.zeros(2))
