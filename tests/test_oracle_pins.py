"""Pins of the oracle against things that are NOT the oracle: dense LU (LAPACK), closed forms,
invariants, textbook physics.  All CPU (`-m "not gpu"`).  Each test names the mistake it would catch."""
import math
import os

import numpy as np
import pytest

from oracle import cn_oracle as O
from oracle import nshape_table1 as T1
from paper_2205_00856_b200 import workloads as W


def hamiltonian_dense(dx, V):
    """H = -1/2 d^2/dx^2 + V with the 3-point stencil, Dirichlet ends; built from the definition of the
    second difference, not from the oracle's (b, a, c)."""
    n = len(V)
    D2 = (np.diag(np.ones(n - 1), -1) - 2.0 * np.eye(n) + np.diag(np.ones(n - 1), 1)) / dx ** 2
    return -0.5 * D2 + np.diag(V)


def rand_tridiag(n, seed):
    rng = np.random.default_rng(seed)
    b = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    c = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    a = (3.0 + rng.random(n)) * np.exp(2j * math.pi * rng.random(n)) + 0.0
    a *= (np.abs(b) + np.abs(c)).max() / 2.0
    d = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    return b, a, c, d


def dense_from(b, a, c):
    n = len(a)
    M = np.zeros((n, n), complex)
    M[np.arange(n), np.arange(n)] = a
    M[np.arange(1, n), np.arange(n - 1)] = b[1:]
    M[np.arange(n - 1), np.arange(1, n)] = c[:-1]
    return M


# ---- dense complex LU, N <= 64 (north_star) -------------------------------------------------------
@pytest.mark.parametrize("n", [1, 2, 3, 8, 33, 64])
def test_thomas_vs_dense_lu(n):
    # catches: swapped b/c, wrong pivot update, off-by-one in back substitution
    b, a, c, d = rand_tridiag(n, 100 + n)
    x = O.thomas(b, a, c, d)
    ref = np.linalg.solve(dense_from(b, a, c), d)
    assert np.max(np.abs(x - ref)) <= 1e-13 * max(1.0, np.max(np.abs(ref)))


@pytest.mark.parametrize("n,steps", [(2, 3), (5, 4), (33, 10), (64, 25)])
def test_step_vs_dense_cayley(n, steps):
    # catches: T on the wrong side, missing conjugate, sign of i, stencil weights, V term
    rng = np.random.default_rng(7 + n)
    V = rng.uniform(-2.0, 3.0, n)
    psi = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    dx, dt = 0.3, 0.07
    H = hamiltonian_dense(dx, V)
    Tm = np.eye(n) + 0.5j * dt * H
    ref = psi.copy()
    for _ in range(steps):
        ref = np.linalg.solve(Tm, Tm.conj().T @ ref)      # Eq. 2: T psi' = T^dagger psi
    out = O.step(dx, dt, V, psi, steps)
    assert np.max(np.abs(out - ref)) <= 1e-13
    assert np.max(np.abs(O.step(dx, dt, V, psi, steps, lean=True) - ref)) <= 1e-13
    assert np.allclose(O.dense_T(dx, dt, V), Tm, rtol=0, atol=1e-15)


# ---- closed form: sine modes of the discrete Dirichlet Laplacian at V = 0 (north_star) -------------
@pytest.mark.parametrize("n,k", [(33, 1), (33, 7), (33, 33), (1000, 1), (1000, 7), (1000, 1000), (4096, 513)])
def test_cayley_phase_closed_form(n, k):
    # catches: wrong 1/2 in H, wrong dx power, boundary rows, sign of i (phase would be conjugated)
    dx, dt, steps = 0.1, 0.01, 1000
    j = np.arange(1, n + 1)
    v = np.sin(math.pi * k * j / (n + 1)).astype(complex)
    lam = (1.0 - math.cos(math.pi * k / (n + 1))) / dx ** 2          # eigenvalue of -1/2 D2
    phase = ((1.0 - 0.5j * lam * dt) / (1.0 + 0.5j * lam * dt)) ** steps
    out = O.step(dx, dt, np.zeros(n), v, steps)
    assert np.max(np.abs(out - phase * v)) <= 2e-12
    # the phase is far from 1 and from its conjugate for these parameters unless lam*dt*steps ~ 0
    if k > 1:
        assert abs(phase - np.conj(phase)) > 1e-3
    out_lean = O.step(dx, dt, np.zeros(n), v, steps, lean=True)
    assert np.max(np.abs(out_lean - phase * v)) <= 2e-12


def test_cayley_phase_2d():
    # C4: product of two sine modes -> product of the two phases (Lie split of commuting factors is exact)
    nx, ny, dx, dt, steps = 24, 17, 0.2, 0.05, 40
    kx, ky = 3, 5
    vx = np.sin(math.pi * kx * np.arange(1, nx + 1) / (nx + 1))
    vy = np.sin(math.pi * ky * np.arange(1, ny + 1) / (ny + 1))
    psi = (vy[:, None] * vx[None, :]).astype(complex)
    lx = (1 - math.cos(math.pi * kx / (nx + 1))) / dx ** 2
    ly = (1 - math.cos(math.pi * ky / (ny + 1))) / dx ** 2
    ph = (((1 - 0.5j * lx * dt) / (1 + 0.5j * lx * dt)) * ((1 - 0.5j * ly * dt) / (1 + 0.5j * ly * dt))) ** steps
    out = O.step_2d(dx, dt, np.zeros(nx), np.zeros(ny), psi, steps)
    assert np.max(np.abs(out - ph * psi)) <= 1e-12


def test_step_2d_vs_dense():
    # catches: row/column stride mix-up, Vx/Vy swapped, order of the two sweeps
    nx, ny, dx, dt = 7, 5, 0.4, 0.1
    rng = np.random.default_rng(3)
    Vx, Vy = rng.uniform(-1, 1, nx), rng.uniform(-1, 1, ny)
    psi = rng.standard_normal((ny, nx)) + 1j * rng.standard_normal((ny, nx))
    Tx = np.eye(nx) + 0.5j * dt * hamiltonian_dense(dx, Vx)
    Ty = np.eye(ny) + 0.5j * dt * hamiltonian_dense(dx, Vy)
    ref = psi.copy()
    for _ in range(3):
        ref = np.linalg.solve(Tx, Tx.conj().T @ ref.T).T          # x sweep: every row
        ref = np.linalg.solve(Ty, Ty.conj().T @ ref)              # then y sweep: every column
    out = O.step_2d(dx, dt, Vx, Vy, psi, 3)
    assert np.max(np.abs(out - ref)) <= 1e-13


def test_step_2d_omp_is_bitwise_serial():
    # the multi-core timing copy (bench.py's C4 cpu_baseline) runs the unchanged per-system step: same bits, and the
    # dense reference of the test above pins it independently
    nx, ny, dx, dt = 37, 29, 0.3, 0.07
    rng = np.random.default_rng(5)
    Vx, Vy = rng.uniform(-1, 1, nx), rng.uniform(-1, 1, ny)
    psi = rng.standard_normal((ny, nx)) + 1j * rng.standard_normal((ny, nx))
    out, sec, threads = O.step_2d_omp(dx, dt, Vx, Vy, psi, 4)
    assert threads >= 1 and sec >= 0.0
    assert np.array_equal(out, O.step_2d(dx, dt, Vx, Vy, psi, 4))
    Tx = np.eye(nx) + 0.5j * dt * hamiltonian_dense(dx, Vx)
    Ty = np.eye(ny) + 0.5j * dt * hamiltonian_dense(dx, Vy)
    ref = psi.copy()
    for _ in range(4):
        ref = np.linalg.solve(Tx, Tx.conj().T @ ref.T).T
        ref = np.linalg.solve(Ty, Ty.conj().T @ ref)
    assert np.max(np.abs(out - ref)) <= 1e-13


# ---- invariants -----------------------------------------------------------------------------------
def test_norm_conservation_c1():
    cfg = W.CONFIGS["C1"]
    V, psi = W.potential(cfg), W.psi0(cfg)
    out = O.step(cfg.dx, cfg.dt, V, psi, 1000)
    n0, n1 = np.vdot(psi, psi).real, np.vdot(out, out).real
    assert abs(n1 / n0 - 1.0) <= 1e-12                          # north_star: 1e-12 per 1000 steps
    assert abs(n0 * cfg.dx - 1.0) <= 1e-12


def test_residual_every_step():
    cfg = W.scaled(W.CONFIGS["C1"], N=512, P=8)
    V, psi = W.potential(cfg), W.psi0(cfg)
    Tm = np.eye(cfg.N) + 0.5j * cfg.dt * hamiltonian_dense(cfg.dx, V)
    for _ in range(20):
        new = O.step(cfg.dx, cfg.dt, V, psi, 1)
        d = Tm.conj().T @ psi
        assert np.linalg.norm(Tm @ new - d) / np.linalg.norm(d) <= 1e-13
        psi = new


def test_rhs_is_T_dagger():
    n, dx, dt = 40, 0.2, 0.03
    rng = np.random.default_rng(5)
    V = rng.uniform(-1, 1, n)
    psi = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    Tm = np.eye(n) + 0.5j * dt * hamiltonian_dense(dx, V)
    b, a, c = O.diagonals(dx, dt, V)
    assert np.max(np.abs(O.rhs(b, a, c, psi) - Tm.conj().T @ psi)) <= 1e-14


def test_time_reversal():
    cfg = W.scaled(W.CONFIGS["C1"], N=1024, P=16)
    V, psi = W.potential(cfg), W.psi0(cfg)
    fwd = O.step(cfg.dx, cfg.dt, V, psi, 50)
    back = O.step(cfg.dx, -cfg.dt, V, fwd, 50)
    assert np.max(np.abs(back - psi)) <= 1e-12


def test_lean_equals_full():
    cfg = W.scaled(W.CONFIGS["C3"], N=1 << 14, P=64)
    V, psi = W.potential(cfg), W.psi0(cfg)
    a = O.step(cfg.dx, cfg.dt, V, psi, 7)
    b = O.step(cfg.dx, cfg.dt, V, psi, 7, lean=True)
    assert np.max(np.abs(a - b)) <= 1e-14


# ---- textbook physics: pins the sign and weight of the V term and of the kinetic term ----------------
def test_harmonic_coherent_state_trajectory():
    # <x>(t) = x0 cos t + k0 sin t for m = omega = 1 (Ehrenfest, exact for the harmonic oscillator);
    # a wrong sign of V or of i, or a missing 1/2, moves <x>(1) by O(1).  The reference is the exact
    # propagator exp(-i H t) of the SAME discrete H (dense eigh); CN with dt = 1e-3 is within O(dt^2) of it.
    n, dx, dt, steps, x0, k0 = 600, 0.05, 0.001, 1000, -5.0, 1.0
    x = (np.arange(n) - 0.5 * (n - 1)) * dx
    V = 0.5 * x * x
    psi = math.pi ** -0.25 * np.exp(-(x - x0) ** 2 / 2) * np.exp(1j * k0 * x)
    psi /= math.sqrt(np.vdot(psi, psi).real * dx)
    E, U = np.linalg.eigh(hamiltonian_dense(dx, V))
    exact = U @ (np.exp(-1j * E * dt * steps) * (U.T @ psi))
    out = O.step(dx, dt, V, psi, steps)                          # t = 1
    mean = lambda f: float(np.sum(x * np.abs(f) ** 2) * dx)
    assert abs(mean(exact) - (x0 * math.cos(1.0) + k0 * math.sin(1.0))) < 3e-2   # discrete H vs continuum
    assert abs(mean(out) - mean(exact)) < 1e-3
    assert np.max(np.abs(out - exact)) < 5e-3


def test_harmonic_ground_state_phase():
    # discrete ground state of H (dense eigh) must only pick up the Cayley phase of its eigenvalue
    n, dx, dt, steps = 200, 0.1, 0.01, 100
    x = (np.arange(n) - 0.5 * (n - 1)) * dx
    V = 0.5 * x * x
    E, U = np.linalg.eigh(hamiltonian_dense(dx, V))
    g = U[:, 0].astype(complex)
    assert abs(E[0] - 0.5) < 1e-3
    ph = ((1 - 0.5j * E[0] * dt) / (1 + 0.5j * E[0] * dt)) ** steps
    out = O.step(dx, dt, V, g, steps)
    assert np.max(np.abs(out - ph * g)) <= 1e-12


# ---- the method itself, stage by stage (Table 1 reconstruction) --------------------------------------
@pytest.mark.parametrize("n,nbl", [(9, 2), (10, 3), (40, 7), (8, 2), (64, 8), (65, 64), (33, 32), (12, 11)])
def test_table1_solves_the_system(n, nbl):
    # ragged blocks, single-interior-row blocks, adjacent joints
    b, a, c, d = rand_tridiag(n, 11 * n + nbl)
    J = T1.joints_paper(n, nbl)
    psi, st = T1.solve(b, a, c, d, J)
    ref = np.linalg.solve(dense_from(b, a, c), d)
    assert np.max(np.abs(psi - ref)) <= 1e-12
    assert np.max(np.abs(psi - O.thomas(b, a, c, d))) <= 1e-12
    assert len(st["support"]) == nbl + 1                         # reduced system of size n_bl + 1


def test_table1_typo():
    # PAPER.md:311 prints r_i = -T_{i,i-1}/T_{i,i}; with it the method does not solve the system (reading R2)
    n, nbl = 40, 4
    b, a, c, d = rand_tridiag(n, 77)
    ref = np.linalg.solve(dense_from(b, a, c), d)
    good, _ = T1.solve(b, a, c, d, T1.joints_paper(n, nbl))
    bad, _ = T1.solve(b, a, c, d, T1.joints_paper(n, nbl), multiplier="printed")
    assert np.max(np.abs(good - ref)) <= 1e-12
    assert np.max(np.abs(bad - ref)) > 1e-3


@pytest.mark.parametrize("n,nbl", [(9, 2), (16, 4), (25, 3)])
def test_stacked_N_sparsity(n, nbl):
    # after joining, non-zeros only on the diagonal and in columns J_w, on rows J_{w-1} <= i <= J_{w+1}
    b, a, c, d = rand_tridiag(n, 5 * n)
    J = T1.joints_paper(n, nbl)
    M = T1.dense_after_joining(dense_from(b, a, c), J)
    scale = np.abs(M).max()
    for i in range(1, n + 1):
        for j in range(1, n + 1):
            allowed = (i == j)
            for w, Jw in enumerate(J):
                lo = J[w - 1] if w > 0 else Jw
                hi = J[w + 1] if w < nbl else Jw
                if j == Jw and lo <= i <= hi:
                    allowed = True
            if not allowed:
                assert abs(M[i - 1, j - 1]) <= 1e-13 * scale, (i, j)
    # the joint rows alone form a tridiagonal system in the joint unknowns
    psi_ref = np.linalg.solve(dense_from(b, a, c), d)
    _, st = T1.solve(b, a, c, d, J)
    rb, ra, rc, rd = st["reduced"]
    sup = psi_ref[np.array(J) - 1]
    res = ra * sup + np.concatenate([[0], rb[1:] * sup[:-1]]) + np.concatenate([rc[:-1] * sup[1:], [0]]) - rd
    assert np.max(np.abs(res)) <= 1e-12 * max(1.0, np.abs(rd).max())


def test_uniform_padded_layout_equals_paper_layout():
    # DESIGN.md reading R8: pad with an identity row 0 (psi_0 = 0) and put joints at rows m, 2m, ..., n_tot
    n, nbl = 32, 4
    cfgV = np.linspace(-1, 2, n)
    b, a, c = O.diagonals(0.3, 0.05, cfgV)
    rng = np.random.default_rng(9)
    d = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    bp = np.concatenate([[0], b]); ap = np.concatenate([[1], a]); cp = np.concatenate([[0], c]); dp = np.concatenate([[0], d])
    psi_pad, _ = T1.solve(bp, ap, cp, dp, T1.joints_uniform(n, nbl))
    assert abs(psi_pad[0]) == 0.0
    assert np.max(np.abs(psi_pad[1:] - O.thomas(b, a, c, d))) <= 1e-13


def test_workloads_chunked_generation_is_bitwise_stable():
    cfg = W.scaled(W.CONFIGS["C2dense"], N=(1 << 21) + 13)
    full = W.psi0_unnormalised(cfg)
    parts = np.concatenate([W.psi0_unnormalised(cfg, s, min(cfg.N, s + 777_777)) for s in range(0, cfg.N, 777_777)])
    assert np.array_equal(full, parts)


# ---- values the paper prints (tests/golden/paper_operation_counts.txt) ---------------------------------------
def _golden():
    out = {}
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_operation_counts.txt")
    for line in open(path):
        line = line.split("#")[0].strip()
        if "=" in line:
            k, v = line.split("=")
            out[k.strip()] = float(v)
    return out


class _Counted:
    """complex scalar that counts the arithmetic done with it"""
    ops = {"div": 0, "mul": 0, "add": 0}

    def __init__(self, v):
        self.v = complex(v)

    @staticmethod
    def _v(o):
        return o.v if isinstance(o, _Counted) else complex(o)

    def __add__(self, o):
        _Counted.ops["add"] += 1
        return _Counted(self.v + self._v(o))
    __radd__ = __add__

    def __sub__(self, o):
        _Counted.ops["add"] += 1
        return _Counted(self.v - self._v(o))

    def __mul__(self, o):
        if isinstance(o, (int, float)) and o == 0:      # building zeros, not arithmetic of the method
            return _Counted(0)
        _Counted.ops["mul"] += 1
        return _Counted(self.v * self._v(o))
    __rmul__ = __mul__

    def __truediv__(self, o):
        _Counted.ops["div"] += 1
        return _Counted(self.v / self._v(o))

    def __rtruediv__(self, o):
        _Counted.ops["div"] += 1
        return _Counted(self._v(o) / self.v)

    def __neg__(self):
        return _Counted(-self.v)


def test_table1_operation_counts():
    """The reconstruction of the lost Table 1 (reading R1) costs what the paper says its method costs, PAPER.md:215:
    3 divisions, 9 multiplications, 6 additions per interior row.  A missing or extra term anywhere in RD/RU/SS
    changes one of the three counts."""
    from oracle import nshape_table1 as T1
    g = _golden()
    n, nbl = 241, 8                                   # J = 1, 31, 61, ...: 30 rows per block, 29 interior
    J = T1.joints_paper(n, nbl)
    V, rhs = W.random_system(n, seed=2)
    b, a, c = O.diagonals(0.1, 0.02, V)

    def counted(x):
        return np.array([_Counted(z) for z in x], dtype=object)

    def run(JJ):
        _Counted.ops = {"div": 0, "mul": 0, "add": 0}
        psi, _ = T1.solve(counted(b), counted(a), counted(c), counted(rhs), JJ)
        return dict(_Counted.ops), np.array([z.v for z in psi])

    ops1, psi1 = run(J)
    assert np.max(np.abs(psi1 - O.thomas(b, a, c, rhs))) < 1e-12
    # growing every block by 10 interior rows isolates the per-interior-row cost from the per-block / RS cost
    n2 = n + 10 * nbl
    V2, rhs2 = W.random_system(n2, seed=2)
    b2, a2, c2 = O.diagonals(0.1, 0.02, V2)
    b, a, c, rhs = b2, a2, c2, rhs2
    ops2, _ = run(T1.joints_paper(n2, nbl))
    per_row = {k: (ops2[k] - ops1[k]) / (10 * nbl) for k in ops1}
    assert per_row["div"] == g["divisions_per_interior_row"]
    assert per_row["mul"] == g["multiplications_per_interior_row"]
    assert per_row["add"] == g["additions_per_interior_row"]


def test_performance_model_optimum():
    """Eq. 7: t = alpha n_tot / n_bl + beta n_bl is minimal at n_bl* = sqrt(alpha/beta) sqrt(n_tot),
    where t* = 2 sqrt(alpha beta n_tot) -- the formula the P sweep of config C2 is compared with."""
    g = _golden()
    alpha, beta = 1.41e-6, 0.36e-6
    for ntot in (3e5, 2.0 ** 24, 2.0 ** 30):
        P = np.arange(1, 200000, dtype=np.float64)
        t = alpha * ntot / P + beta * P
        k = int(np.argmin(t))
        pstar = math.sqrt(alpha / beta) * ntot ** g["model_optimum_exponent"]
        assert abs(P[k] - pstar) <= 1.0
        assert abs(t[k] - 2 * math.sqrt(alpha * beta * ntot)) / t[k] < 1e-8


# ---- time-dependent H: oracle/cn_oracle.step_td ---------------------------------------------------
def test_td_uniform_shift_closed_form():
    """g = 1 (spatially uniform f(t)): T_k = T0 + i dt/2 f_k commutes with the Laplacian, so a Dirichlet sine mode is
    multiplied at step k by the exact Cayley phase of lambda + f_k -- a closed form that pins the midpoint rule, the
    sign of i and the order of the steps independently of the code."""
    N, dx, dt = 97, 0.13, 0.021
    rng = np.random.default_rng(5)
    field = rng.uniform(-3.0, 3.0, 40)
    j = np.arange(1, N + 1)
    for k in (1, 5, N):
        v = np.sin(np.pi * k * j / (N + 1)).astype(np.complex128)
        lam = (1.0 - np.cos(np.pi * k / (N + 1))) / dx ** 2
        phase = np.prod((1 - 0.5j * dt * (lam + field)) / (1 + 0.5j * dt * (lam + field)))
        out = O.step_td(dx, dt, np.zeros(N), np.ones(N), field, v)
        assert np.max(np.abs(out - phase * v)) <= 1e-12


def test_td_dense_lu_per_step_and_norm():
    N, dx, dt = 48, 0.2, 0.05
    rng = np.random.default_rng(6)
    V0, g = rng.uniform(-1, 1, N), rng.uniform(-2, 2, N)
    field = rng.uniform(-1, 1, 7)
    psi = rng.normal(size=N) + 1j * rng.normal(size=N)
    ref = psi.copy()
    lap = (np.diag(np.full(N, 2.0)) - np.diag(np.ones(N - 1), 1) - np.diag(np.ones(N - 1), -1)) / (2 * dx * dx)
    for f in field:  # H typed out here, dense solve per step
        H = lap + np.diag(V0 + f * g)
        ref = np.linalg.solve(np.eye(N) + 0.5j * dt * H, (np.eye(N) - 0.5j * dt * H) @ ref)
    out = O.step_td(dx, dt, V0, g, field, psi)
    assert np.max(np.abs(out - ref)) <= 1e-12
    assert abs(np.vdot(out, out).real / np.vdot(psi, psi).real - 1.0) <= 1e-12
    # field = 0 is the static stepper
    assert np.array_equal(O.step_td(dx, dt, V0, g, np.zeros(5), psi), O.step(dx, dt, V0, psi, 5))
