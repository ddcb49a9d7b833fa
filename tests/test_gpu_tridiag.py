"""General complex tridiagonal front end (cn_tridiag_*; Eq. 5) against the oracle's plain
serial Thomas solve (oracle.thomas, pinned by dense LU in test_oracle_pins.py) on seeded random systems with
NON-constant complex off-diagonals.  Tolerance: the static path's residual bar, relative 1e-12, and 1e-10 on x."""
import numpy as np
import pytest

from oracle import cn_oracle as O
from paper_2205_00856_b200 import binding as B

pytestmark = pytest.mark.gpu


def system(n, seed, dominance=2.5):
    rng = np.random.default_rng(seed)
    z = lambda: rng.normal(size=n) + 1j * rng.normal(size=n)
    b, c, d = z(), z(), z()
    # strictly diagonally dominant (no pivoting anywhere, as in the paper), random phase on the diagonal
    a = (np.abs(b) + np.abs(c)) * dominance * np.exp(1j * rng.uniform(0, 2 * np.pi, n)) + 0.1 * z()
    return b, a, c, d


def residual(b, a, c, d, x):
    r = a * x - d
    r[1:] += b[1:] * x[:-1]
    r[:-1] += c[:-1] * x[1:]
    return np.linalg.norm(r) / np.linalg.norm(d)


# 1 level (<= 4096 rows, every K of the single-CTA kernel), 2 levels (ragged last group, single-row last group), 3 levels
SIZES = [1, 2, 3, 31, 255, 256, 257, 1000, 4096, 4097, 65536, 70001, 256 * 300 + 1, (1 << 20) + 3, 256 * 4097]


@pytest.mark.parametrize("n", SIZES)
def test_tridiag_random(n):
    import torch
    b, a, c, d = system(n, seed=100 + n % 97)
    ref = O.thomas(b, a, c, d)
    dd = torch.from_numpy(d).cuda()
    xx = torch.empty_like(dd)
    with B.Tridiag(b, a, c) as t:
        t.solve(dd, xx)
        torch.cuda.synchronize()
        x = xx.cpu().numpy()
        assert np.max(np.abs(x - ref)) <= 1e-10 * max(1.0, np.max(np.abs(ref)))
        assert residual(b, a, c, d, x) <= 1e-12
        # in place, device-resident coefficients, several right-hand sides with one factorization
        for k in range(3):
            d2 = np.roll(d, k + 1) * (1 + k)
            buf = torch.from_numpy(d2).cuda()
            t.solve(buf)
            torch.cuda.synchronize()
            assert residual(b, a, c, d2, buf.cpu().numpy()) <= 1e-12
    with B.Tridiag(torch.from_numpy(b).cuda(), torch.from_numpy(a).cuda(), torch.from_numpy(c).cuda()) as t2:
        t2.solve(dd, xx)
        torch.cuda.synchronize()
        assert np.array_equal(xx.cpu().numpy(), x)


def test_tridiag_is_the_cn_matrix():
    """With b = c = -i s and a = 1 + i (2 s + dt V / 2) the front end solves Eq. 4 of the paper: same psi as the stepper."""
    import torch
    from paper_2205_00856_b200 import workloads as W
    cfg = W.scaled(W.CONFIGS["C1"], N=1 << 15)
    V, psi = W.potential(cfg), W.psi0(cfg)
    b, a, c = O.diagonals(cfg.dx, cfg.dt, V)
    d = O.rhs(b, a, c, psi)
    with B.Tridiag(b, a, c) as t:
        x = t.solve(torch.from_numpy(d).cuda())
        torch.cuda.synchronize()
    assert np.max(np.abs(x.cpu().numpy() - O.step(cfg.dx, cfg.dt, V, psi, 1))) <= 1e-10


def test_tridiag_breakdown_and_errors():
    n = 600
    b, a, c, d = system(n, 7)
    a[300] = 0.0
    b[300] = 0.0
    c[299] = 0.0
    a[299] = 1.0  # row 300 is all zero: a zero pivot whatever the partition
    c[300] = 0.0
    with pytest.raises(B.CnError) as e:
        B.Tridiag(b, a, c)
    assert e.value.status == B.CN_EBREAKDOWN
    assert B.lib().cn_tridiag_solve(None, None, None, None) == B.CN_EINVAL
    assert B.lib().cn_tridiag_destroy(None) == B.CN_EINVAL


def ragged_joints(n, kind, seed):
    """caller-placed joint lines (blocks may differ in size); always end at row n - 1"""
    rng = np.random.default_rng(seed)
    if kind == "single":            # one block: the whole system is the interior of the last row's block
        return [n - 1]
    if kind == "every_row":         # every row is a joint line (blocks of one row, no interior anywhere)
        return list(range(n))
    if kind == "pairs":             # blocks of two rows: one interior row each (+ a one-row block if n is odd)
        return sorted(set(list(range(1, n, 2)) + [n - 1]))
    if kind == "paper":             # the paper's literal placement J_w = round(w (n - 1) / P), P ~ sqrt(n)
        P = max(1, int(round(n ** 0.5)))
        return sorted(set(int(round(w * (n - 1) / P)) for w in range(1, P + 1)))
    # random unequal blocks of 1 .. ~3 sqrt(n) rows, with some runs of adjacent joint lines
    out, j = [], -1
    top = max(2, int(3 * n ** 0.5))
    while True:
        j += int(rng.integers(1, top)) if rng.random() > 0.2 else 1
        if j >= n - 1:
            break
        out.append(j)
    return out + [n - 1]


@pytest.mark.parametrize("n,kind", [(1, "single"), (2, "every_row"), (2, "single"), (9, "random"), (10, "pairs"),
                                    (40, "random"), (257, "paper"), (1000, "every_row"), (4096, "random"),
                                    (4097, "pairs"), (70001, "random"), (300000, "paper"), (300000, "single"),
                                    ((1 << 20) + 3, "random"), ((1 << 21), "pairs")])
def test_tridiag_caller_placed_joints(n, kind):
    """The same solve with the joint lines where the CALLER puts them: x does not depend on the partition."""
    import torch
    if kind == "single" and n > 100000:
        n = 50000  # one thread sweeps the whole system: keep it short
    b, a, c, d = system(n, seed=300 + n % 89)
    ref = O.thomas(b, a, c, d)
    J = ragged_joints(n, kind, seed=n)
    assert J[-1] == n - 1 and all(J[i] < J[i + 1] for i in range(len(J) - 1))
    dd = torch.from_numpy(d).cuda()
    xx = torch.empty_like(dd)
    with B.Tridiag(b, a, c, joints=J) as t:
        t.solve(dd, xx)
        torch.cuda.synchronize()
        x = xx.cpu().numpy()
        assert np.max(np.abs(x - ref)) <= 1e-10 * max(1.0, np.max(np.abs(ref)))
        assert residual(b, a, c, d, x) <= 1e-12
        buf = torch.from_numpy(d).cuda()   # in place (x aliases d)
        t.solve(buf)
        t.solve(dd, xx)                    # and again: the factors are not consumed
        torch.cuda.synchronize()
        assert np.array_equal(buf.cpu().numpy(), x) and np.array_equal(xx.cpu().numpy(), x)


def test_tridiag_joints_rejected():
    n = 100
    b, a, c, d = system(n, 5)
    for J in ([10, 5, 99], [10, 10, 99], [10, 50], [-1, 99], [10, 100], []):
        with pytest.raises((B.CnError, ValueError)) as e:
            B.Tridiag(b, a, c, joints=J)
        if isinstance(e.value, B.CnError):
            assert e.value.status == B.CN_EINVAL
