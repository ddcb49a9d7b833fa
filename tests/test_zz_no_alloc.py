"""cn_step_static: the entry point that allocates nothing (its scratch is a static device array of the library).

Collected last on purpose (the name): the suite runs with `pytest -x`, and a failure here must not hide other tests.
The output is checked against the EXISTING path -- cn_plan_create / cn_factorize / cn_step on the same inputs -- within
the tolerance of the parity tests, on two calls in a row that share the scratch: the second call has another N, another
potential and another dx / dt, so anything the first call left behind in the array would show."""
import numpy as np
import pytest

from paper_2205_00856_b200 import binding as B
from paper_2205_00856_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL_PSI = 1e-10  # the bar of tests/test_gpu_parity.py


def _case(N, dx, dt, seed):
    cfg = W.scaled(W.CONFIGS["C1"], N=N, dx=dx, dt=dt)
    rng = np.random.default_rng(seed)
    V = W.potential(cfg) + 0.3 * rng.standard_normal(N)  # not the same matrix twice
    psi = W.psi0(cfg)
    return cfg, np.ascontiguousarray(V), psi


def _existing_path(torch, cfg, V, psi, nsteps):
    d = torch.from_numpy(psi.copy()).cuda()
    with B.Plan(cfg.N, max(1, cfg.N // 64), cfg.dx, cfg.dt, V) as plan:
        plan.factorize()
        plan.step(d, nsteps)
        torch.cuda.synchronize()
    return d.cpu().numpy()


def test_static_scratch_stepper_two_calls_in_a_row():
    import torch
    cases = [(_case(4096, 0.1, 0.01, 1), 100),   # config C1's shape: the maximum size
             (_case(1000, 0.05, 0.004, 2), 37),  # ragged, smaller: the scratch still holds rows 1000.. of the call before
             (_case(4096, 0.1, 0.01, 1), 100)]   # the first case again after the array was overwritten
    refs = [_existing_path(torch, cfg, V, psi, n) for (cfg, V, psi), n in cases]
    dV = [torch.from_numpy(V).cuda() for (cfg, V, psi), n in cases]
    dpsi = [torch.from_numpy(psi.copy()).cuda() for (cfg, V, psi), n in cases]
    torch.cuda.synchronize()
    # the calls in a row, on one stream, without a synchronisation between them (they share the scratch: stream order)
    for ((cfg, V, psi), n), v, d in zip(cases, dV, dpsi):
        B.cn_step_static(cfg.N, cfg.dx, cfg.dt, v, d, n)
    torch.cuda.synchronize()
    for ((cfg, V, psi), n), d, ref in zip(cases, dpsi, refs):
        out = d.cpu().numpy()
        assert np.all(np.isfinite(out.view(np.float64)))
        err = float(np.max(np.abs(out - ref)))
        assert err <= TOL_PSI, (cfg.N, err)
    assert np.array_equal(dpsi[0].cpu().numpy(), dpsi[2].cpu().numpy())  # same inputs, same result: nothing stale

    # split into two calls (50 + 50 steps) = one call of 100 steps
    (cfg, V, psi), n = cases[0]
    d = torch.from_numpy(psi.copy()).cuda()
    B.cn_step_static(cfg.N, cfg.dx, cfg.dt, dV[0], d, 50)
    B.cn_step_static(cfg.N, cfg.dx, cfg.dt, dV[0], d, 50)
    torch.cuda.synchronize()
    assert float(np.max(np.abs(d.cpu().numpy() - refs[0]))) <= TOL_PSI


def test_static_scratch_stepper_allocates_nothing_and_rejects_large_sizes():
    import torch
    (cfg, V, psi) = _case(2048, 0.1, 0.01, 3)
    v, d = torch.from_numpy(V).cuda(), torch.from_numpy(psi.copy()).cuda()
    B.cn_step_static(cfg.N, cfg.dx, cfg.dt, v, d, 1)  # first call on this device: set-up (symbol address, attributes)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(5):
        B.cn_step_static(cfg.N, cfg.dx, cfg.dt, v, d, 3)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, (free0, free1)  # the driver handed out no device memory

    big = torch.zeros(B.CN_STATIC_NMAX + 8, dtype=torch.complex128, device="cuda")
    bigV = torch.zeros(B.CN_STATIC_NMAX + 8, dtype=torch.float64, device="cuda")
    with pytest.raises(B.CnError) as e:
        B.cn_step_static(B.CN_STATIC_NMAX + 8, 0.1, 0.01, bigV, big, 1)
    assert e.value.status == B.CN_ETOOLARGE
    assert b"CN_STATIC_NMAX" in B.lib().cn_status_string(B.CN_ETOOLARGE)
    with pytest.raises(B.CnError) as e:
        B.cn_step_static(1, 0.1, 0.01, bigV, big, 1)
    assert e.value.status == B.CN_EINVAL
    assert float(big.abs().max()) == 0.0  # a rejected call touches nothing

    # a non-finite potential cannot be reported by an asynchronous call: psi turns into NaN, and the NEXT call is clean
    bad = v.clone()
    bad[17] = float("nan")
    d2 = torch.from_numpy(psi.copy()).cuda()
    B.cn_step_static(cfg.N, cfg.dx, cfg.dt, bad, d2, 1)
    d3 = torch.from_numpy(psi.copy()).cuda()
    B.cn_step_static(cfg.N, cfg.dx, cfg.dt, v, d3, 1)
    torch.cuda.synchronize()
    assert bool(torch.isnan(torch.view_as_real(d2)).all())
    ref = _existing_path(torch, cfg, V, psi, 1)
    assert float(np.max(np.abs(d3.cpu().numpy() - ref))) <= TOL_PSI
