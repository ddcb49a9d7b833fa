"""Every BASELINE.json config against the oracle AFTER THE CONFIG'S FULL STEP COUNT (`north_star`: "max elementwise
|dpsi| <= 1e-10 after the config's step count"), in the launch configuration a user gets by default and bench.py times.

  C1  100 steps   tests/test_gpu_parity.py::test_config_c1_both_paths
  C2  1000 steps  here: every element, oracle run on a background thread of the session (tests/conftest.py)
  C3  50 steps    tests/test_gpu_fullsize.py::test_config_c3_full_size: the oracle-written golden file
                  tests/golden/c3_golden.npz (make_c3_golden.py: 9 windows of 2^16 points compared element by element +
                  two full-vector checksums; the 50 lean-oracle steps take ~25 min), and every element after 3 steps
  C4  20 steps    here: every element, oracle on a background thread
  C5  10 steps    tests/test_gpu_fullsize.py::test_config_c5_full_size (every element)

The file name sorts last so that the background oracle runs overlap the rest of the GPU session."""
import numpy as np
import pytest

from paper_2205_00856_b200 import binding as B
from paper_2205_00856_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL_PSI = 1e-10


def torch_():
    import torch
    return torch


def test_config_c2_all_steps(oracle_jobs):
    """C2 (dense twin, N = 2^24, P = 2^16): 1000 steps as 10 cn_step calls of 100 (what bench.py issues), every element
    against 1000 oracle steps; norm to the oracle's own pin (1e-12 per 1000 steps)."""
    torch = torch_()
    cfg = W.CONFIGS["C2dense"]
    V, psi, ref, sec = oracle_jobs.result("c2_full")
    d = torch.from_numpy(psi).cuda()
    with B.Plan(cfg.N, cfg.P, cfg.dx, cfg.dt, V) as plan:
        plan.factorize()
        info = plan.info()
        assert info["path"] == B.PATH_TILED and info["rs_levels"] >= 2
        for _ in range(cfg.steps // 100):
            plan.step(d, 100)
        torch.cuda.synchronize()
    out = d.cpu().numpy()
    err = float(np.max(np.abs(out - ref)))
    nrm = float(np.vdot(out, out).real) * cfg.dx
    print("\nC2 x %d steps: max|dpsi| %.2e, |norm - 1| %.1e, oracle %.0f s (%.1f ns per point-step, 1 core)"
          % (cfg.steps, err, abs(nrm - 1.0), sec, 1e9 * sec / (cfg.N * cfg.steps)))
    assert err <= TOL_PSI, err
    assert abs(nrm - 1.0) <= 1e-12, nrm


def test_config_c4_all_steps(oracle_jobs):
    """C4 (8192 x 8192, x-sweep then y-sweep per step, reading R18): all 20 steps, every element."""
    torch = torch_()
    cfg = W.CONFIGS["C4"]
    n = cfg.N
    Vx, Vy, psi, ref, sec = oracle_jobs.result("c4_full")
    d = torch.from_numpy(psi).cuda()
    with B.Plan(n, cfg.P, cfg.dx, cfg.dt, Vx) as px, B.Plan(n, cfg.P, cfg.dx, cfg.dt, Vy) as py:
        px.factorize()
        py.factorize()
        for _ in range(cfg.steps):
            px.batched_sweep(d, n, 1, n, 1)
            py.batched_sweep(d, n, n, 1, 1)
        torch.cuda.synchronize()
    out = d.cpu().numpy()
    err = float(np.max(np.abs(out - ref)))
    nrm = float(np.vdot(out, out).real) * cfg.dx * cfg.dx
    print("\nC4 x %d steps: max|dpsi| %.2e, |norm - 1| %.1e, oracle %.0f s (%.1f ns per point-sweep, 1 core)"
          % (cfg.steps, err, abs(nrm - 1.0), sec, 1e9 * sec / (2.0 * n * n * cfg.steps)))
    assert err <= TOL_PSI, err
    assert abs(nrm - 1.0) <= 1e-12, nrm
