"""BASELINE.json configs C3, C4, C5 at FULL size in the launch configuration a user gets by default, against the
oracle element by element: C5 after all its 10 steps; C3 after 3 steps on every element and after all its 50 steps on
the windows and full-vector checksums of the oracle-written golden file (tests/golden/make_c3_golden.py: 50 lean-oracle
steps at N = 2^30 take ~25 min); C4 after 2 steps here and after all 20 in test_gpu_zz_fullsteps.py (with C2 x 1000).
Plus the size-independent properties (norm, residual of one solve on sampled windows).
These tests need ~80 GB of host memory and a few minutes."""
import math
import os
import sys
import time

import numpy as np
import pytest

from oracle import cn_oracle as O
from paper_2205_00856_b200 import binding as B
from paper_2205_00856_b200 import workloads as W

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden"))
import make_c3_golden as G3  # noqa: E402  (oracle side: window positions and checksum weights of the golden file)

pytestmark = pytest.mark.gpu
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "c3_golden.npz")
TOL_PSI = 1e-10
TOL_RES = 1e-12


def torch_():
    import torch
    return torch


def host_gb():
    try:
        with open("/proc/meminfo") as f:
            for line in f:
                if line.startswith("MemAvailable"):
                    return int(line.split()[1]) / 2 ** 20
    except OSError:
        pass
    return 0.0


def build_inputs(cfg, chunk=1 << 24):
    """V and psi0 chunk by chunk (bit-identical to the one-shot generators, see test_oracle_pins)."""
    V = np.empty(cfg.N, np.float64)
    psi = np.empty(cfg.N, np.complex128)
    norm = W.psi0_norm2(cfg)
    for s in range(0, cfg.N, chunk):
        e = min(cfg.N, s + chunk)
        V[s:e] = W.potential(cfg, s, e)
        psi[s:e] = W.psi0(cfg, s, e, norm=norm)
    return V, psi


def window_residual(dx, dt, V, old, new, lo, hi):
    """|| (T new - T^dagger old)[lo:hi] || / || (T^dagger old)[lo:hi] || by a numpy stencil typed here (not the oracle);
    rows lo..hi-1 need their neighbours lo-1 and hi, taken from the full arrays."""
    n = V.size
    a, b = max(lo - 1, 0), min(hi + 1, n)
    s = dt / (4 * dx * dx)
    diag = 1 + 1j * (2 * s + 0.5 * dt * V[a:b])

    def apply(dg, off, x):
        y = dg * x
        y[1:] += off * x[:-1]
        y[:-1] += off * x[1:]
        return y
    d = apply(np.conj(diag), 1j * s, old[a:b])
    r = apply(diag, -1j * s, new[a:b]) - d
    sl = slice(lo - a, hi - a)
    return np.linalg.norm(r[sl]) / np.linalg.norm(d[sl])


def test_config_c3_full_size():
    """N = 2^30 (psi 17 GB + factors 26 GB on the device).  P from the paper's P* = delta sqrt(N)
    with the delta fitted on C2's paper-literal sweep: P = 2^16, which the tiled path partitions again.
    After 1 step: residual windows; after 3 steps: every element against the lean oracle; after the config's 50 steps:
    the oracle-written golden file (9 windows of 2^16 points element by element at 1e-10, the full-vector norm, and the
    full-vector weighted checksum with tolerance 1e-10 * sum |w_j| |psi_j| -- what an elementwise error of 1e-10 moves)."""
    torch = torch_()
    assert host_gb() >= 85, "needs ~85 GB of host memory"
    assert os.path.exists(GOLDEN), "tests/golden/c3_golden.npz is missing: run tests/golden/make_c3_golden.py"
    gold = np.load(GOLDEN)
    cfg = W.CONFIGS["C3"]
    assert int(gold["N"]) == cfg.N and int(gold["steps"]) == cfg.steps and int(gold["seed"]) == cfg.seed
    assert float(gold["dx"]) == cfg.dx and float(gold["dt"]) == cfg.dt
    t0 = time.time()
    V, psi = build_inputs(cfg)
    t_gen = time.time() - t0
    d = torch.from_numpy(psi).cuda()
    with B.Plan(cfg.N, cfg.P, cfg.dx, cfg.dt, V) as plan:
        plan.factorize()
        info = plan.info()
        assert info["path"] == B.PATH_TILED and info["rs_levels"] >= 3
        # one solve: residual on windows sampled over the whole grid (incl. both ends and a tile boundary)
        plan.step(d, 1)
        torch.cuda.synchronize()
        out = d.cpu().numpy()
        for lo in (0, 2048 - 7, cfg.N // 3, cfg.N // 2 - 1000, cfg.N - (1 << 20)):
            assert window_residual(cfg.dx, cfg.dt, V, psi, out, lo, lo + (1 << 20)) <= TOL_RES
        # the oracle (lean variant, 34 GB) for the first 3 steps, every element
        nref = 3
        t0 = time.time()
        ref = psi
        O.step_inplace(cfg.dx, cfg.dt, V, ref, nref, lean=True)
        t_or = time.time() - t0
        plan.step(d, nref - 1)
        torch.cuda.synchronize()
        torch.from_numpy(out).copy_(d)
        err = 0.0
        for s in range(0, cfg.N, 1 << 26):
            err = max(err, float(np.max(np.abs(out[s:s + (1 << 26)] - ref[s:s + (1 << 26)]))))
        assert err <= TOL_PSI, err
        del ref, psi, V
        # the remaining steps of the config, then the golden file
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        plan.step(d, cfg.steps - nref)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / (cfg.steps - nref)
    starts = [int(s) for s in gold["starts"]]
    assert starts == G3.window_starts(cfg.N, cfg.dx, cfg.x0)
    worst = 0.0
    for s, win in zip(starts, gold["windows"]):
        worst = max(worst, float(np.max(np.abs(d[s:s + win.size].cpu().numpy() - win))))
    torch.from_numpy(out).copy_(d)
    del d
    n2, dot, scale = G3.checksums(out, cfg.seed)
    print("\nC3: gen %.0fs oracle %.1fs/step, GPU %.3f ms/step = %.1f Gpt-steps/s, 3 steps max|dpsi| %.2e, P_eff %d; "
          "%d steps vs golden: windows max|dpsi| %.2e, |norm - 1| %.1e, checksum diff %.2e (allowed %.2e), golden oracle %.0f s"
          % (t_gen, t_or / nref, ms, cfg.N / ms / 1e6, err, info["P_effective"], cfg.steps, worst,
             abs(n2 * cfg.dx - 1.0), abs(dot - float(gold["wdot"])), TOL_PSI * scale, float(gold["oracle_seconds"])))
    assert worst <= TOL_PSI, worst
    assert abs(n2 * cfg.dx - 1.0) <= 1e-12, n2 * cfg.dx
    assert abs(n2 - float(gold["norm2"])) <= 1e-12 * float(gold["norm2"]), (n2, float(gold["norm2"]))
    assert abs(dot - float(gold["wdot"])) <= TOL_PSI * scale, (dot, float(gold["wdot"]), scale)


def test_config_c4_full_size():
    """8192 x 8192, x-sweep then y-sweep per step (reading R18), 20 steps; oracle for the first 2 steps."""
    torch = torch_()
    cfg = W.CONFIGS["C4"]
    n = cfg.N
    psi = W.psi0_2d(cfg)
    Vx, Vy = W.potential(cfg), W.potential_y(cfg)
    nref = 2
    t0 = time.time()
    ref = O.step_2d(cfg.dx, cfg.dt, Vx, Vy, psi, nref)
    t_or = time.time() - t0
    d = torch.from_numpy(psi).cuda()
    with B.Plan(n, cfg.P, cfg.dx, cfg.dt, Vx) as px, B.Plan(n, cfg.P, cfg.dx, cfg.dt, Vy) as py:
        px.factorize()
        py.factorize()

        def steps(k):
            for _ in range(k):
                px.batched_sweep(d, n, 1, n, 1)
                py.batched_sweep(d, n, n, 1, 1)
        steps(nref)
        torch.cuda.synchronize()
        err = float(np.max(np.abs(d.cpu().numpy() - ref)))
        assert err <= TOL_PSI, err
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        steps(cfg.steps - nref)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / (cfg.steps - nref)
        nrm = float((d.real.square().sum() + d.imag.square().sum()).item()) * cfg.dx * cfg.dx
        assert abs(nrm - 1.0) <= 1e-12, nrm
    print("\nC4: oracle %.1fs/step, GPU %.3f ms per 2-D step = %.1f Gpoint-sweeps/s, max|dpsi| %.2e"
          % (t_or / nref, ms, 2 * n * n / ms / 1e6, err))


def test_config_c5_full_size():
    """N = 2^29 in pinned host memory, device budget 2 GB, 10 steps; oracle (lean) for all 10 steps."""
    torch = torch_()
    assert host_gb() >= 55, "needs ~55 GB of host memory"
    cfg = W.CONFIGS["C5"]
    V, psi = build_inputs(cfg)
    h = torch.from_numpy(psi).pin_memory()
    budget = 2 << 30
    with B.Plan(cfg.N, cfg.P, cfg.dx, cfg.dt, V, device_budget=budget) as plan:
        plan.factorize()
        info = plan.info()
        assert info["out_of_core"] == 1 and info["device_bytes"] <= budget, info
        t0 = time.time()
        plan.step(h, cfg.steps)
        torch.cuda.synchronize()
        t_gpu = time.time() - t0
    t0 = time.time()
    O.step_inplace(cfg.dx, cfg.dt, V, psi, cfg.steps, lean=True)
    t_or = time.time() - t0
    out = h.numpy()
    err = 0.0
    for s in range(0, cfg.N, 1 << 26):
        err = max(err, float(np.max(np.abs(out[s:s + (1 << 26)] - psi[s:s + (1 << 26)]))))
    assert err <= TOL_PSI, err
    nrm = float(np.vdot(out, out).real) * cfg.dx
    assert abs(nrm - 1.0) <= 1e-12, nrm
    gb = cfg.N * (24 * (cfg.steps + 1)) / 1e9
    print("\nC5: oracle %.1fs/step, GPU %.3f s/step = %.2f Gpt-steps/s, H2D %.1f GB/s, device bytes %.2f GB, part %d pts, "
          "max|dpsi| %.2e" % (t_or / cfg.steps, t_gpu / cfg.steps, cfg.N * cfg.steps / t_gpu / 1e9, gb / t_gpu,
                              info["device_bytes"] / 2 ** 30, info["tile_points"], err))
