"""Parity of the CUDA path (through the C-ABI) with the oracle, element by element, on the same seeded
inputs.  Tolerances are BASELINE.json's: max |dpsi| <= 1e-10 after the config's step count, relative
residual <= 1e-12 per solve."""
import math

import numpy as np
import pytest

from oracle import cn_oracle as O
from paper_2205_00856_b200 import binding as B
from paper_2205_00856_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL_PSI = 1e-10
TOL_RES = 1e-12


def torch_():
    import torch
    return torch


def gpu_step(N, P, dx, dt, V, psi, nsteps, path=B.PATH_AUTO, tile_threads=0, calls=1, **opts):
    torch = torch_()
    d_psi = torch.from_numpy(np.ascontiguousarray(psi)).cuda()
    with B.Plan(N, P, dx, dt, np.ascontiguousarray(V), path=path, tile_threads=tile_threads, **opts) as plan:
        plan.factorize()
        for _ in range(calls):
            plan.step(d_psi, nsteps)
        torch.cuda.synchronize()
        info = plan.info()
    return d_psi.cpu().numpy(), info


def residual(dx, dt, V, old, new):
    """|| T new - T^dagger old || / || T^dagger old || with T applied as a stencil in numpy (not the oracle)."""
    s = dt / (4 * dx * dx)
    a = 1 + 1j * (2 * s + 0.5 * dt * V)

    def apply(diag, off, x):
        y = diag * x
        y[1:] += off * x[:-1]
        y[:-1] += off * x[1:]
        return y
    d = apply(np.conj(a), 1j * s, old)
    r = apply(a, -1j * s, new) - d
    return np.linalg.norm(r) / np.linalg.norm(d)


GENERIC_SHAPES = [(2, 1), (2, 2), (9, 2), (10, 3), (40, 7), (64, 64), (65, 32), (33, 33), (100, 1), (1000, 37),
                  (4096, 64), (5000, 123), (777, 776)]


@pytest.mark.parametrize("N,P", GENERIC_SHAPES)
def test_generic_path_random(N, P):
    # ragged blocks, blocks of one interior row, joint-only blocks (m = 1), a single block
    V, psi = W.random_system(N, seed=17)
    dx, dt = 0.2, 0.03
    for nsteps in (1, 4):
        ref = O.step(dx, dt, V, psi, nsteps)
        out, info = gpu_step(N, P, dx, dt, V, psi, nsteps, path=B.PATH_GENERIC)
        assert info["path"] == B.PATH_GENERIC
        assert np.max(np.abs(out - ref)) <= TOL_PSI, (N, P, nsteps)
    out1, _ = gpu_step(N, P, dx, dt, V, psi, 1, path=B.PATH_GENERIC)
    assert residual(dx, dt, V, psi, out1) <= TOL_RES


TILED_SHAPES = [
    # (N, P, tile_threads)   m = N/P must be 8 * 2^k
    (64, 8, 0), (64, 1, 0), (256, 1, 0), (2048, 1, 0), (4096, 1, 512), (4096, 64, 0), (4096, 64, 128),
    (4096, 64, 512), (1 << 16, 1 << 13, 0), (1 << 16, 1 << 12, 0), (1 << 16, 1 << 11, 128), (1 << 16, 1 << 10, 0),
    (1 << 16, 1 << 9, 0), (1 << 16, 1 << 8, 0), (1 << 16, 1 << 7, 512), (1 << 16, 1 << 6, 0), (1 << 16, 1 << 5, 0),
    (1 << 16, 1 << 4, 512), (6656, 26, 0), (6656, 26, 128), (8 * 1000, 1000, 0), (2048 * 3 + 512, 13, 0),
    (2048 * 5 + 1024, 11, 0), (4096, 64, 32), (4096, 64, 64), (1 << 16, 1 << 13, 32), (1 << 16, 1 << 8, 32), (1 << 16, 1 << 9, 64),
    (6656, 26, 64), (6656 + 256, 27, 32), (1 << 16, 1 << 7, 64),
]


@pytest.mark.parametrize("keep_p", [1, 0])
@pytest.mark.parametrize("N,P,tt", TILED_SHAPES)
def test_tiled_path_random(N, P, tt, keep_p):
    # several tiles and a ragged last tile; every scan depth (block inside a warp, across warps: keep_p = 1 keeps the
    # caller's blocks of 512..4096 rows, keep_p = 0 partitions them again into blocks of 256 rows)
    V, psi = W.random_system(N, seed=23)
    dx, dt = 0.1, 0.02
    for nsteps in (1, 3):
        ref = O.step(dx, dt, V, psi, nsteps)
        out, info = gpu_step(N, P, dx, dt, V, psi, nsteps, path=B.PATH_TILED, tile_threads=tt, keep_p=keep_p)
        assert info["path"] == B.PATH_TILED
        if keep_p or N // P <= 256:
            assert info["P_effective"] == P
        else:
            assert info["P_effective"] == N // 256
        err = np.max(np.abs(out - ref))
        assert err <= TOL_PSI, (N, P, tt, nsteps, err)
    out1, _ = gpu_step(N, P, dx, dt, V, psi, 1, path=B.PATH_TILED, tile_threads=tt, keep_p=keep_p)
    assert residual(dx, dt, V, psi, out1) <= TOL_RES


AUTO_PARTITION_CASES = [
    # (N, P, expected block size): by default P is a hint, the tiled kernels run on blocks of the largest 8 * 2^k <= 256
    # rows that divides N unless the caller's blocks already have such a shape (m = 300, m = 768, N % P != 0
    # used to fall to the thread-per-block kernels)
    (3 << 15, 128, 256),       # m = 768
    (300000, 1000, 32),        # m = 300; 300000 = 2^5 * 9375
    (300000, 7, 32),           # N % P != 0
    (8 * 4097, 4097 * 2, 8),   # m = 4 -> blocks of 8 rows (N / 8 odd)
    (1 << 16, 1 << 10, 64),    # the caller's blocks of 64 rows are kept
    (1 << 16, 3, 256),
]


@pytest.mark.parametrize("N,P,m_eff", AUTO_PARTITION_CASES)
def test_auto_partition(N, P, m_eff):
    cfg = W.scaled(W.CONFIGS["C2dense"], N=N)
    V, psi = W.potential(cfg), W.psi0(cfg)
    dx, dt = 0.01, 0.005
    ref = O.step(dx, dt, V, psi, 3)
    out, info = gpu_step(N, P, dx, dt, V, psi, 3, onchip=0)
    assert info["path"] == B.PATH_TILED and info["P"] == P and info["P_effective"] == N // m_eff, info
    err = np.max(np.abs(out - ref))
    assert err <= TOL_PSI, (N, P, err)
    # the caller's partition taken literally (generic kernels unless the shape fits the tiled ones) gives the same psi
    out2, info2 = gpu_step(N, P, dx, dt, V, psi, 3, onchip=0, keep_p=1)
    assert info2["P_effective"] == P
    assert np.max(np.abs(out2 - ref)) <= TOL_PSI


ONCHIP_SHAPES = [2, 3, 8, 9, 64, 100, 255, 256, 257, 777, 1000, 2048, 4095, 4096]


@pytest.mark.parametrize("N", ONCHIP_SHAPES)
def test_onchip_path_random(N):
    # whole system in the registers of one CTA, all steps inside one launch (cn_onchip.cuh): every CTA size,
    # ragged last chunk, a single chunk; P is irrelevant to psi (reading R8)
    V, psi = W.random_system(N, seed=31)
    dx, dt = 0.1, 0.02
    for nsteps in (1, 2, 25):
        ref = O.step(dx, dt, V, psi, nsteps)
        out, info = gpu_step(N, 1, dx, dt, V, psi, nsteps)
        assert info["path"] == B.PATH_ONCHIP
        err = np.max(np.abs(out - ref))
        assert err <= TOL_PSI, (N, nsteps, err)
    out1, _ = gpu_step(N, 1, dx, dt, V, psi, 1)
    assert residual(dx, dt, V, psi, out1) <= TOL_RES
    # the same plan with the on-chip stepper switched off takes the per-step kernels and agrees
    out2, info2 = gpu_step(N, 1, dx, dt, V, psi, 3, onchip=0)
    out3, _ = gpu_step(N, 1, dx, dt, V, psi, 3)
    assert info2["path"] != B.PATH_ONCHIP
    assert np.max(np.abs(out2 - out3)) <= 1e-12


RS_CASES = [
    # (N, P, opts): nested RS levels, ragged last group, single-row groups, serial RS
    (1 << 13, 1 << 10, dict(rs_topmax=64)),            # 1024 -> 4 groups of 256
    (8 * 1000, 1000, dict(rs_topmax=64)),               # ragged last group (232 rows)
    (8 * 1025, 1025, dict(rs_topmax=64)),               # last group is a single joint row
    (8 * 513, 513, dict(rs_topmax=2)),                  # 513 -> 3 -> 1 : three levels
    (1 << 16, 1 << 13, dict(rs_levels=1)),              # single CTA, K = 8
    (1 << 15, 3000, dict(rs_levels=1)),                 # single CTA, K = 4, generic path (ragged blocks)
    (1 << 16, 1 << 13, dict(rs_levels=2)),
    (1 << 17, 1 << 14, dict()),                         # auto: 16384 > 4096 -> two levels
    (1 << 13, 1 << 10, dict(rs_levels=-1)),             # paper-literal serial RS
    (1 << 13, 1 << 10, dict(pdl=0)),
    (5000, 700, dict(rs_topmax=16)),                    # generic path + nested RS
    # last level by its own kernel instead of inside the substitution kernel
    (1 << 13, 1 << 10, dict(rs_topmax=64, rs_top_in_subst=0)),
    (8 * 1000, 1000, dict(rs_topmax=64, rs_top_in_subst=0)),
    (8 * 513, 513, dict(rs_topmax=2, rs_top_in_subst=0)),
    (1 << 17, 1 << 14, dict(rs_top_in_subst=0)),
    (8 * 98304, 98304, dict(rs_top_in_subst=0)),
    (8 * 98304, 98304, dict(rs_top_in_subst=1024)),      # last level of 384 rows inside the substitution (KT = 4)
    (1 << 21, 1 << 18, dict(rs_top_in_subst=1024)),      # 1024 rows (KT = 8)
    # paper-shaped nested levels: one thread per group of any size, serial last level
    (8 * 1000, 1000, dict(rs_group=10, rs_levels=3, rs_serial_top=1)),
    (1 << 13, 1 << 10, dict(rs_group=32, rs_levels=2)),
    (5000, 700, dict(rs_group=7, rs_levels=3, rs_serial_top=1)),
    (300000, 4489, dict(rs_group=67, rs_levels=2, rs_serial_top=1)),
    (300000, 12167, dict(rs_group=23, rs_levels=3, rs_serial_top=1)),
]


@pytest.mark.parametrize("N,P,opts", RS_CASES)
def test_rs_levels(N, P, opts):
    cfg = W.scaled(W.CONFIGS["C2dense"], N=N)
    V, psi = W.potential(cfg), W.psi0(cfg)
    # strongly implicit step (s = dt / 4 dx^2 = 12.5) so that the reduced system is NOT nearly diagonal
    dx, dt = 0.01, 0.005
    ref = O.step(dx, dt, V, psi, 3)
    out, info = gpu_step(N, P, dx, dt, V, psi, 3, **opts)
    err = np.max(np.abs(out - ref))
    assert err <= TOL_PSI, (N, P, opts, info, err)
    if "rs_levels" in opts and opts["rs_levels"] > 0:
        assert info["rs_levels"] == opts["rs_levels"]
    out1, _ = gpu_step(N, P, dx, dt, V, psi, 1, **opts)
    assert residual(dx, dt, V, psi, out1) <= TOL_RES


@pytest.mark.parametrize("N,P,opts", [(1 << 21, 1 << 18, dict()), (1 << 21, 1 << 18, dict(pdl=0)),
                                       (8 * 98304, 98304, dict())])
def test_refill_race_stress(N, P, opts):
    """Repeated fresh plans on L2-resident systems with m = 8: the shapes on which the TMA refill of the input tile
    overtook shared-memory loads still queued behind the CTA barrier (about 1 call in 10 before the
    fence.proxy.async in k_pass_tiled, hazards)."""
    cfg = W.scaled(W.CONFIGS["C2dense"], N=N)
    V, psi = W.potential(cfg), W.psi0(cfg)
    dx, dt = 0.01, 0.005
    ref = O.step(dx, dt, V, psi, 3)
    worst = 0.0
    for _ in range(40):
        out, _ = gpu_step(N, P, dx, dt, V, psi, 3, **opts)
        worst = max(worst, float(np.max(np.abs(out - ref))))
    assert worst <= TOL_PSI, worst


def test_config_c1_both_paths():
    cfg = W.CONFIGS["C1"]
    V, psi = W.potential(cfg), W.psi0(cfg)
    ref = O.step(cfg.dx, cfg.dt, V, psi, cfg.steps)
    for path in (B.PATH_GENERIC, B.PATH_TILED, B.PATH_AUTO):
        out, info = gpu_step(cfg.N, cfg.P, cfg.dx, cfg.dt, V, psi, cfg.steps, path=path)
        assert np.max(np.abs(out - ref)) <= TOL_PSI
        assert abs(np.vdot(out, out).real * cfg.dx - 1.0) <= 1e-12
    # the same 100 steps as 10 calls of 10 (prologue / epilogue per call)
    out, _ = gpu_step(cfg.N, cfg.P, cfg.dx, cfg.dt, V, psi, 10, calls=10)
    assert np.max(np.abs(out - ref)) <= TOL_PSI


def test_p_invariance_and_linearity():
    cfg = W.scaled(W.CONFIGS["C2dense"], N=1 << 15)
    V, psi = W.potential(cfg), W.psi0(cfg)
    outs = [gpu_step(cfg.N, P, cfg.dx, cfg.dt, V, psi, 5)[0] for P in (1 << 3, 1 << 6, 1 << 9, 1 << 12)]
    for o in outs[1:]:
        assert np.max(np.abs(o - outs[0])) <= 1e-13
    a, _ = gpu_step(cfg.N, 1 << 7, cfg.dx, cfg.dt, V, (2 - 3j) * psi, 5)
    assert np.max(np.abs(a - (2 - 3j) * outs[0])) <= 1e-12


def test_time_reversal_gpu():
    cfg = W.scaled(W.CONFIGS["C1"], N=1 << 14, P=1 << 6)
    V, psi = W.potential(cfg), W.psi0(cfg)
    fwd, _ = gpu_step(cfg.N, cfg.P, cfg.dx, cfg.dt, V, psi, 20)
    back, _ = gpu_step(cfg.N, cfg.P, cfg.dx, -cfg.dt, V, fwd, 20)
    assert np.max(np.abs(back - psi)) <= 1e-11


def test_cayley_phase_gpu():
    # closed form straight against the CUDA path (V = 0, sine mode)
    n, k, dx, dt, steps = 4096, 7, 0.1, 0.01, 200
    j = np.arange(1, n + 1)
    v = np.sin(math.pi * k * j / (n + 1)).astype(complex)
    lam = (1.0 - math.cos(math.pi * k / (n + 1))) / dx ** 2
    ph = ((1 - 0.5j * lam * dt) / (1 + 0.5j * lam * dt)) ** steps
    out, _ = gpu_step(n, 32, dx, dt, np.zeros(n), v, steps)
    assert np.max(np.abs(out - ph * v)) <= 1e-11


def test_errors_on_device():
    torch = torch_()
    V = np.zeros(64)
    plan = B.Plan(64, 8, 0.1, 0.01, V)
    psi = torch.zeros(64, dtype=torch.complex128, device="cuda")
    with pytest.raises(B.CnError) as ei:
        plan.step(psi, 1)
    assert ei.value.status == B.CN_ENOTFACTORIZED
    plan.factorize()
    plan.step(psi, 0)
    with pytest.raises(B.CnError) as ei:
        B.cn_step(plan.h, psi.data_ptr() + 8, 1)
    assert ei.value.status == B.CN_EINVAL
    # every option value the header documents is accepted, everything else is CN_EINVAL (include/cn_nshape.h)
    good = {B.CN_OPT_PATH: (0, 1, 2), B.CN_OPT_TILE_THREADS: (0, 32, 64, 128, 256, 512), B.CN_OPT_RS_TOPMAX: (1, 4096, 8192),
            B.CN_OPT_RS_LEVELS: (-1, 0, 1, 8), B.CN_OPT_PROFILE: (0, 1), B.CN_OPT_PDL: (0, 1), B.CN_OPT_ONCHIP: (0, 1),
            B.CN_OPT_RS_GROUP: (2, 256, 1 << 20), B.CN_OPT_RS_SERIAL_TOP: (0, 1), B.CN_OPT_RS_TOP_IN_SUBST: (0, 1, 1024),
            B.CN_OPT_KEEP_P: (0, 1), B.CN_OPT_BY_COLS: (0, 4, 8)}
    bad = {B.CN_OPT_PATH: (-1, 3), B.CN_OPT_TILE_THREADS: (16, 96, 1024), B.CN_OPT_RS_TOPMAX: (0, 8193),
           B.CN_OPT_RS_LEVELS: (-2, 9), B.CN_OPT_RS_GROUP: (1, (1 << 20) + 1), B.CN_OPT_BY_COLS: (1, 2, 16), 4: (0, 1), 9: (0, 1), 0: (0,), 15: (0,)}
    for key, vals in good.items():
        for v in vals:
            plan.set_option(key, v)
    for key, vals in bad.items():
        for v in vals:
            with pytest.raises(B.CnError) as ei:
                plan.set_option(key, v)
            assert ei.value.status == B.CN_EINVAL, (key, v)
    plan.close()
    # V given as a device tensor
    dV = torch.zeros(64, dtype=torch.float64, device="cuda")
    with B.Plan(64, 8, 0.1, 0.01, dV) as p2:
        p2.factorize()
        p2.step(psi, 2)
    # breakdown: mu = -gamma + i rho hits a non-finite pivot when V is not finite
    Vbad = np.zeros(64)
    Vbad[10] = np.inf
    with B.Plan(64, 8, 0.1, 0.01, Vbad) as p3:
        with pytest.raises(B.CnError) as ei:
            p3.factorize()
        assert ei.value.status == B.CN_EBREAKDOWN


@pytest.mark.parametrize("name", ["C2dense", "C2"])
def test_config_c2_full_size(name):
    """BASELINE configs[1] at full N = 2^24 in the launch configuration bench.py times (default P, tiled path,
    nested RS, PDL): every element against the oracle after 20 of the 1000 steps (the oracle needs ~0.3 s per
    step at this size), plus the size-independent properties: norm and the residual of one solve."""
    cfg = W.CONFIGS[name]
    V, psi = W.potential(cfg), W.psi0(cfg)
    nsteps = 20
    ref = O.step(cfg.dx, cfg.dt, V, psi, nsteps)
    out, info = gpu_step(cfg.N, cfg.P, cfg.dx, cfg.dt, V, psi, nsteps)
    assert info["path"] == B.PATH_TILED and info["rs_levels"] >= 2
    err = np.max(np.abs(out - ref))
    assert err <= TOL_PSI, err
    assert abs(np.vdot(out, out).real * cfg.dx - 1.0) <= 1e-12
    out1, _ = gpu_step(cfg.N, cfg.P, cfg.dx, cfg.dt, V, psi, 1)
    assert residual(cfg.dx, cfg.dt, V, psi, out1) <= TOL_RES


def test_config_c2_full_step_count():
    """C2 at full size for the config's FULL step count (1000 steps, 10 calls of 100 as bench.py issues them) by
    properties that hold at any size -- the norm (CN is unitary: 1e-12 per 1000 steps is the oracle's own pin), time
    reversal with a plan of -dt, and the oracle on the last 5 steps restarted from the GPU state after 995.  The
    element-by-element comparison with 1000 ORACLE steps is tests/test_gpu_zz_fullsteps.py::test_config_c2_all_steps."""
    torch = torch_()
    cfg = W.CONFIGS["C2dense"]
    V, psi = W.potential(cfg), W.psi0(cfg)
    d = torch.from_numpy(psi).cuda()
    with B.Plan(cfg.N, cfg.P, cfg.dx, cfg.dt, V) as plan:
        plan.factorize()
        for _ in range(9):
            plan.step(d, 100)
        plan.step(d, 95)
        torch.cuda.synchronize()
        mid = d.cpu().numpy()
        plan.step(d, 5)
        torch.cuda.synchronize()
        out = d.cpu().numpy()
    assert abs(np.vdot(out, out).real * cfg.dx - 1.0) <= 1e-12
    assert np.max(np.abs(out - O.step(cfg.dx, cfg.dt, V, mid, 5))) <= TOL_PSI
    with B.Plan(cfg.N, cfg.P, cfg.dx, -cfg.dt, V) as back:
        back.factorize()
        for _ in range(10):
            back.step(d, 100)
        torch.cuda.synchronize()
    assert np.max(np.abs(d.cpu().numpy() - psi)) <= 1e-9   # 2000 steps of rounding, forward and back
