"""ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes front end of `oracle/cn_thomas.c`: the plain serial Thomas-algorithm
Crank-Nicolson stepper in complex128 (Eq. 2-5).  Only tests/,
`__graft_entry__.smoke()` and bench.py's `cpu_baseline` / `--impl reference` legs
may import this module.  It imports nothing from the CUDA package
`paper_2205_00856_b200` and the package imports nothing from here.

Every function is pinned in tests/test_oracle_pins.py (dense LU, closed-form
Cayley phase, norm, residual, time reversal); nothing here is "parity unpinned".
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cn_thomas.c")
_SO = os.path.join(_HERE, "libcn_oracle.so")
# no -ffast-math, no FTZ/DAZ; see the header of cn_thomas.c for -fcx-limited-range
CFLAGS = ["-O2", "-std=c11", "-fPIC", "-shared", "-ffp-contract=off", "-fcx-limited-range", "-Wall"]

_SO_OMP = os.path.join(_HERE, "libcn_oracle_omp.so")  # the same source + -fopenmp: adds cn_oracle_step_2d_omp (timing aid)

_lib = None
_lib_omp = None
_lock = threading.Lock()


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", *CFLAGS, "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _SO)
    if force or not os.path.exists(_SO_OMP) or os.path.getmtime(_SO_OMP) < os.path.getmtime(_SRC):
        tmp = _SO_OMP + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", *CFLAGS, "-fopenmp", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _SO_OMP)
    return _SO


def _load_omp():
    global _lib_omp
    with _lock:
        if _lib_omp is None:
            build()
            lib = ctypes.CDLL(_SO_OMP)
            i64, dbl, ptr = ctypes.c_int64, ctypes.c_double, ctypes.c_void_p
            lib.cn_oracle_step_2d_omp.restype = i64
            lib.cn_oracle_step_2d_omp.argtypes = [i64, i64, dbl, dbl, ptr, ptr, ptr, i64, ctypes.POINTER(dbl),
                                                  ctypes.POINTER(i64)]
            _lib_omp = lib
    return _lib_omp


def _load():
    global _lib
    with _lock:
        if _lib is None:
            lib = ctypes.CDLL(build())
            i64, dbl, ptr = ctypes.c_int64, ctypes.c_double, ctypes.c_void_p
            lib.cn_oracle_thomas.restype = i64
            lib.cn_oracle_thomas.argtypes = [i64, ptr, ptr, ptr, ptr, ptr]
            lib.cn_oracle_diagonals.restype = None
            lib.cn_oracle_diagonals.argtypes = [i64, dbl, dbl, ptr, ptr, ptr, ptr]
            lib.cn_oracle_rhs.restype = None
            lib.cn_oracle_rhs.argtypes = [i64, ptr, ptr, ptr, ptr, ptr]
            lib.cn_oracle_step.restype = i64
            lib.cn_oracle_step.argtypes = [i64, dbl, dbl, ptr, ptr, i64, i64, ctypes.POINTER(dbl)]
            lib.cn_oracle_step_lean.restype = i64
            lib.cn_oracle_step_lean.argtypes = [i64, dbl, dbl, ptr, ptr, i64, ctypes.POINTER(dbl)]
            lib.cn_oracle_step_2d.restype = i64
            lib.cn_oracle_step_2d.argtypes = [i64, i64, dbl, dbl, ptr, ptr, ptr, i64, ctypes.POINTER(dbl)]
            _lib = lib
    return _lib


def _z(x):
    x = np.ascontiguousarray(x, dtype=np.complex128)
    return x


def _p(x):
    return x.ctypes.data_as(ctypes.c_void_p)


def diagonals(dx: float, dt: float, V):
    """(b, a, c) of T = 1 + i dt/2 H for the 3-point H (reading R3)."""
    V = np.ascontiguousarray(V, dtype=np.float64)
    n = V.size
    b, a, c = (np.empty(n, np.complex128) for _ in range(3))
    _load().cn_oracle_diagonals(n, dx, dt, _p(V), _p(b), _p(a), _p(c))
    return b, a, c


def rhs(b, a, c, psi):
    """d = T^dagger psi (Eq. 3)."""
    b, a, c, psi = _z(b), _z(a), _z(c), _z(psi)
    d = np.empty_like(psi)
    _load().cn_oracle_rhs(psi.size, _p(b), _p(a), _p(c), _p(psi), _p(d))
    return d


def thomas(b, a, c, d):
    """Solve the general complex tridiagonal system of Eq. 5 serially."""
    b, a, c = _z(b), _z(a), _z(c)
    x = _z(d).copy()
    scratch = np.empty_like(x)
    rc = _load().cn_oracle_thomas(x.size, _p(b), _p(a), _p(c), _p(x), _p(scratch))
    if rc:
        raise ZeroDivisionError("zero or non-finite pivot at row %d" % (rc - 1))
    return x


def step(dx: float, dt: float, V, psi, nsteps: int = 1, lean: bool = False, return_seconds: bool = False):
    """nsteps CN steps of one 1-D system; returns the new psi (input untouched)."""
    V = np.ascontiguousarray(V, dtype=np.float64)
    out = _z(psi).copy()
    assert out.ndim == 1 and out.size == V.size
    sec = ctypes.c_double(0.0)
    if lean:
        rc = _load().cn_oracle_step_lean(out.size, dx, dt, _p(V), _p(out), nsteps, ctypes.byref(sec))
    else:
        rc = _load().cn_oracle_step(out.size, dx, dt, _p(V), _p(out), 1, nsteps, ctypes.byref(sec))
    if rc:
        raise RuntimeError("oracle failed rc=%d" % rc)
    return (out, sec.value) if return_seconds else out


def step_inplace(dx: float, dt: float, V, psi, nsteps: int = 1, lean: bool = False) -> float:
    """As `step` but overwrites psi (contiguous complex128); returns seconds of the step loop."""
    assert psi.dtype == np.complex128 and psi.flags.c_contiguous
    V = np.ascontiguousarray(V, dtype=np.float64)
    sec = ctypes.c_double(0.0)
    if lean:
        rc = _load().cn_oracle_step_lean(psi.size, dx, dt, _p(V), _p(psi), nsteps, ctypes.byref(sec))
    else:
        rc = _load().cn_oracle_step(psi.size, dx, dt, _p(V), _p(psi), 1, nsteps, ctypes.byref(sec))
    if rc:
        raise RuntimeError("oracle failed rc=%d" % rc)
    return sec.value


def step_td(dx: float, dt: float, V0, g, field, psi):
    """Time-dependent H(t) = H0 + f(t) g(x) (the propagator of step k uses H at t_k + dt/2):
    len(field) plain CN steps, step k with the potential V0 + field[k] * g -- the definition written out, one
    full Thomas solve (with its own diagonals) per step.  Pinned in tests/test_oracle_pins.py by the closed-form
    Cayley phases for a uniform shift g = 1, per-step dense LU, norm conservation and field = 0."""
    V0 = np.ascontiguousarray(V0, dtype=np.float64)
    g = np.ascontiguousarray(g, dtype=np.float64)
    out = np.array(psi, dtype=np.complex128, copy=True)
    for f in np.asarray(field, dtype=np.float64):
        out = step(dx, dt, V0 + float(f) * g, out, 1)
    return out


def step_2d(dx: float, dt: float, Vx, Vy, psi, nsteps: int = 1, return_seconds: bool = False):
    """C4: psi[y][x] <- (CN_y(dt) CN_x(dt))^nsteps psi (reading R18)."""
    Vx = np.ascontiguousarray(Vx, dtype=np.float64)
    Vy = np.ascontiguousarray(Vy, dtype=np.float64)
    out = _z(psi).copy()
    ny, nx = out.shape
    assert Vx.size == nx and Vy.size == ny
    sec = ctypes.c_double(0.0)
    rc = _load().cn_oracle_step_2d(nx, ny, dx, dt, _p(Vx), _p(Vy), _p(out), nsteps, ctypes.byref(sec))
    if rc:
        raise RuntimeError("oracle failed rc=%d" % rc)
    return (out, sec.value) if return_seconds else out


def step_2d_omp(dx: float, dt: float, Vx, Vy, psi, nsteps: int = 1):
    """`step_2d` with the independent systems of every sweep shared out over all host cores by OpenMP (the multi-core
    C4 CPU baseline of BASELINE.md section 3).  Each thread runs the unchanged serial per-system step, so the result
    is bit-identical to `step_2d` (pinned in tests/test_oracle_pins.py).  Returns (psi, seconds, threads used)."""
    Vx = np.ascontiguousarray(Vx, dtype=np.float64)
    Vy = np.ascontiguousarray(Vy, dtype=np.float64)
    out = _z(psi).copy()
    ny, nx = out.shape
    assert Vx.size == nx and Vy.size == ny
    sec, nth = ctypes.c_double(0.0), ctypes.c_int64(0)
    rc = _load_omp().cn_oracle_step_2d_omp(nx, ny, dx, dt, _p(Vx), _p(Vy), _p(out), nsteps, ctypes.byref(sec),
                                           ctypes.byref(nth))
    if rc:
        raise RuntimeError("oracle failed rc=%d" % rc)
    return out, sec.value, int(nth.value)


def dense_T(dx: float, dt: float, V) -> np.ndarray:
    """Assemble T densely (tests only, small N)."""
    b, a, c = diagonals(dx, dt, V)
    n = a.size
    T = np.zeros((n, n), np.complex128)
    T[np.arange(n), np.arange(n)] = a
    T[np.arange(1, n), np.arange(n - 1)] = b[1:]
    T[np.arange(n - 1), np.arange(1, n)] = c[:-1]
    return T
