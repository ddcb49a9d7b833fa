"""Seeded synthetic inputs for the five BASELINE.json configs (C1..C5).

This module holds NONE of the method's arithmetic: it only builds grids, real
potentials V(x) and initial wave functions psi0.  It is the one module that both
the oracle-side tests and the CUDA-side tests/bench import, so that both sides
see bit-identical inputs (numpy PCG64, seeds written out below).  It imports
neither `oracle/` nor the CUDA binding.

Every constant that BASELINE.json leaves open is fixed here and listed in
DESIGN.md ("Input recipe"); they are the [proposed] readings of SURVEY.md §8(c)
rows 7 and 15-19.  The paper itself has no dataset: its workload is "TDSE on
large 1-D grids" (one size printed, n_tot = 3e5).

All generators are chunkable: `psi0(cfg, start, stop)` returns rows
[start, stop) and the concatenation over any chunking is bit-identical, because
the noise/phase stream is drawn per fixed-size segment of SEG points from
`default_rng([seed, segment_index])`.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace

import numpy as np

SEG = 1 << 20  # points per independently seeded noise segment


@dataclass(frozen=True)
class Config:
    name: str
    N: int                      # points per 1-D system
    dx: float
    dt: float
    potential: str              # "harmonic" | "soft_coulomb" | "random_gaussians" | "zero"
    state: str                  # "packet_noise" | "gaussian_random_phase" | "gaussian_phase_noise"
    P: int                      # default partition count
    steps: int
    seed: int
    x0: float = -5.0
    sigma: float = 1.0
    k0: float = 1.0
    noise: float = 1e-3
    nsys: int = 1               # C4: number of systems per sweep (2-D grid is nsys x N)
    P_sweep: tuple = field(default_factory=tuple)
    note: str = ""


CONFIGS = {
    # PAPER-free constants come from BASELINE.json configs[0..4]
    "C1": Config("C1", 4096, 0.1, 0.01, "harmonic", "packet_noise", 64, 100, seed=20220501),
    "C2": Config("C2", 1 << 24, 0.05, 0.005, "soft_coulomb", "gaussian_random_phase", 1 << 16, 1000,
                 seed=20220502, x0=0.0, P_sweep=tuple(1 << k for k in range(8, 17))),
    # dense-support twin of C2: same envelope + C1-style noise so that far blocks are exercised
    "C2dense": Config("C2dense", 1 << 24, 0.05, 0.005, "soft_coulomb", "gaussian_phase_noise", 1 << 16, 1000,
                      seed=20220502, x0=0.0, P_sweep=tuple(1 << k for k in range(8, 17))),
    "C3": Config("C3", 1 << 30, 0.01, 0.001, "random_gaussians", "packet_noise", 1 << 16, 50, seed=20220503),
    "C4": Config("C4", 8192, 0.05, 0.002, "harmonic", "packet_noise", 8, 20, seed=20220504, nsys=8192,
                 x0=-5.0, k0=1.0),
    "C5": Config("C5", 1 << 29, 0.01, 0.01, "harmonic", "packet_noise", 1 << 17, 10, seed=20220505),
}


def scaled(cfg: Config, N: int, P: int | None = None, steps: int | None = None, **kw) -> Config:
    """Same recipe at another size (parity tests run the oracle at sizes it finishes in seconds)."""
    return replace(cfg, N=N, P=cfg.P if P is None else P, steps=cfg.steps if steps is None else steps, **kw)


def grid(cfg: Config, start: int = 0, stop: int | None = None) -> np.ndarray:
    """x_j = (j - (N-1)/2) dx, j = start..stop-1."""
    stop = cfg.N if stop is None else stop
    j = np.arange(start, stop, dtype=np.float64)
    return (j - 0.5 * (cfg.N - 1)) * cfg.dx


def _gaussians_params(cfg: Config):
    rng = np.random.default_rng([cfg.seed, 0xC3])
    amp = rng.uniform(-1.0, 1.0, 32)
    width = rng.uniform(0.5, 5.0, 32)
    lo = -0.5 * (cfg.N - 1) * cfg.dx
    centre = rng.uniform(lo, -lo, 32)
    return amp, width, centre


def potential(cfg: Config, start: int = 0, stop: int | None = None) -> np.ndarray:
    """Real potential V(x_j) on rows [start, stop) as float64."""
    x = grid(cfg, start, stop)
    if cfg.potential == "harmonic":
        return 0.5 * x * x
    if cfg.potential == "soft_coulomb":
        return -1.0 / np.sqrt(x * x + 2.0)
    if cfg.potential == "zero":
        return np.zeros_like(x)
    if cfg.potential == "random_gaussians":
        amp, width, centre = _gaussians_params(cfg)
        V = np.zeros_like(x)
        for A, w, c in zip(amp, width, centre):
            # each Gaussian only within +-40 widths (exp(-800) == 0 in fp64 anyway)
            lo = np.searchsorted(x, c - 40.0 * w)
            hi = np.searchsorted(x, c + 40.0 * w)
            if hi > lo:
                z = (x[lo:hi] - c) / w
                V[lo:hi] += A * np.exp(-0.5 * z * z)
        return V
    raise ValueError(cfg.potential)


def _segments(start: int, stop: int):
    s = start
    while s < stop:
        k = s // SEG
        e = min(stop, (k + 1) * SEG)
        yield k, s - k * SEG, e - k * SEG, s, e
        s = e


def _noise(cfg: Config, start: int, stop: int, kind: str) -> np.ndarray:
    out = np.empty(stop - start, dtype=np.complex128 if kind == "normal" else np.float64)
    for k, lo, hi, s, e in _segments(start, stop):
        rng = np.random.default_rng([cfg.seed, 1 if kind == "normal" else 2, k])
        if kind == "normal":
            z = rng.standard_normal((SEG, 2))
            out[s - start:e - start] = z[lo:hi, 0] + 1j * z[lo:hi, 1]
        else:
            u = rng.uniform(0.0, 2.0 * math.pi, SEG)
            out[s - start:e - start] = u[lo:hi]
    return out


def psi0_unnormalised(cfg: Config, start: int = 0, stop: int | None = None) -> np.ndarray:
    stop = cfg.N if stop is None else stop
    x = grid(cfg, start, stop)
    env = (math.pi * cfg.sigma ** 2) ** -0.25 * np.exp(-((x - cfg.x0) ** 2) / (2.0 * cfg.sigma ** 2))
    if cfg.state == "packet_noise":
        psi = env * np.exp(1j * cfg.k0 * x) + cfg.noise * _noise(cfg, start, stop, "normal")
    elif cfg.state == "gaussian_random_phase":
        psi = env * np.exp(1j * _noise(cfg, start, stop, "phase"))
    elif cfg.state == "gaussian_phase_noise":
        psi = env * np.exp(1j * _noise(cfg, start, stop, "phase")) + cfg.noise * _noise(cfg, start, stop, "normal")
    else:
        raise ValueError(cfg.state)
    return psi.astype(np.complex128, copy=False)


def psi0(cfg: Config, start: int = 0, stop: int | None = None, norm: float | None = None) -> np.ndarray:
    """Initial state on rows [start, stop), normalised so that sum |psi|^2 dx = 1 over the FULL grid.

    For a chunked build pass `norm` = psi0_norm2(cfg) computed once."""
    if norm is None:
        norm = psi0_norm2(cfg)
    return psi0_unnormalised(cfg, start, stop) / math.sqrt(norm)


def psi0_norm2(cfg: Config, chunk: int = 1 << 22) -> float:
    """sum_j |psi_j|^2 dx of the unnormalised state, accumulated chunk by chunk."""
    tot = 0.0
    for s in range(0, cfg.N, chunk):
        p = psi0_unnormalised(cfg, s, min(cfg.N, s + chunk))
        tot += float(np.vdot(p, p).real)
    return tot * cfg.dx


def psi0_2d(cfg: Config) -> np.ndarray:
    """C4: row-major psi[y][x], product packet in x and y + dense complex noise, normalised (dx*dy)."""
    assert cfg.nsys > 1
    cx = replace(cfg, nsys=1, noise=0.0)
    gx = psi0_unnormalised(cx)                                   # along x (fast axis), length N
    cy = replace(cfg, N=cfg.nsys, nsys=1, noise=0.0, x0=0.0, k0=0.0)
    gy = psi0_unnormalised(cy)                                   # along y, length nsys
    psi = np.empty((cfg.nsys, cfg.N), dtype=np.complex128)
    rows = max(1, SEG // cfg.N)
    for r0 in range(0, cfg.nsys, rows):
        r1 = min(cfg.nsys, r0 + rows)
        rng = np.random.default_rng([cfg.seed, 4, r0 // rows])
        z = rng.standard_normal((r1 - r0, cfg.N, 2))
        psi[r0:r1] = gy[r0:r1, None] * gx[None, :] + cfg.noise * (z[..., 0] + 1j * z[..., 1])
    psi /= math.sqrt(float(np.vdot(psi, psi).real) * cfg.dx * cfg.dx)
    return psi


def potential_y(cfg: Config) -> np.ndarray:
    """C4 y-sweep potential 0.5 y^2 on the nsys-point y grid (dy = dx)."""
    cy = replace(cfg, N=cfg.nsys, nsys=1)
    return potential(cy)


def random_system(N: int, seed: int, scale: float = 1.0):
    """Unstructured seeded test input: real V ~ U[-scale, scale], psi ~ complex normal."""
    rng = np.random.default_rng([seed, N])
    V = rng.uniform(-scale, scale, N)
    z = rng.standard_normal((N, 2))
    return V, (z[:, 0] + 1j * z[:, 1]).astype(np.complex128)
