"""Writes tests/golden/c3_golden.npz: config C3 (N = 2^30, 50 steps) advanced by the ORACLE ONLY.

The lean Thomas oracle needs ~25 min for the 50 steps of C3 on one host core -- too long for a test run -- so this
script runs it once and stores what `tests/test_gpu_fullsteps.py::test_config_c3_all_steps` compares the CUDA path with:

  * psi after `cfg.steps` steps on NWIN windows of WLEN points each (both ends of the grid, the wave packet, windows
    that straddle a tile boundary (2048 points), an RS group boundary of level 1 (2^16 points) and of level 2
    (2^24 points), a streamed-part-like boundary (2^23) and a few unaligned offsets), compared element by element;
  * two full-vector float64 checksums: sum |psi|^2 and Re sum w_j psi_j for the seeded weights `checksum_weights`
    (any wrong element anywhere in the vector moves the second one).

It imports ONLY `oracle/` and the shared input generators (`workloads.py`, no arithmetic of the method); nothing in
the file it writes comes from the CUDA path.  Usage (from the repo root, ~45 GB of host memory, ~30 min):

    python tests/golden/make_c3_golden.py            # full C3
    python tests/golden/make_c3_golden.py --log2n 22 # a small self-test of the same code path (writes to /tmp)
"""
from __future__ import annotations

import argparse
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import cn_oracle as O  # noqa: E402
from paper_2205_00856_b200 import workloads as W  # noqa: E402

WLEN = 1 << 16
CHUNK = 1 << 24


def window_starts(N: int, dx: float, x0: float) -> list[int]:
    """Start indices of the stored windows (clipped to the grid, multiples of nothing in particular)."""
    packet = int(round(x0 / dx + 0.5 * (N - 1)))  # grid index of the packet centre
    raw = [
        0,                                  # first rows (Dirichlet end, first tile, first block)
        N - WLEN,                           # last rows
        packet - WLEN // 2,                 # the wave packet
        (1 << 24) - WLEN // 2,              # level-2 RS group boundary (256 * 256 * 256 rows), also tile/part boundaries
        3 * (1 << 28) - WLEN // 2 + 1024,   # a 2^28 boundary, offset by half a tile
        N // 3,                             # nothing special
        5 * (1 << 27) + 12345,              # unaligned
        (1 << 29) + 7 * (1 << 23) - WLEN // 2,  # a 2^23 boundary (largest streamed part / TMA box multiple)
        (1 << 16) * 4097 - WLEN // 2,       # level-1 RS group boundary (256 blocks of 256 rows)
    ]
    out = []
    for s in raw:
        s = max(0, min(N - WLEN, s))
        if s not in out:
            out.append(s)
    return out


WL = 1 << 15  # the checksum weights are the rank-1 array w_j = v[j // WL] * u[j % WL]


def checksum_weights(seed: int, N: int) -> tuple[np.ndarray, np.ndarray]:
    """Seeded complex weights (u, v) of the full-vector checksum; w_j = v[j // WL] u[j % WL] costs nothing to rebuild."""
    rng = np.random.default_rng([seed, 0xC5])
    nrow = (N + WL - 1) // WL
    zu, zv = rng.standard_normal((WL, 2)), rng.standard_normal((nrow, 2))
    return zu[:, 0] + 1j * zu[:, 1], zv[:, 0] + 1j * zv[:, 1]


def checksums(psi: np.ndarray, seed: int) -> tuple[float, float, float]:
    """(sum |psi|^2, Re sum_j w_j psi_j, sum_j |w_j| |psi_j|) accumulated chunk by chunk in float64; the third scales
    the tolerance of the second.  N must be a multiple of WL (or smaller than it)."""
    N = psi.size
    u, v = checksum_weights(seed, N)
    if N < WL:
        u = u[:N]
    rows = max(1, CHUNK // WL)
    n2 = dot = scale = 0.0
    M = psi.reshape(-1, u.size)
    for r in range(0, M.shape[0], rows):
        blk = M[r:r + rows]
        n2 += float(np.vdot(blk, blk).real)
        dot += float((v[r:r + rows] @ (blk @ u)).real)
        scale += float(np.abs(v[r:r + rows]) @ (np.abs(blk) @ np.abs(u)))
    return n2, dot, scale


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--log2n", type=int, default=0, help="self-test at N = 2^k instead of the full config")
    ap.add_argument("--out", default="")
    a = ap.parse_args()
    cfg = W.CONFIGS["C3"]
    if a.log2n:
        cfg = W.scaled(cfg, 1 << a.log2n)
    out = a.out or (os.path.join(HERE, "c3_golden.npz") if not a.log2n else "/tmp/c3_golden_2p%d.npz" % a.log2n)
    N = cfg.N
    t0 = time.time()
    V = np.empty(N, np.float64)
    psi = np.empty(N, np.complex128)
    norm = W.psi0_norm2(cfg)
    for s in range(0, N, CHUNK):
        e = min(N, s + CHUNK)
        V[s:e] = W.potential(cfg, s, e)
        psi[s:e] = W.psi0(cfg, s, e, norm=norm)
    t_gen = time.time() - t0
    print("inputs: %.0f s" % t_gen, flush=True)
    sec = O.step_inplace(cfg.dx, cfg.dt, V, psi, cfg.steps, lean=True)
    print("oracle: %d steps in %.0f s (%.2f ns per point-step)" % (cfg.steps, sec, 1e9 * sec / (N * cfg.steps)), flush=True)
    starts = window_starts(N, cfg.dx, cfg.x0) if N >= 16 * WLEN else [0, N - min(N, WLEN)]
    wl = min(WLEN, N)
    windows = np.stack([psi[s:s + wl] for s in starts])
    n2, dot, scale = checksums(psi, cfg.seed)
    np.savez(out, starts=np.asarray(starts, np.int64), windows=windows, norm2=np.float64(n2), wdot=np.float64(dot),
             wscale=np.float64(scale), N=np.int64(N), steps=np.int64(cfg.steps), dx=np.float64(cfg.dx),
             dt=np.float64(cfg.dt), seed=np.int64(cfg.seed), oracle_seconds=np.float64(sec))
    print("wrote %s: %d windows of %d points, sum|psi|^2 dx = %.15f, wdot = %.15e" % (out, len(starts), wl, n2 * cfg.dx, dot))


if __name__ == "__main__":
    main()
