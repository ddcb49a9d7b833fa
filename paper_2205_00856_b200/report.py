"""Per-config throughput report (BASELINE.json: "report throughput on each config at 1 GPU in Gpoint-steps/s and as
achieved fraction of the HBM roofline, along with the sweep over partition count P").

    python -m paper_2205_00856_b200.report [--configs C1,C2,C3,C4,C5] [--sweep] [--out FILE]

One JSON line per config on stdout (and appended to --out).  Everything runs through the C-ABI binding; nothing here
touches oracle/ (parity of the same configs is in tests/).  Timing: CUDA events on the launching stream after a
warm-up call.  `bytes_per_point` is the algorithmic figure of DESIGN.md section 5 (56 B per point-step, 32 B per
point-sweep for C4, host link 24 B in + 16 B out for C5); `hbm_frac` divides by MEASURED_PEAKS.json's copy rate.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import time

import numpy as np

from . import binding as B
from . import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"])
    except Exception:
        return 6650.0  # B200_PROFILING.md fallback


def _events(torch):
    return torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)


def _inputs(cfg, chunk=1 << 24):
    V = np.empty(cfg.N, np.float64)
    psi = np.empty(cfg.N, np.complex128)
    norm = W.psi0_norm2(cfg)
    for s in range(0, cfg.N, chunk):
        e = min(cfg.N, s + chunk)
        V[s:e] = W.potential(cfg, s, e)
        psi[s:e] = W.psi0(cfg, s, e, norm=norm)
    return V, psi


def time_plan(torch, plan, d_psi, nsteps, reps=3):
    """best and median ms per CN step over `reps` cn_step(nsteps) calls"""
    plan.step(d_psi, min(nsteps, 5))
    torch.cuda.synchronize()
    ms = []
    for _ in range(reps):
        e0, e1 = _events(torch)
        e0.record()
        plan.step(d_psi, nsteps)
        e1.record()
        torch.cuda.synchronize()
        ms.append(e0.elapsed_time(e1) / nsteps)
    ms.sort()
    return ms[0], ms[len(ms) // 2]


def run_1d(torch, name, peak, nsteps=None, P=None, **opts):
    cfg = W.CONFIGS[name]
    V, psi = _inputs(cfg)
    d = torch.from_numpy(psi).cuda()
    del psi
    with B.Plan(cfg.N, P or cfg.P, cfg.dx, cfg.dt, V, **opts) as plan:
        t0 = time.time()
        plan.factorize()
        torch.cuda.synchronize()
        fms = 1e3 * (time.time() - t0)
        n = nsteps or cfg.steps
        best, med = time_plan(torch, plan, d, n)
        info = plan.info()
    gbs = 56.0 * cfg.N / (best * 1e-3) / 1e9
    moved = info["bytes_per_point_step"]  # 48 on the tiled path (gamma recovered from the pivots), else 56
    return {"config": name, "bytes_moved_per_point": moved, "hbm_frac_on_bytes_moved": gbs * moved / 56.0 / peak, "N": cfg.N, "P": P or cfg.P, "P_effective": info["P_effective"], "path": info["path"],
            "rs_levels": info["rs_levels"], "cn_steps_per_call": n, "us_per_cn_step_best": 1e3 * best,
            "us_per_cn_step_median": 1e3 * med, "Gpoint_steps_per_s": cfg.N / best / 1e6, "bytes_per_point": 56,
            "whole_step_GBps": gbs, "hbm_frac_measured_peak": gbs / peak, "hbm_frac_8TBps": gbs / 8000.0,
            "factorize_ms": fms, "device_bytes": info["device_bytes"]}


def run_c4(torch, peak):
    """x-sweep then y-sweep per 2-D step (reading R18); 32 B per point per sweep."""
    cfg = W.CONFIGS["C4"]
    n = cfg.N
    d = torch.from_numpy(W.psi0_2d(cfg)).cuda()
    out = {"config": "C4", "N": n, "nsys": cfg.nsys, "bytes_per_point": 32}
    with B.Plan(n, cfg.P, cfg.dx, cfg.dt, W.potential(cfg)) as px, \
            B.Plan(n, cfg.P, cfg.dx, cfg.dt, W.potential_y(cfg)) as py:
        px.factorize()
        py.factorize()
        sweeps = {"x": lambda: px.batched_sweep(d, n, 1, n, 1), "y": lambda: py.batched_sweep(d, n, n, 1, 1)}
        sweeps["xy"] = lambda: (sweeps["x"](), sweeps["y"]())
        for key, fn in sweeps.items():
            for _ in range(3):
                fn()
            torch.cuda.synchronize()
            e0, e1 = _events(torch)
            e0.record()
            for _ in range(cfg.steps):
                fn()
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / cfg.steps
            nsw = 2 if key == "xy" else 1
            gbs = 32.0 * n * n * nsw / (ms * 1e-3) / 1e9
            out[key] = {"ms": ms, "Gpoint_sweeps_per_s": nsw * n * n / ms / 1e6, "GBps": gbs,
                        "hbm_frac_measured_peak": gbs / peak, "hbm_frac_8TBps": gbs / 8000.0}
    out["Gpoint_steps_per_s"] = n * n / out["xy"]["ms"] / 1e6  # one 2-D step = both sweeps
    return out


def run_c4_sizes(torch, peak, total=8192 * 8192):
    """The shared-matrix sweeps at C4's total size (2^26 points) cut into systems of 512 ... 8192 rows: where the
    kernels lose their bandwidth (cross-warp scan from 512 rows, one CTA per system at 2048, clusters of 2 / 4 CTAs at
    4096 / 8192 rows for x; clusters from 2048 rows for y)."""
    cfg = W.CONFIGS["C4"]
    d = torch.randn(total, dtype=torch.complex128, device="cuda")
    rows = []
    for n in (512, 1024, 2048, 4096, 8192):
        nsys = total // n
        c = W.scaled(cfg, N=n)
        with B.Plan(n, 8, c.dx, c.dt, W.potential(c)) as p:
            p.factorize()
            for key, args in (("x", (nsys, 1, n)), ("y", (nsys, nsys, 1))):
                for _ in range(3):
                    p.batched_sweep(d, *args, 1)
                torch.cuda.synchronize()
                e0, e1 = _events(torch)
                e0.record()
                for _ in range(20):
                    p.batched_sweep(d, *args, 1)
                e1.record()
                torch.cuda.synchronize()
                ms = e0.elapsed_time(e1) / 20
                gbs = 32.0 * total / (ms * 1e-3) / 1e9
                rows.append({"rows_per_system": n, "systems": nsys, "sweep": key, "ms": ms, "GBps": gbs,
                             "hbm_frac_measured_peak": gbs / peak})
    return {"config": "C4 total size, systems of 512..8192 rows (shared matrix)", "rows": rows}


def link_rate(torch, nbytes=1 << 30):
    """pinned host <-> device copy rates of this box (GB/s): H2D alone, D2H alone, both at once."""
    h0 = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    h1 = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    d0 = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    d1 = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    s0, s1 = torch.cuda.Stream(), torch.cuda.Stream()
    res = {}
    for key in ("h2d", "d2h", "both"):
        best = 1e30
        for _ in range(3):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            if key in ("h2d", "both"):
                with torch.cuda.stream(s0):
                    d0.copy_(h0, non_blocking=True)
            if key in ("d2h", "both"):
                with torch.cuda.stream(s1):
                    h1.copy_(d1, non_blocking=True)
            torch.cuda.synchronize()
            best = min(best, time.perf_counter() - t0)
        res[key] = nbytes / best / 1e9
    return res


def run_c5(torch):
    """psi in pinned host memory, 2 GB device budget: bound by the host link (24 B in + 16 B out per point-step)."""
    cfg = W.CONFIGS["C5"]
    V, psi = _inputs(cfg)
    h = torch.from_numpy(psi).pin_memory()
    del psi
    link = link_rate(torch)
    with B.Plan(cfg.N, cfg.P, cfg.dx, cfg.dt, V, device_budget=2 << 30) as plan:
        plan.factorize()
        info = plan.info()
        plan.step(h, 1)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        plan.step(h, cfg.steps)
        torch.cuda.synchronize()
        sec = time.perf_counter() - t0
    # a call of n steps makes n + 1 passes in (prologue + n) and n passes out
    h2d = 24.0 * cfg.N * (cfg.steps + 1) / sec / 1e9
    d2h = 16.0 * cfg.N * cfg.steps / sec / 1e9
    return {"config": "C5", "N": cfg.N, "P": cfg.P, "cn_steps_per_call": cfg.steps, "s_per_cn_step": sec / cfg.steps,
            "Gpoint_steps_per_s": cfg.N * cfg.steps / sec / 1e9, "h2d_GBps": h2d, "d2h_GBps": d2h,
            "link_GBps": link, "h2d_frac_of_link": h2d / link["both"] if link["both"] else None,
            "device_bytes": info["device_bytes"], "part_points": info["tile_points"]}


def p_sweep(torch, peak, name="C2dense"):
    """t(P) for P = 2^8..2^16 on both kernel families against the paper's model t = alpha N/P + beta P
    (PAPER.md:217-237): least-squares fit of alpha, beta (and a floor t0 the model lacks), P* = sqrt(alpha/beta) sqrt(N)."""
    cfg = W.CONFIGS[name]
    V, psi = _inputs(cfg)
    d = torch.from_numpy(psi).cuda()
    rows = []
    arms = (("tiled_default", dict()),          # the library partitions the system itself (P is a hint): flat in P by construction
            ("tiled_keep_p", dict(keep_p=1)),   # the caller's blocks on the tiled kernels (blocks of at most 4096 rows fit a CTA tile)
            ("paper_shape", dict(path=B.PATH_GENERIC, rs_levels=-1)),
            ("generic_nested_rs", dict(path=B.PATH_GENERIC)))
    for arm, opts in arms:
        for Pk in cfg.P_sweep:
            if arm == "tiled_keep_p" and cfg.N // Pk > 4096:
                continue  # such blocks do not fit a tile: CN_OPT_KEEP_P would run them on the thread-per-block kernels (= generic_nested_rs)
            with B.Plan(cfg.N, Pk, cfg.dx, cfg.dt, V, **opts) as plan:
                plan.factorize()
                info = plan.info()
                best, med = time_plan(torch, plan, d, 20 if arm.startswith("tiled") else 3, reps=3)
            rows.append({"arm": arm, "P": Pk, "P_effective": info["P_effective"], "rs_levels": info["rs_levels"],
                         "path": info["path"], "us_per_cn_step": 1e3 * best})
    fits = {}
    for arm in ("paper_shape", "generic_nested_rs"):  # (the tiled arms are flat / not of the model's shape: not fitted)
        Ps = np.array([r["P"] for r in rows if r["arm"] == arm], float)
        ts = np.array([r["us_per_cn_step"] for r in rows if r["arm"] == arm], float)
        A = np.stack([cfg.N / Ps, Ps, np.ones_like(Ps)], 1)
        (alpha, beta, t0), *_ = np.linalg.lstsq(A, ts, rcond=None)
        fit = {"alpha_us_per_point": alpha, "beta_us_per_block": beta, "floor_us": t0,
               "P_measured_argmin": int(Ps[int(np.argmin(ts))])}
        if alpha > 0 and beta > 0:
            fit["delta"] = math.sqrt(alpha / beta)
            fit["P_star_model"] = fit["delta"] * math.sqrt(cfg.N)
        fits[arm] = fit
    return {"config": name + " P sweep", "N": cfg.N, "sqrtN": math.isqrt(cfg.N), "rows": rows, "fit": fits}


# HBM bytes per point of one driven step: factor kernel V 8 + g 8 in, q 16 out; prologue pass
# psi 16 + q 16 in; epilogue pass the same in + psi 16 out (gamma is recovered from q by the passes: 136 before that)
TD_BYTES_PER_POINT = 112


def run_td(torch, peak, name="C2dense", nsteps=20):
    """Driven steps (H(t) = H0 + f(t) x, cn_step_td): factorization inside the step loop, two passes per step."""
    cfg = W.CONFIGS[name]
    V, psi = _inputs(cfg)
    d = torch.from_numpy(psi).cuda()
    x = W.grid(cfg)
    t = (np.arange(nsteps) + 0.5) * cfg.dt
    field = 0.05 * np.sin(0.3 * t)
    with B.Plan(cfg.N, cfg.P, cfg.dx, cfg.dt, V) as plan:
        plan.factorize()
        plan.set_td_shape(x)
        plan.step_td(d, field[:2])
        torch.cuda.synchronize()
        ms = []
        for _ in range(3):
            e0, e1 = _events(torch)
            e0.record()
            plan.step_td(d, field)
            e1.record()
            torch.cuda.synchronize()
            ms.append(e0.elapsed_time(e1) / (nsteps + 1))  # + the restoring factorization at the end of a call
    best = min(ms)
    return {"config": name + " time-dependent H", "N": cfg.N, "P": cfg.P, "us_per_driven_step": 1e3 * best,
            "Gpoint_steps_per_s": cfg.N / best / 1e6}


def run_tridiag(torch, peak, N=1 << 24):
    """General complex tridiagonal front end (cn_tridiag_*): seeded random diagonally dominant system, solves per
    second; algorithmic bytes per row and solve: the reduction reads l, rp, u, d and the zero slot (80 B), the
    substitution reads them again and writes x (96 B) = 176 B."""
    W.random_system  # the generators of the workloads module hold no arithmetic of the method
    rng = np.random.default_rng(2205)
    z = lambda: rng.normal(size=N) + 1j * rng.normal(size=N)
    b, c, d = z(), z(), z()
    a = (np.abs(b) + np.abs(c)) * 2.5 * np.exp(1j * rng.uniform(0, 2 * np.pi, N))
    dd = torch.from_numpy(d).cuda()
    xx = torch.empty_like(dd)
    t0 = time.time()
    with B.Tridiag(b, a, c) as t:
        torch.cuda.synchronize()
        fms = 1e3 * (time.time() - t0)
        for _ in range(3):
            t.solve(dd, xx)
        torch.cuda.synchronize()
        e0, e1 = _events(torch)
        e0.record()
        for _ in range(20):
            t.solve(dd, xx)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / 20
    gbs = 176.0 * N / (ms * 1e-3) / 1e9
    return {"config": "general tridiagonal", "N": N, "us_per_solve": 1e3 * ms, "Grows_per_s": N / ms / 1e6,
            "bytes_per_row": 176, "GBps": gbs, "hbm_frac_measured_peak": gbs / peak, "create_ms": fms}


def run_systems(torch, peak, n=8192, nsys=8192, nsteps=20):
    """Many systems with a potential of their own each (cn_plan_set_systems, row f-3) at C4's shape: a non-separable
    V(x, y) gives every line its own matrix.  Contiguous systems (the x sweep) run on the fused tiled pass: 56 B per
    point and step; interleaved systems (the y sweep) on one thread per system (correctness path)."""
    cfg = W.CONFIGS["C4"]
    x = W.grid(cfg)
    rng = np.random.default_rng(cfg.seed)
    V2 = 0.5 * (x[None, :n] ** 2 + x[:nsys, None] ** 2) + 0.1 * np.cos(x[None, :n] * x[:nsys, None])
    psi = rng.standard_normal((nsys, n)) + 1j * rng.standard_normal((nsys, n))
    d = torch.from_numpy(psi.reshape(-1)).cuda()
    out = {"config": "C4 shape, per-system potentials", "n": n, "nsys": nsys}
    for key, lay in (("contiguous", (1, n)), ("interleaved", (nsys, 1))):
        Vl = np.ascontiguousarray(V2 if key == "contiguous" else V2.T).reshape(-1)
        with B.Plan(n * nsys, nsys, cfg.dx, cfg.dt, Vl) as plan:
            plan.set_systems(nsys, *lay).factorize()
            k = nsteps if key == "contiguous" else 2
            plan.batched_sweep_v(d, 2)
            torch.cuda.synchronize()
            e0, e1 = _events(torch)
            e0.record()
            plan.batched_sweep_v(d, k)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / k
            gbs = 56.0 * n * nsys / (ms * 1e-3) / 1e9
            info = plan.info()
            moved = info["bytes_per_point_step"] if key == "contiguous" else 56
            out[key] = {"ms_per_sweep": ms, "Gpoint_sweeps_per_s": n * nsys / ms / 1e6, "path": info["path"],
                        "bytes_per_point": 56, "GBps": gbs, "hbm_frac_measured_peak": gbs / peak,
                        "bytes_moved_per_point": moved, "hbm_frac_on_bytes_moved": gbs * moved / 56.0 / peak}
    return out


def run_shards(torch, peak, name="C2dense", S=8, nsteps=50, **opts):
    """Sharded mode (cn_shard_*, row f-4) on ONE device: the S shards of one system stepped in-process, their records
    "gathered" by concatenation (sharded.LocalShards).  The shards' kernels run one after the other on the one GPU,
    so this is NOT a scaling figure: it measures what the sharded protocol adds per step in kernel time and launches
    (S x (pack + last-level solve + one launch more on the RS chain), smaller tiles per launch) over the unsharded
    plan on the same rows.  The network leg of a real job (one all-gather of step_count values per shard) is absent."""
    from . import sharded as SH
    cfg = W.CONFIGS[name]
    V, psi = _inputs(cfg)
    n = cfg.N // S
    plans = [B.ShardPlan(n, max(1, n // 256), cfg.dx, cfg.dt, V[r * n:(r + 1) * n], r, S, **opts) for r in range(S)]
    grp = SH.LocalShards(plans, lambda c: torch.zeros(c, dtype=torch.complex128, device="cuda"), torch.cat)
    grp.factorize()
    parts = [torch.from_numpy(psi[r * n:(r + 1) * n].copy()).cuda() for r in range(S)]
    grp.step(parts, 3)
    torch.cuda.synchronize()
    ms = []
    for _ in range(3):
        e0, e1 = _events(torch)
        e0.record()
        grp.step(parts, nsteps)
        e1.record()
        torch.cuda.synchronize()
        ms.append(e0.elapsed_time(e1) / nsteps)
    counts = plans[0].counts()
    launches = sum(p.info()["launches"] for p in plans)
    for p in plans:
        p.close()
    best = min(ms)
    return {"config": name + " sharded in-process", "N": cfg.N, "shards": S, "N_local": n, "record_values_per_step": counts[1],
            "record_values_matrix": counts[0], "us_per_cn_step_all_shards_serialised": 1e3 * best,
            "us_per_cn_step_per_shard": 1e3 * best / S, "Gpoint_steps_per_s_one_device": cfg.N / best / 1e6,
            "launches_total": launches}


def levels_study(torch, N=300000):
    """Nested multi-iteration study (Eq. 8-9, Fig. 2) with the paper-shaped kernels:
    one thread per block, one thread per group at every nested level, serial last level.  n_it = number of
    partition levels; for a given thread count P0 of the first iteration the later fan-outs are equal
    (r = P0^(1/n_it), the optimal split of Eq. 8).  Predicted optimum "up to a fixed constant": P0* = N^(n_it/(n_it+1))."""
    cfg = W.scaled(W.CONFIGS["C2dense"], N=N)
    V, psi = _inputs(cfg)
    d = torch.from_numpy(psi).cuda()
    rows = []
    big = N > (1 << 20)  # at 2^24 the far ends of the curves cost seconds per step: start at 2^8, cap the serial RS
    for n_it in (1, 2, 3):
        for k in range(8 if big else 4, 23 if big else 18):
            P0 = 1 << k
            if P0 > N // 2 or (big and n_it == 1 and k > 17):
                break
            if n_it == 1:
                opts = dict(path=B.PATH_GENERIC, rs_levels=-1)
                r = None
            else:
                r = max(2, int(round(P0 ** (1.0 / n_it))))
                r += (r == 256)  # 256 would select the warp-per-group kernels, not the paper-shaped ones
                opts = dict(path=B.PATH_GENERIC, rs_levels=n_it, rs_group=r, rs_serial_top=1)
            with B.Plan(cfg.N, P0, cfg.dx, cfg.dt, V, **opts) as plan:
                plan.factorize()
                best, _ = time_plan(torch, plan, d, 4 if big else 10, reps=2 if big else 3)
            rows.append({"n_it": n_it, "P0": P0, "fanout": r, "us_per_cn_step": 1e3 * best})
    summary = {}
    for n_it in (1, 2, 3):
        sel = [x for x in rows if x["n_it"] == n_it]
        bestrow = min(sel, key=lambda x: x["us_per_cn_step"])
        summary[n_it] = {"P0_measured_argmin": bestrow["P0"], "us_at_argmin": bestrow["us_per_cn_step"],
                         "P0_predicted_eq8": N ** (n_it / (n_it + 1.0))}
    return {"config": "nested levels study", "N": N, "rows": rows, "summary": summary}


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="C1,C2,C3,C4,C5")
    ap.add_argument("--sweep", action="store_true")
    ap.add_argument("--levels", action="store_true", help="nested multi-iteration study (PAPER.md Fig. 2, Eq. 8-9)")
    ap.add_argument("--levels-n", default="300000", help="comma list of system sizes for --levels (paper: 3e5)")
    ap.add_argument("--out", default="")
    args = ap.parse_args(argv)
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("report: no CUDA device; this library has no CPU fallback")
    peak = _peak()
    lines = []

    def emit(obj):
        s = json.dumps(obj)
        print(s, flush=True)
        lines.append(s)
        if args.out:
            with open(args.out, "a") as f:
                f.write(s + "\n")
    for name in [c.strip() for c in args.configs.split(",") if c.strip()]:
        if name == "C1":
            emit(run_1d(torch, "C1", peak))
            emit(dict(run_1d(torch, "C1", peak, onchip=0), variant="three_kernels_per_step"))
        elif name == "C2":
            emit(run_1d(torch, "C2dense", peak, nsteps=100))
        elif name == "C3":
            emit(run_1d(torch, "C3", peak))
        elif name == "C4":
            emit(run_c4(torch, peak))
        elif name == "C5":
            emit(run_c5(torch))
        elif name == "TD":
            emit(run_td(torch, peak))
        elif name == "TRI":
            emit(run_tridiag(torch, peak))
        elif name == "C4SIZES":
            emit(run_c4_sizes(torch, peak))
        elif name == "SYSV":
            emit(run_systems(torch, peak))
        elif name == "SHARD":
            for S, opts in ((1, {}), (2, {}), (8, {}), (8, {"rs_topmax": 1})):
                emit(dict(run_shards(torch, peak, S=S, **opts), options=opts))
    if args.sweep:
        emit(p_sweep(torch, peak))
    if args.levels:
        for n in args.levels_n.split(","):
            emit(levels_study(torch, int(n)))
    return 0


if __name__ == "__main__":
    sys.exit(main())
