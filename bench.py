#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200-native N-shaped partition Crank-Nicolson stepper.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

Metric (BASELINE.json): CN grid-point-steps per second in complex128 on config C2
(N = 2^24, dx = 0.05, dt = 0.005, soft-Coulomb V), plus the achieved fraction of the HBM roofline.

One bench "step" = one `cn_step(plan, psi, nsteps = CN_PER_STEP)` call through the C-ABI, i.e. one pass of
the whole hot path (RHS, RD, RU, JD/JU, RS, SS and psi write -- every row of SURVEY 8a) CN_PER_STEP times
over the resident wave function; K = 10 such steps are the 1000 CN steps of the config.
`value` has psi, V and the factors resident in HBM; `e2e` is the same call with every bench step's wave function
taken from PINNED HOST memory (H2D) and its result returned there (D2H) inside the timed region; the steps are
independent batches, so their copies overlap the neighbouring steps' compute (three streams, two device buffers).

N > 1 (torchrun, one rank per GPU): the path does not shard in this build ("replicas only");
every rank advances its own replica of the system, no data-path collective; value = sum over ranks.

--impl reference times the ORACLE (plain serial Thomas CN stepper, oracle/) on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2205_00856_b200 import replicas as R  # noqa: E402
from paper_2205_00856_b200 import workloads as W  # noqa: E402

CN_PER_STEP = 100            # CN steps per bench step (one cn_step call)
BYTES_PER_POINT_STEP = 56.0  # algorithmic bytes per point-step as SURVEY 8d declares them: psi in 16 + one stored complex factor
                             # 16 + real V / gamma 8 + psi out 16 -- the figure `roofline.achieved` is computed from
BYTES_MOVED_PER_POINT = 48.0  # what the fused pass of this build moves: it recovers gamma from the stored pivots (DESIGN.md
                              # section 5), so it reads psi 16 + q 16 and writes psi 16; reported beside the declared figure
METRIC = "cn_grid_point_steps_per_sec_complex128"
UNIT = "Gpoint-steps/s"
WORKLOAD = ("C2 (N=2^24 complex128, dx=0.05, dt=0.005, soft-Coulomb V, Gaussian x random phase + 1e-3 dense noise, "
            "1000 CN steps)")


def bench_config(cfg, P, world):
    """`config` of the JSON line: the workload only, identical for both arms (--impl ours / reference)."""
    return {"workload": WORKLOAD, "N": cfg.N, "P": P, "dx": cfg.dx, "dt": cfg.dt, "cn_steps": cfg.steps,
            "l2_policy": "inputs_larger_than_L2 (psi 268 MB + factors 403 MB per pass vs 126 MB L2)",
            "parallelism": "replicas x%d" % world}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            with open(path) as f:
                return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic_per_launch():
    """(dram bytes per fused-pass launch, where the figure comes from): the committed ncu --set full capture under
    profiles/ -- ncu cannot run inside a timed bench, so the line says which capture (file, commit) it quotes."""
    rel = os.path.join("profiles", "pass_kernel_traffic.txt")
    val, src = None, None
    try:
        with open(os.path.join(ROOT, rel)) as f:
            for line in f:
                if line.startswith("dram_bytes_per_launch_at_N_2^24="):
                    val = float(line.split("=")[1])
                elif line.startswith("source="):
                    src = line.split("=", 1)[1].strip()
    except Exception:
        pass
    if val is None:
        return None, None
    return val, "%s (%s)" % (rel, src or "ncu --set full capture, see the file")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int, interval_ms: int = 20):
        self.proc = None
        self.lines = []
        self.index = index
        self.interval_ms = interval_ms

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", str(self.interval_ms)],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._pump, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        time.sleep(0.05)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [ln for (ts, ln) in self.lines if t0 <= ts <= t1 + 0.05] or [ln for (_, ln) in self.lines]
        for ln in rows:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1]))
                smax.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(names, f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "reasons": sorted(reasons), "samples": len(sm)}


dist_env = R.dist_env

def per_config_report(torch, peak, full, with_cpu):
    """Every other BASELINE.json config (and the two "next" front ends at C2's shape) under the same clock as the headline:
    a few ms of GPU time each through the C-ABI (paper_2205_00856_b200/report.py holds the timing loops), each with
    the oracle timed on a bounded sample of the same workload on this box's host cores.  C3 (2^30 points, 85 GB of
    host memory, minutes of input generation) and C5 (2^29 points streamed from pinned host memory) only with --full.
    `frac` = algorithmic bytes / time / measured copy peak; the algorithmic bytes per unit are DESIGN.md's."""
    from paper_2205_00856_b200 import report as RP
    out = {}

    def cpu(value, unit, cores, sample):
        return {"value": value, "unit": unit, "cores": cores, "kind": "oracle", "host_cores_available": os.cpu_count(),
                "sample": sample}

    O = None
    if with_cpu:
        from oracle import cn_oracle as O  # noqa: N811  (cpu_baseline leg only)

    # ---- C1: N = 4096 lives on one SM; latency bound, no HBM roofline -------------------------------------------
    cfg = W.CONFIGS["C1"]
    r = RP.run_1d(torch, "C1", peak)
    r3 = RP.run_1d(torch, "C1", peak, onchip=0)
    c1 = {"workload": "C1 (N=4096, P=64, dx=0.1, dt=0.01, harmonic V, 100 CN steps)", "us_per_cn_step": r["us_per_cn_step_best"],
          "Gpoint_steps_per_s": r["Gpoint_steps_per_s"], "path": r["path"],
          "us_per_cn_step_three_launches": r3["us_per_cn_step_best"],
          "roofline": "none: psi (64 KB) stays in the registers of one CTA for the whole call; latency / FP64-issue bound"}
    if O:
        V, psi = W.potential(cfg), W.psi0(cfg)
        sec = sum(O.step(cfg.dx, cfg.dt, V, psi, cfg.steps, return_seconds=True)[1] for _ in range(20))
        c1["cpu_baseline"] = cpu(cfg.N * cfg.steps * 20 / sec / 1e9, UNIT, 1, "20 x the config's 100 steps, serial Thomas")
    out["C1"] = c1

    # ---- C4: many-systems sweeps, 32 B per point per sweep -----------------------------------------------------
    cfg = W.CONFIGS["C4"]
    r = RP.run_c4(torch, peak)
    c4 = {"workload": "C4 (8192 x 8192, dx=dy=0.05, dt=0.002, V=0.5(x^2+y^2), x-sweep then y-sweep, 20 steps)",
          "bytes_per_point_sweep": 32, "x": r["x"], "y": r["y"], "xy": r["xy"],
          "Gpoint_steps_per_s": r["Gpoint_steps_per_s"], "frac": r["xy"]["hbm_frac_measured_peak"]}
    if O:
        psi2 = W.psi0_2d(cfg)
        Vx, Vy = W.potential(cfg), W.potential_y(cfg)
        _, sec = O.step_2d(cfg.dx, cfg.dt, Vx, Vy, psi2, 1, return_seconds=True)
        c4["cpu_baseline"] = cpu(cfg.N * cfg.N / sec / 1e9, UNIT, 1, "1 of the 20 2-D steps at full size, serial loops over the systems")
        _, sec, nth = O.step_2d_omp(cfg.dx, cfg.dt, Vx, Vy, psi2, 2)
        c4["cpu_baseline_all_cores"] = cpu(2 * cfg.N * cfg.N / sec / 1e9, UNIT, nth,
                                           "2 of the 20 2-D steps at full size, OpenMP over the independent systems of a sweep")
        del psi2
    out["C4"] = c4

    # ---- time-dependent H at C2's shape (row f-2) ---------------------------------------------------------------
    cfg = W.CONFIGS["C2dense"]
    r = RP.run_td(torch, peak)
    td_bytes = RP.TD_BYTES_PER_POINT
    td = {"workload": "C2 shape, H(t) = H0 + f(t) x: factorization redone on the device in every step",
          "us_per_driven_step": r["us_per_driven_step"], "Gpoint_steps_per_s": r["Gpoint_steps_per_s"],
          "bytes_per_point": td_bytes, "frac": td_bytes * cfg.N / (r["us_per_driven_step"] * 1e-6) / 1e9 / peak}
    if O:
        V, psi = W.potential(cfg), W.psi0(cfg)
        t0 = time.time()
        O.step_td(cfg.dx, cfg.dt, V, W.grid(cfg), [0.01, -0.02], psi)
        td["cpu_baseline"] = cpu(2 * cfg.N / (time.time() - t0) / 1e9, UNIT, 1,
                                 "2 driven steps at full N=2^24 (each a full Thomas solve with its own pivots)")
    out["TD"] = td

    # ---- general complex tridiagonal front end (row f-3) ------------------------------------------------------------
    r = RP.run_tridiag(torch, peak)
    tri = {"workload": "random diagonally dominant complex tridiagonal system, N=2^24, one right-hand side per solve",
           "us_per_solve": r["us_per_solve"], "Grows_per_s": r["Grows_per_s"], "bytes_per_row": r["bytes_per_row"],
           "frac": r["hbm_frac_measured_peak"]}
    if O:
        n = 1 << 22
        rng = np.random.default_rng(2205)
        z = lambda: rng.normal(size=n) + 1j * rng.normal(size=n)  # noqa: E731
        b, c, d = z(), z(), z()
        a = (np.abs(b) + np.abs(c)) * 2.5 * np.exp(1j * rng.uniform(0, 2 * np.pi, n))
        t0 = time.time()
        O.thomas(b, a, c, d)
        tri["cpu_baseline"] = cpu(n / (time.time() - t0) / 1e9, "Grows/s", 1, "one Thomas solve of 2^22 rows of the same distribution")
    out["TRI"] = tri

    # ---- many systems with a potential of their own each at C4's shape (row f-3) ---------------------------------------
    r = RP.run_systems(torch, peak)
    out["C4V"] = {"workload": "C4 shape (8192 x 8192), non-separable V(x, y): every line of a sweep has its own matrix",
                  "bytes_per_point_sweep": 56, "contiguous": r["contiguous"], "interleaved": r["interleaved"],
                  "frac": r["contiguous"]["hbm_frac_measured_peak"],
                  "frac_on_bytes_moved": r["contiguous"]["hbm_frac_on_bytes_moved"]}

    if full:
        # ---- C3: 2^30 points resident (psi 17 GB + factors 26 GB) -----------------------------------------------------
        cfg = W.CONFIGS["C3"]
        r = RP.run_1d(torch, "C3", peak)
        c3 = {"workload": "C3 (N=2^30, dx=0.01, dt=0.001, 32 seeded Gaussians, 50 CN steps)",
              "us_per_cn_step": r["us_per_cn_step_best"], "Gpoint_steps_per_s": r["Gpoint_steps_per_s"],
              "bytes_per_point": 56, "frac": r["hbm_frac_measured_peak"],
              "frac_on_bytes_moved": r["hbm_frac_on_bytes_moved"], "P_effective": r["P_effective"],
              "rs_levels": r["rs_levels"]}
        if O:
            n = 1 << 26
            sub = W.scaled(cfg, N=n)
            V, psi = RP._inputs(sub)
            sec = O.step_inplace(sub.dx, sub.dt, V, psi, 4, lean=True)
            c3["cpu_baseline"] = cpu(4 * n / sec / 1e9, UNIT, 1, "4 lean-Thomas steps on 2^26 points with C3's parameters")
        out["C3"] = c3
        # ---- C5: out of core, bound by the host link --------------------------------------------------------------------
        r = RP.run_c5(torch)
        c5 = {"workload": "C5 (N=2^29 in pinned host memory, device budget 2 GB, harmonic V, 10 CN steps)",
              "s_per_cn_step": r["s_per_cn_step"], "Gpoint_steps_per_s": r["Gpoint_steps_per_s"], "h2d_GBps": r["h2d_GBps"],
              "d2h_GBps": r["d2h_GBps"], "link_GBps": r["link_GBps"], "frac_of_link": r["h2d_frac_of_link"],
              "bytes_per_point": "24 in + 16 out over the host link", "device_bytes": r["device_bytes"]}
        if O:
            cfg = W.CONFIGS["C5"]
            n = 1 << 26
            sub = W.scaled(cfg, N=n)
            V, psi = RP._inputs(sub)
            sec = O.step_inplace(sub.dx, sub.dt, V, psi, 4, lean=True)
            c5["cpu_baseline"] = cpu(4 * n / sec / 1e9, UNIT, 1, "4 lean-Thomas steps on 2^26 points with C5's parameters")
        out["C5"] = c5
    return out



def oracle_timed(cfg, V, psi, cn_steps: int):
    from oracle import cn_oracle as O
    work = psi.copy()
    sec = O.step_inplace(cfg.dx, cfg.dt, V, work, cn_steps)
    return sec, work


def run_reference(args):
    """The oracle as it stands, on the host cores, same metric/config (bounded sample per step)."""
    rank, world, _ = dist_env()
    if rank != 0:
        return
    cfg = W.CONFIGS["C2dense"]
    V, psi = W.potential(cfg), W.psi0(cfg)
    from oracle import cn_oracle as O
    cn_per = 2                                # bounded sample: 2 CN steps at full N per bench step (~1 s)
    work = psi.copy()
    for _ in range(args.warmup):
        O.step_inplace(cfg.dx, cfg.dt, V, work, 1)
    tot = 0.0
    for _ in range(args.steps):
        tot += O.step_inplace(cfg.dx, cfg.dt, V, work, cn_per)
    value = cfg.N * cn_per * args.steps / tot / 1e9
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": bench_config(cfg, cfg.P, max(1, world)),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle",
                         "host_cores_available": os.cpu_count(),
                         "sample": "%d CN steps at full N=2^24 per bench step (of the config's 1000), serial Thomas, "
                                   "1 thread" % cn_per},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_sharded(args, torch, dist, B, rank, world, local):
    """ONE C2 system over `world` GPUs (row f-4): rank r owns rows [r N / world, (r + 1) N / world) and never sees the
    rest; per step one all-gather of `step_count` complex values per rank (paper_2205_00856_b200/sharded.py).  Same
    timing contract as the replica mode (barrier + synchronize on both sides, CUDA events, max over ranks); value = the
    WHOLE system's point-steps per second, so the scaling is strong."""
    from paper_2205_00856_b200 import sharded as SH
    cfg = W.CONFIGS["C2dense"]
    n = cfg.N // world
    assert n * world == cfg.N and n % 256 == 0, "the shards must be equal and multiples of 256 rows"
    cn_per = args.cn_per_step
    V = W.potential(cfg, rank * n, (rank + 1) * n)
    norm = W.psi0_norm2(cfg)
    d_psi = torch.from_numpy(W.psi0(cfg, rank * n, (rank + 1) * n, norm=norm)).cuda()
    plan = B.ShardPlan(n, max(1, n // 256), cfg.dx, cfg.dt, V, rank, world)
    if world == 1:
        class _One:  # a single process: the gather is the record itself
            def get_world_size(self, group=None):
                return 1

            def all_gather_into_tensor(self, out, inp, group=None):
                out.copy_(inp)
        dist = _One()
    st = SH.DistributedStepper(plan, device=torch.device("cuda", local), dist=dist)
    st.factorize()
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()
    for _ in range(args.warmup):
        st.step(d_psi, cn_per)
    launches0 = plan.info()["launches"]
    sampler = ClockSampler(local, args.clock_interval_ms)
    sampler.start()
    time.sleep(0.1)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    w0 = time.time()
    e0.record(stream)
    for _ in range(args.steps):
        st.step(d_psi, cn_per)
    e1.record(stream)
    barrier()
    w1 = time.time()
    ms = R.max_over_ranks(e0.elapsed_time(e1), world, device="cuda")
    clocks = sampler.stop(w0, w1)
    mcount, scount = plan.counts()
    nrm = d_psi.real.square().sum() + d_psi.imag.square().sum()
    if world > 1:
        dist.all_reduce(nrm)
    if rank == 0:
        line = {
            "metric": METRIC, "value": cfg.N * cn_per * args.steps / (ms * 1e-3) / 1e9, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": dict(bench_config(cfg, cfg.P, world), parallelism="one system over %d shards (cn_shard_*)" % world),
            "launch": {"cn_steps_per_bench_step": cn_per, "rows_per_shard": n, "record_values_per_step": scount,
                       "record_values_matrix": mcount, "exchange": "all_gather_into_tensor per step, %d B per rank" % (16 * scount)},
            "clocks": clocks, "gpu_launches": int(plan.info()["launches"] - launches0),
            "norm_minus_1": float(nrm.item()) * cfg.dx - 1.0,
        }
        print(json.dumps(line), flush=True)
    plan.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--P", type=int, default=0, help="partition count (0 = config default)")
    ap.add_argument("--tile-threads", type=int, default=0)
    ap.add_argument("--cn-per-step", type=int, default=CN_PER_STEP)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--clock-interval-ms", type=int, default=20, help="nvidia-smi sampling period during the timed region")
    ap.add_argument("--sweep", action="store_true", help="also time the P sweep 2^8..2^16 (extra JSON key)")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config object (C1, C4, TD, TRI)")
    ap.add_argument("--full", action="store_true", help="per_config also runs C3 (2^30, 85 GB host) and C5 (2^29, streamed)")
    ap.add_argument("--sharded", action="store_true",
                    help="N > 1: ONE C2 system spread over the N GPUs (cn_shard_*, one all-gather of a small record per step "
                         "over NCCL) instead of N replicas; \"scaling\": \"strong\".  Not what the driver runs; unmeasured on "
                         "hardware in this build (DESIGN.md section 9)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2205_00856_b200 import binding as B

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; this library has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    if args.sharded:
        return run_sharded(args, torch, dist, B, rank, world, local)

    cfg = W.CONFIGS["C2dense"]
    P = args.P or cfg.P
    cn_per = args.cn_per_step
    V, psi_h = W.potential(cfg), W.psi0(cfg)
    psi_pin = torch.from_numpy(psi_h).pin_memory()
    d_psi = psi_pin.cuda()
    plan = B.Plan(cfg.N, P, cfg.dx, cfg.dt, V, tile_threads=args.tile_threads)
    t0 = time.time()
    plan.factorize()
    torch.cuda.synchronize()
    factor_ms = 1e3 * (time.time() - t0)
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def timed_region(fn, steps, begin=None, finish=None):
        """EXACTLY `steps` calls of fn between barrier+sync, CUDA events on the launching stream, max over ranks.
        begin / finish: fork side streams from / join them into the launching stream inside the timed region."""
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        w0 = time.time()
        e0.record(stream)
        if begin:
            begin()
        for _ in range(steps):
            fn()
        if finish:
            finish()
        e1.record(stream)
        barrier()
        w1 = time.time()
        ms = R.max_over_ranks(e0.elapsed_time(e1), world, device="cuda")
        return ms, w0, w1

    # ---- value: everything resident in HBM, the call a user makes (kernels chained by programmatic launch) ----
    for _ in range(args.warmup):
        plan.step(d_psi, cn_per)
    torch.cuda.synchronize()
    launches0 = plan.info()["launches"]
    sampler = ClockSampler(local, args.clock_interval_ms)
    sampler.start()
    time.sleep(0.1)
    ms, w0, w1 = timed_region(lambda: plan.step(d_psi, cn_per), args.steps)
    launches = plan.info()["launches"] - launches0
    value = R.whole_job_throughput(cfg.N, cn_per * args.steps, ms, world)

    # ---- the same K steps again with a CUDA-event pair around every fused-pass launch and every RS chain on the
    # launching stream (CN_OPT_PROFILE).  Events between launches switch the programmatic overlap off, so this
    # second region is only used for the per-kernel duration of the roofline, never for `value`. ----------------
    plan.set_option(B.CN_OPT_PROFILE, 1)
    plan.step(d_psi, cn_per)
    torch.cuda.synchronize()
    plan.profile()  # drop warm-up samples
    ms_prof, _, w1 = timed_region(lambda: plan.step(d_psi, cn_per), args.steps)
    clocks = sampler.stop(w0, w1)
    prof = plan.profile()
    plan.set_option(B.CN_OPT_PROFILE, 0)

    # ---- roofline of the dominant kernel (fused pass) -----------------------------------------------------
    peak, peak_src = measured_peaks()
    pass_ms = prof["pass_ms"] / max(1, prof["pass_count"])
    achieved = BYTES_PER_POINT_STEP * cfg.N / (pass_ms * 1e-3) / 1e9 if prof["pass_count"] else None
    traffic, traffic_src = ncu_traffic_per_launch()
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": (achieved / peak) if achieved else None, "traffic": traffic, "traffic_source": traffic_src,
                "kernel": "k_pass_tiled<TPB,LOGC,P1=1,P2=1> (fused SS(k) + RHS/RD/RU/JD/JU(k+1))",
                "kernel_ms": pass_ms, "launches_timed": prof["pass_count"],
                "rs_chain_ms": prof["rs_ms"] / max(1, prof["rs_count"]),
                "timing": "CUDA-event pair around each fused-pass launch over a second timed region of the same K steps "
                          "(events between launches disable the PDL overlap that `value` has)",
                "ms_per_step_profiled": ms_prof / args.steps,
                "algorithmic_bytes_per_launch": BYTES_PER_POINT_STEP * cfg.N, "peak_source": peak_src,
                "bytes_per_point": {"declared_minimum_SURVEY_8d": BYTES_PER_POINT_STEP,
                                    "moved_by_this_formulation": BYTES_MOVED_PER_POINT},
                "achieved_on_bytes_moved": (BYTES_MOVED_PER_POINT * cfg.N / (pass_ms * 1e-3) / 1e9) if prof["pass_count"] else None,
                "frac_on_bytes_moved": (BYTES_MOVED_PER_POINT * cfg.N / (pass_ms * 1e-3) / 1e9 / peak) if prof["pass_count"] else None,
                "whole_step_GBps": BYTES_PER_POINT_STEP * cfg.N * cn_per * args.steps / (ms * 1e-3) / 1e9}

    # ---- e2e: every bench step takes its wave function from PINNED HOST memory (H2D), advances it by cn_per CN steps
    # through the public API and returns the result to pinned host memory (D2H), all inside the timed region.  The
    # steps are independent batches, so the copies of neighbouring steps overlap the compute: two device buffers,
    # copy-in / compute / copy-out on three streams chained by events (the API is asynchronous on the caller's stream).
    e2e = None
    if not args.no_e2e:
        s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
        d_buf = [d_psi, torch.empty_like(d_psi)]
        h_out = [torch.empty_like(psi_pin).pin_memory(), torch.empty_like(psi_pin).pin_memory()]
        ev_in = [torch.cuda.Event() for _ in range(2)]
        ev_cmp = [torch.cuda.Event() for _ in range(2)]
        ev_out = [torch.cuda.Event() for _ in range(2)]
        state = {"i": 0}

        def e2e_begin():
            s_in.wait_stream(stream)
            s_out.wait_stream(stream)
            for b in range(2):
                ev_out[b].record(s_out)

        def e2e_step():
            b = state["i"] & 1
            state["i"] += 1
            s_in.wait_event(ev_out[b])            # the buffer's previous result has left the device
            with torch.cuda.stream(s_in):
                d_buf[b].copy_(psi_pin, non_blocking=True)
                ev_in[b].record(s_in)
            stream.wait_event(ev_in[b])
            plan.step(d_buf[b], cn_per)
            ev_cmp[b].record(stream)
            s_out.wait_event(ev_cmp[b])
            with torch.cuda.stream(s_out):
                h_out[b].copy_(d_buf[b], non_blocking=True)
                ev_out[b].record(s_out)

        def e2e_finish():
            stream.wait_stream(s_out)
            stream.wait_stream(s_in)

        timed_region(e2e_step, 2, e2e_begin, e2e_finish)  # warm-up
        ms_e, _, _ = timed_region(e2e_step, args.steps, e2e_begin, e2e_finish)
        e2e = {"value": R.whole_job_throughput(cfg.N, cn_per * args.steps, ms_e, world), "unit": UNIT,
               "h2d_bytes_per_step": 16 * cfg.N, "d2h_bytes_per_step": 16 * cfg.N,
               "ms_per_step": ms_e / args.steps,
               "pipeline": "independent batches; H2D | cn_step | D2H on three streams over two device buffers"}

    # ---- optional P sweep (config C2: P = 2^8..2^16 against the paper's optimal-P model) -----------------
    sweep = None
    if args.sweep and rank == 0:
        sweep = []
        for Pk in cfg.P_sweep:
            pl = B.Plan(cfg.N, Pk, cfg.dx, cfg.dt, V).factorize()
            info = pl.info()
            n = 20 if info["path"] == B.PATH_TILED else 2
            pl.step(d_psi, 2)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            pl.step(d_psi, n)
            e1.record(stream)
            torch.cuda.synchronize()
            sweep.append({"P": Pk, "path": info["path"], "us_per_cn_step": 1e3 * e0.elapsed_time(e1) / n})
            pl.close()

    # ---- cpu_baseline: the oracle as it stands on this box's host cores, bounded sample (rank 0, N = 1) ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        nsamp = 24
        sec, _ = oracle_timed(cfg, V, psi_h, nsamp)
        cpu = {"value": cfg.N * nsamp / sec / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
               "host_cores_available": os.cpu_count(),
               "sample": "first %d of the 1000 CN steps of C2 at full N=2^24 (serial Thomas, 1 thread)" % nsamp}

    # ---- the other configs under the same clock (rank 0, N = 1): a few ms of GPU time each ------------------
    info = plan.info()
    per_config = None
    if rank == 0 and world == 1 and not args.no_per_config:
        per_config = per_config_report(torch, peak, args.full, not args.no_cpu_baseline)

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": bench_config(cfg, P, world),
            "launch": {"cn_steps_per_bench_step": cn_per, "path": info["path"], "P_effective": info["P_effective"],
                       "tile_threads": info["tile_threads"], "rs_levels": info["rs_levels"], "factorize_ms": factor_ms},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
            "cpu_baseline": cpu, "per_config": per_config,
        }
        if sweep is not None:
            line["p_sweep"] = sweep
        print(json.dumps(line), flush=True)
    plan.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
