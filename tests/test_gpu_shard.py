"""Sharded mode (cn_shard_*): ONE system spread over 1..8 shards, every shard a plan of its own that
sees only its rows of V and psi and the gathered records -- here all shards live on the one GPU of this build and
the all-gather is a concatenation (paper_2205_00856_b200.sharded.LocalShards; the same protocol generators drive a
real multi-process job).  psi of all shards, concatenated, against the oracle's plain Thomas stepper on the whole
system, element by element."""
import numpy as np
import pytest

from oracle import cn_oracle as O
from paper_2205_00856_b200 import binding as B
from paper_2205_00856_b200 import sharded as SH
from paper_2205_00856_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL_PSI = 1e-10
TOL_RES = 1e-12


def torch_():
    import torch
    return torch


def make_shards(cfg, V, S, P_local=None, **opts):
    torch = torch_()
    n = cfg.N // S
    assert n * S == cfg.N
    plans = [B.ShardPlan(n, P_local or max(1, n // 256), cfg.dx, cfg.dt, V[r * n:(r + 1) * n], r, S, **opts) for r in range(S)]
    alloc = lambda c: torch.zeros(c, dtype=torch.complex128, device="cuda")  # noqa: E731
    return plans, SH.LocalShards(plans, alloc, torch.cat)


def run_sharded(cfg, V, psi, S, nsteps, calls=1, P_local=None, **opts):
    torch = torch_()
    n = cfg.N // S
    plans, grp = make_shards(cfg, V, S, P_local, **opts)
    try:
        grp.factorize()
        parts = [torch.from_numpy(psi[r * n:(r + 1) * n].copy()).cuda() for r in range(S)]
        for _ in range(calls):
            grp.step(parts, nsteps)
        torch.cuda.synchronize()
        info = [p.info() for p in plans]
        counts = plans[0].counts()
        return np.concatenate([x.cpu().numpy() for x in parts]), info, counts
    finally:
        for p in plans:
            p.close()


def residual(dx, dt, V, old, new):
    s = dt / (4 * dx * dx)
    diag = 1 + 1j * (2 * s + 0.5 * dt * V)

    def apply(dg, off, x):
        y = dg * x
        y[1:] += off * x[:-1]
        y[:-1] += off * x[1:]
        return y
    d = apply(np.conj(diag), 1j * s, old)
    return np.linalg.norm(apply(diag, -1j * s, new) - d) / np.linalg.norm(d)


@pytest.mark.parametrize("S", [1, 2, 4, 8])
def test_c1_shape(S):
    """Config C1 (N = 4096, 100 steps) over S shards; level 0 is the last level (nt = joint lines of a shard)."""
    cfg = W.CONFIGS["C1"]
    V, psi = W.potential(cfg), W.psi0(cfg)
    ref = O.step(cfg.dx, cfg.dt, V, psi, cfg.steps)
    out, info, counts = run_sharded(cfg, V, psi, S, 10, calls=10)
    assert np.max(np.abs(out - ref)) <= TOL_PSI
    assert all(i["path"] == B.PATH_TILED for i in info) or S == 1  # (one shard: cn_plan_info reports what cn_step would run)
    one, _, _ = run_sharded(cfg, V, psi, S, 1)
    assert residual(cfg.dx, cfg.dt, V, psi, one) <= TOL_RES


@pytest.mark.parametrize("S,opts,P_local", [
    (2, {}, None),                   # 2048 joint lines per shard, one level: 2049 values per record
    (4, {}, None),
    (2, {"rs_topmax": 64}, None),    # two levels per shard (2048 -> 8 rows)
    (4, {"rs_topmax": 64}, None),
    (4, {"rs_topmax": 64, "rs_top_in_subst": 0}, None),  # the replicated last level by its own kernel under two-level shards
    (8, {"rs_topmax": 4, "pdl": 0}, None),               # three levels, plain launches
    (4, {"rs_topmax": 1}, None),     # levels down to ONE row per shard: 2 values per shard and step
    (8, {"rs_topmax": 1}, None),
    (2, {"rs_topmax": 1}, 1 << 16),  # blocks of 8 rows: 65536 -> 256 -> 1
    (3, {"rs_topmax": 16}, None),    # N is not a multiple of 3 * 256 for 2^20: uses the 786432 case below
])
def test_2p20_shape(S, opts, P_local):
    N = 786432 if S == 3 else 1 << 20
    cfg = W.scaled(W.CONFIGS["C2dense"], N=N)
    V, psi = W.potential(cfg), W.psi0(cfg)
    nsteps = 7
    ref = O.step(cfg.dx, cfg.dt, V, psi, nsteps)
    out, info, counts = run_sharded(cfg, V, psi, S, nsteps, P_local=P_local, **opts)
    err = float(np.max(np.abs(out - ref)))
    assert err <= TOL_PSI, (err, counts, [i["rs_levels"] for i in info])
    if opts.get("rs_topmax") == 1:
        assert counts[1] == 2  # the two values per process of PAPER.md:175
    one, _, _ = run_sharded(cfg, V, psi, S, 1, P_local=P_local, **opts)
    assert residual(cfg.dx, cfg.dt, V, psi, one) <= TOL_RES


@pytest.mark.parametrize("nsteps", [1, 2, 3])
def test_short_runs_and_strong_coupling(nsteps):
    """s = dt / (4 dx^2) = 12.5: the reduced systems are far from diagonal, so a wrong coupling between shards shows."""
    cfg = W.scaled(W.CONFIGS["C1"], N=1 << 16, dx=0.01, dt=0.005)
    V, psi = W.potential(cfg), W.psi0(cfg)
    ref = O.step(cfg.dx, cfg.dt, V, psi, nsteps)
    for S, opts in ((2, {}), (4, {"rs_topmax": 4}), (8, {"rs_topmax": 1})):
        out, _, _ = run_sharded(cfg, V, psi, S, nsteps, **opts)
        assert np.max(np.abs(out - ref)) <= TOL_PSI, (S, opts)


def test_sharded_equals_unsharded_plan():
    """The same system through cn_step (one plan) and through 4 shards: both within 1e-10 of the oracle and of each other."""
    torch = torch_()
    cfg = W.scaled(W.CONFIGS["C3"], N=1 << 18)
    V, psi = W.potential(cfg), W.psi0(cfg)
    d = torch.from_numpy(psi).cuda()
    with B.Plan(cfg.N, cfg.N // 256, cfg.dx, cfg.dt, V) as plan:
        plan.factorize()
        plan.step(d, 5)
        torch.cuda.synchronize()
    out, _, _ = run_sharded(cfg, V, psi, 4, 5, rs_topmax=8)
    assert np.max(np.abs(out - d.cpu().numpy())) <= 1e-12


def test_rejects_unequal_shards_and_wrong_calls():
    torch = torch_()
    cfg = W.scaled(W.CONFIGS["C1"], N=4096)
    V = W.potential(cfg)
    alloc = lambda c: torch.zeros(c, dtype=torch.complex128, device="cuda")  # noqa: E731
    with B.ShardPlan(2048, 8, cfg.dx, cfg.dt, V[:2048], 0, 2) as a, B.ShardPlan(1024, 4, cfg.dx, cfg.dt, V[2048:3072], 1, 2) as b:
        ma, mb = alloc(a.counts()[0]), alloc(b.counts()[0])
        a.factorize_local(ma)
        b.factorize_local(mb)
        with pytest.raises(B.CnError) as e:  # records of different lengths / shapes: the stamp check refuses them
            a.factorize_finish(torch.cat([ma, mb, alloc(64)]))
        assert e.value.status == B.CN_EINVAL
        with pytest.raises(B.CnError) as e:
            B.cn_factorize(a.h)          # a sharded plan is not factored by cn_factorize
        assert e.value.status == B.CN_EINVAL
        with pytest.raises(B.CnError) as e:
            a.prologue(alloc(2048), alloc(2), alloc(a.counts()[1]))
        assert e.value.status == B.CN_ENOTFACTORIZED
    with pytest.raises(B.CnError) as e:
        B.ShardPlan(1000, 4, cfg.dx, cfg.dt, V[:1000], 0, 2)  # N_local must be a multiple of 256
    assert e.value.status == B.CN_EINVAL


def test_callback_driven_run_threads():
    """cn_shard_factorize / cn_shard_run: the library drives the protocol and calls back for every exchange.  Four
    shards of one system, ONE HOST THREAD AND ONE STREAM PER SHARD on the single device (as four ranks would run); the
    callback emulates the all-gather with device copies into a shared buffer, events and a host barrier.  Against the
    oracle on the whole system."""
    import threading
    torch = torch_()
    from cuda.bindings import runtime as rt
    S, nsteps = 4, 9
    cfg = W.scaled(W.CONFIGS["C2dense"], N=1 << 19)
    V, psi = W.potential(cfg), W.psi0(cfg)
    ref = O.step(cfg.dx, cfg.dt, V, psi, nsteps)
    n = cfg.N // S
    maxc = 8192
    G = [torch.zeros(S * maxc, dtype=torch.complex128, device="cuda") for _ in range(2)]  # shared gather buffers (ping-pong)
    ev = [[torch.cuda.Event() for _ in range(2)] for _ in range(S)]
    bar = threading.Barrier(S)
    parts, errors = [None] * S, []

    def worker(r):
        try:
            torch.cuda.set_device(0)
            stream = torch.cuda.Stream()
            calls = [0]

            def exchange(send, recv, count, stream_ptr):
                idx = calls[0] & 1
                calls[0] += 1
                nb = 16 * count
                assert count <= maxc and stream_ptr == stream.cuda_stream
                e, = rt.cudaMemcpyAsync(G[idx].data_ptr() + r * nb, send, nb, rt.cudaMemcpyKind.cudaMemcpyDeviceToDevice, stream_ptr)
                assert e == rt.cudaError_t.cudaSuccess
                ev[r][idx].record(stream)
                bar.wait()                      # every shard has enqueued its contribution and recorded its event
                for k in range(S):
                    stream.wait_event(ev[k][idx])
                e, = rt.cudaMemcpyAsync(recv, G[idx].data_ptr(), S * nb, rt.cudaMemcpyKind.cudaMemcpyDeviceToDevice, stream_ptr)
                assert e == rt.cudaError_t.cudaSuccess
                bar.wait()                      # every shard has enqueued its waits: the events may be recorded again
                return B.CN_OK

            with torch.cuda.stream(stream):
                d = torch.from_numpy(psi[r * n:(r + 1) * n].copy()).cuda()
                with B.ShardPlan(n, n // 256, cfg.dx, cfg.dt, V[r * n:(r + 1) * n], r, S, rs_topmax=16) as plan:
                    plan.factorize(exchange, stream)
                    plan.run(d, 4, exchange, stream)
                    plan.run(d, nsteps - 4, exchange, stream)
                    stream.synchronize()
                parts[r] = d.cpu().numpy()
        except Exception as ex:  # pragma: no cover
            errors.append((r, repr(ex)))
            bar.abort()

    threads = [threading.Thread(target=worker, args=(r,)) for r in range(S)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=300)
    assert not errors, errors
    out = np.concatenate(parts)
    assert np.max(np.abs(out - ref)) <= TOL_PSI
