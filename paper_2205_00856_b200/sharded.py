"""Sharded mode: the host protocol around the `cn_shard_*` calls.

One system is spread over `nshards` processes; the wave function is never gathered.  Per step
every shard all-gathers ONE small record around the RS stage ("collecting four values per process
... after the RS stage, two support values must be made available to each process"; here 2 nt values per shard with
the matrix pre-factored, and the support values are computed locally from the gathered records because the last RS
level is replicated).  This module holds no arithmetic of the method: it moves opaque records.

The protocol is written ONCE, as a generator that yields a record to send and is resumed with the gathered records:

    factorize_protocol(plan, alloc) / run_protocol(plan, psi, nsteps, alloc)

and driven either by `DistributedStepper` (one process per GPU, `torch.distributed.all_gather_into_tensor`: NCCL over
NVLink on GPUs, gloo in the CPU test of the protocol) or by `LocalShards` (all shards in one process on one device,
the gather is a concatenation: how the GPU parity tests run 2 and 4 shards on the single GPU of this build).
`plan` is a `binding.ShardPlan` or anything with the same methods (the CPU test uses a numpy stand-in).
"""
from __future__ import annotations


def factorize_protocol(plan, alloc):
    """Matrix side, once per (H, dt).  alloc(count) -> zeroed complex128 record on the plan's device."""
    mcount, _ = plan.counts()
    send = alloc(mcount)
    plan.factorize_local(send)
    gathered = yield send
    plan.factorize_finish(gathered)


def run_protocol(plan, psi, nsteps, alloc):
    """nsteps CN steps of this shard's rows `psi`, in place: nsteps + 1 exchanges (one of them the psi^0 edge values)."""
    if nsteps <= 0:
        return
    _, scount = plan.counts()
    edge = alloc(1)
    plan.edge(psi, edge)
    edges = yield edge
    send = [alloc(scount), alloc(scount)]  # two records: the one in flight must not be overwritten by the next pass
    plan.prologue(psi, edges, send[0])
    gathered = yield send[0]
    for k in range(1, nsteps):
        plan.advance(psi, gathered, send[k & 1])
        gathered = yield send[k & 1]
    plan.epilogue(psi, gathered)


class LocalShards:
    """All shards of one system in ONE process (one device, one stream): drives the per-shard generators in lockstep;
    the all-gather is a concatenation of the records.  Used by the single-GPU parity tests and by `bench`-style
    measurements of the protocol's launch overhead; a real multi-GPU job uses `DistributedStepper`."""

    def __init__(self, plans, alloc, cat):
        self.plans, self.alloc, self.cat = list(plans), alloc, cat

    def _drive(self, gens):
        sends = [next(g) for g in gens]
        while True:
            gathered = self.cat(sends)
            nxt, done = [], 0
            for g in gens:
                try:
                    nxt.append(g.send(gathered))
                except StopIteration:
                    done += 1
            if done:
                assert done == len(gens), "shards left the protocol at different points"
                return
            sends = nxt

    def factorize(self):
        self._drive([factorize_protocol(p, self.alloc) for p in self.plans])

    def step(self, psis, nsteps):
        if nsteps > 0:
            self._drive([run_protocol(p, x, nsteps, self.alloc) for p, x in zip(self.plans, psis)])


class DistributedStepper:
    """One shard per process: the records are all-gathered with `torch.distributed` on the current stream (NCCL orders
    the collective after the kernels that wrote the record and before the kernels that read the result, so the host
    never synchronises inside a run).  Masking: the exchange is one small message per step; while
    it is in flight the next pass kernel is already resident and prefetching its first psi / q / gamma tiles
    (programmatic dependent launch), which depend on nothing that is exchanged."""

    def __init__(self, plan, group=None, device=None, dist=None):
        """dist: anything with get_world_size / all_gather_into_tensor (default: torch.distributed, initialised)."""
        import torch
        if dist is None:
            import torch.distributed as dist
        self.torch, self.dist, self.plan, self.group = torch, dist, plan, group
        self.world = dist.get_world_size(group)
        self.device = device if device is not None else (torch.device("cuda", torch.cuda.current_device())
                                                         if torch.cuda.is_available() else torch.device("cpu"))

    def _alloc(self, count):
        return self.torch.zeros(count, dtype=self.torch.complex128, device=self.device)

    def _gather(self, send):
        out = self.torch.empty(self.world * send.numel(), dtype=send.dtype, device=send.device)
        # complex128 travels as pairs of float64 (every backend moves those)
        self.dist.all_gather_into_tensor(self.torch.view_as_real(out), self.torch.view_as_real(send), group=self.group)
        return out

    def _drive(self, gen):
        try:
            send = next(gen)
            while True:
                send = gen.send(self._gather(send))
        except StopIteration:
            pass

    def factorize(self):
        self._drive(factorize_protocol(self.plan, self._alloc))

    def step(self, psi, nsteps):
        if nsteps > 0:
            self._drive(run_protocol(self.plan, psi, nsteps, self._alloc))
