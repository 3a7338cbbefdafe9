"""Multi-GPU step loop: the workload sharded BY SOURCE, one integer all-reduce per step.

Rank r owns the sources s with s % world == r and every particle they emit (`set_shard`; the other sources still
consume their particle ids, so each particle's Philox stream -- hence its trajectory -- equals the 1-GPU run).  Every
rank senses ALL cones over its own particles; the per-cone integer sums (n_s, M_s) are additive over disjoint particle
sets, so one all-reduce(sum) between P3 and P4 gives every rank the 1-GPU sums exactly, and P4/P5 run replicated,
bit-identical on every rank.  No particle ever moves between ranks.

Host logic only (no arithmetic of the method): the loop drives any object with the boundary's call names -- the
CUDA binding (NCCL all-reduce on the device buffer, no host synchronisation inside the loop) or, in the world_size-2
`gloo` tests, the CPU oracle binding.
"""
from __future__ import annotations

import numpy as np

PHASE_DIFFUSE, PHASE_BIN, PHASE_SENSE, PHASE_ADVANCE, PHASE_COMMIT = 1, 2, 4, 8, 16


class _DevBuf:
    """A raw device pointer presented through __cuda_array_interface__ so that torch can wrap it without a copy."""

    def __init__(self, ptr, n_int32):
        self.__cuda_array_interface__ = {"shape": (n_int32,), "typestr": "<i4", "data": (int(ptr), False), "version": 2}


def nccl_exchange(sim):
    """all-reduce(sum) of the ctx-owned int32 sense buffer, in place, on torch's current stream (= the ctx stream)."""
    import torch
    import torch.distributed as dist
    ptr, nbytes = sim.sense_buffer()
    if not ptr:
        return lambda: None
    t = torch.as_tensor(_DevBuf(ptr, nbytes // 4), device="cuda")

    def run():
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return run


def host_exchange(sim):
    """The same exchange for a binding whose sums live on the host (oracle): read -> all-reduce (gloo) -> load."""
    import torch
    import torch.distributed as dist

    def run():
        c = torch.from_numpy(sim.read_state("CONE_COUNTS").astype(np.int64))
        m = torch.from_numpy(sim.read_state("CONE_MOMENT").astype(np.int64))
        if c.numel() == 0:
            return
        # frozen cones keep stale sums on every rank; they are not read by P4, only kept consistent here
        dist.all_reduce(c, op=dist.ReduceOp.SUM)
        dist.all_reduce(m, op=dist.ReduceOp.SUM)
        sim.load_sense(c.numpy(), m.numpy())
    return run


class ShardedStepper:
    """`step(n)` of a simulation sharded over `world` ranks.  `exchange` is nccl_exchange or host_exchange."""

    def __init__(self, sim, rank, world, exchange):
        self.sim, self.rank, self.world = sim, int(rank), int(world)
        sim.set_shard(self.rank, self.world)
        self._exchange = exchange(sim) if self.world > 1 else (lambda: None)

    def step(self, n=1):
        sim = self.sim
        sim.check_capacity(n)
        for _ in range(n):
            sim.enqueue_phase(PHASE_DIFFUSE | PHASE_BIN | PHASE_SENSE)
            self._exchange()
            sim.enqueue_phase(PHASE_ADVANCE | PHASE_COMMIT)
        sim.sync()


def owned_sources(n_sources, rank, world):
    """Indices of the sources rank `rank` emits (the rule both libraries implement in set_shard)."""
    return [s for s in range(n_sources) if s % world == rank]
