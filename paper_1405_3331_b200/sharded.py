"""Multi-GPU step loop: the workload sharded BY SOURCE, one integer all-reduce per step.

Rank r owns the sources s with s % world == r and every particle they emit (`set_shard`; the other sources still
consume their particle ids, so each particle's Philox stream -- hence its trajectory -- equals the 1-GPU run).  Every
rank senses ALL cones over its own particles; the per-cone integer sums (n_s, M_s) are additive over disjoint particle
sets, so one all-reduce(sum) between P3 and P4 gives every rank the 1-GPU sums exactly, and P4/P5 run replicated,
bit-identical on every rank.  No particle ever moves between ranks.

Host logic only (no arithmetic of the method): the loop drives any object with the boundary's call names -- the
CUDA binding (NCCL all-reduce on the device buffer, no host synchronisation inside the loop) or, in the world_size-2
`gloo` tests, any other object with the same calls and an exchange function of the test's own.
"""
from __future__ import annotations

import numpy as np

PHASE_DIFFUSE, PHASE_BIN, PHASE_SENSE, PHASE_ADVANCE, PHASE_COMMIT, PHASE_CONNECT = 1, 2, 4, 8, 16, 32


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


class ShardedStepper:
    """`step(n)` of a simulation sharded over `world` ranks.  `exchange(sim)` returns the callable that all-reduces the
    per-cone sums between P3 and P4 (nccl_exchange here; the CPU tests pass their own).

    With the CUDA binding (an object that has `enqueue_phase_on`) the loop is the one `axg_step` runs on one GPU, with
    the all-reduce in it: P3, the all-reduce and P4 / P5 of step t go to a side stream BESIDE P1 of step t+1 on the main
    stream (they share no data), joined before P2 of step t+1; for n >= 4 one such unit is captured once as a CUDA graph
    (NCCL collectives are capturable) and replayed, re-captured when `params_fingerprint` says a launch would be stale.
    Bindings without streams (the oracle in the gloo tests) run the plain sequence."""

    GRAPH_MIN_STEPS = 4

    def __init__(self, sim, rank, world, exchange, overlap=None, graph=True):
        self.sim, self.rank, self.world = sim, int(rank), int(world)
        sim.set_shard(self.rank, self.world)
        self._exchange = exchange(sim) if self.world > 1 else (lambda: None)
        self._overlap = hasattr(sim, "enqueue_phase_on") if overlap is None else bool(overlap)
        import os
        self._use_graph = bool(graph) and os.environ.get("AXG_SHARDED_GRAPH", "1") != "0"
        self._side = None
        self._graph = None
        self._graph_fp = None
        self._graph_stream = None

    # ---- plain sequence (any binding) ----------------------------------------------------------------------------
    def _step_plain(self, n):
        sim = self.sim
        for _ in range(n):
            sim.enqueue_phase(PHASE_DIFFUSE | PHASE_BIN | PHASE_SENSE)
            self._exchange()
            sim.enqueue_phase(PHASE_ADVANCE | PHASE_CONNECT | PHASE_COMMIT)

    # ---- overlapped sequence (CUDA binding) ---------------------------------------------------------------------------
    def _cones(self, stream, torch):
        sim = self.sim
        sim.enqueue_phase_on(PHASE_SENSE, stream.cuda_stream)
        with torch.cuda.stream(stream):
            self._exchange()
        sim.enqueue_phase_on(PHASE_ADVANCE | PHASE_CONNECT | PHASE_COMMIT, stream.cuda_stream, overlapped=True)

    def _unit(self, main, prev_cones, torch):
        """[cones of the previous step on the side stream || P1 of this step] -> P2 of this step"""
        sim = self.sim
        if prev_cones:
            self._side.wait_stream(main)
            self._cones(self._side, torch)
        sim.enqueue_phase_on(PHASE_DIFFUSE, main.cuda_stream)
        if prev_cones:
            main.wait_stream(self._side)
        sim.enqueue_phase_on(PHASE_BIN, main.cuda_stream)

    def _step_overlapped(self, n):
        import torch
        main = torch.cuda.current_stream()
        if self._side is None:
            self._side = torch.cuda.Stream()
        self._unit(main, False, torch)
        rest = n - 1
        if rest > 0 and self._use_graph and n >= self.GRAPH_MIN_STEPS:
            fp = self.sim.params_fingerprint()
            if self._graph is None or self._graph_fp != fp:
                # one unit eagerly first: the first collective on a communicator / stream allocates, which a capture
                # does not allow
                self._unit(main, True, torch)
                rest -= 1
                try:
                    g = torch.cuda.CUDAGraph()
                    torch.cuda.synchronize()
                    with torch.cuda.graph(g, capture_error_mode="thread_local"):
                        self._unit(torch.cuda.current_stream(), True, torch)
                    self._graph, self._graph_fp = g, fp
                except Exception as e:   # a collective that cannot be captured here: nothing of the unit has run (the
                    # library's host-side flags end a unit as they began it), so go on without graphs
                    import sys
                    print("[sharded] CUDA-graph capture of the step failed (%s): running without graphs" % e,
                          file=sys.stderr, flush=True)
                    self._graph, self._use_graph = None, False
                    try:
                        torch.cuda.synchronize()
                    except Exception:
                        pass
            if self._graph is not None:
                for _ in range(rest):
                    self._graph.replay()
            else:
                for _ in range(rest):
                    self._unit(main, True, torch)
        else:
            for _ in range(rest):
                self._unit(main, True, torch)
        self._cones(main, torch)      # P3..P5 of the last step

    def step(self, n=1):
        if n <= 0:
            return
        self.sim.check_capacity(n)
        if self._overlap:
            self._step_overlapped(n)
        else:
            self._step_plain(n)
        self.sim.sync()


def owned_sources(n_sources, rank, world):
    """Indices of the sources rank `rank` emits (the rule both libraries implement in set_shard)."""
    return [s for s in range(n_sources) if s % world == rank]
