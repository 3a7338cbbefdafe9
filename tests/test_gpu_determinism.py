"""Determinism as the race detector: every field axg_read_state reports is a function of (seed, inputs)
alone.  The atomics of count binning arrive in arbitrary order, the look-back chains of the radix path resolve in
arbitrary order, P3..P5 of a step run on a side stream beside the next step's P1 -- none of it may show:
  * the same run twice, byte for byte;
  * one axg_step(n) call (streams overlapped) against n calls of axg_step(1);
  * count binning against radix binning, two different algorithms for P1d / P2, after 30 whole steps.
"""
import numpy as np
import pytest

from paper_1405_3331_b200 import workloads as W

pytestmark = pytest.mark.gpu

FIELDS = ("PART_X", "PART_Y", "PART_Z", "PART_SPECIES", "PART_ID", "KEYS_SORTED", "PERM", "CELL_START", "CELL_END",
          "CONE_POS", "CONE_HEADING", "CONE_STATE", "CONE_COUNTS", "CONE_MOMENT", "CONE_GRADIENT", "POLY_LEN",
          "POLYLINE", "PRE_X", "PRE_Y", "PRE_Z", "PRE_ID", "PRE_SPECIES", "PRE_KEY")
STEPS = 30


@pytest.fixture(scope="module")
def axg():
    from paper_1405_3331_b200 import axg as m
    m.lib()
    return m


def _run(axg, binning, calls, steering=None, sensing=0):
    w = W.small(seed=41, grid=(40, 33, 21), n_cones=300, n_sources=4, rate=300)
    w.max_particles = 1 << 18
    g = axg.Axg(w.grid, w.D, w.emission, w.radius, w.speed, w.noise, w.seed)
    g.set_binning(binning)
    if steering:
        g.set_steering(*steering)
    g.set_sensing(sensing)
    W.apply(g, w)
    x, y, z, sp, ids = W.random_particles(43, 120_007, w.grid, n_species=2)
    g.load_particles(x, y, z, sp, ids, next_id=len(ids), step=0)
    for n in calls:
        g.step(n)
    out = {f: g.read_state(f) for f in FIELDS}
    out["counters"] = g.counters()
    g.close()
    return out


def _same(a, b):
    assert a["counters"] == b["counters"]
    for f in FIELDS:
        assert a[f].shape == b[f].shape and a[f].dtype == b[f].dtype, f
        assert np.array_equal(a[f].view(np.uint8), b[f].view(np.uint8)), f


@pytest.mark.parametrize("binning", ["count", "radix"])
def test_same_run_twice(axg, binning):
    mode = axg.BIN_COUNT if binning == "count" else axg.BIN_RADIX
    _same(_run(axg, mode, [STEPS]), _run(axg, mode, [STEPS]))


@pytest.mark.parametrize("binning", ["count", "radix"])
def test_one_call_equals_many_calls(axg, binning):
    mode = axg.BIN_COUNT if binning == "count" else axg.BIN_RADIX
    _same(_run(axg, mode, [STEPS]), _run(axg, mode, [1] * STEPS))
    _same(_run(axg, mode, [STEPS]), _run(axg, mode, [7, 1, 22]))
    # n = 2, 3: the overlapped path without the CUDA graph (enqueue_phases with P3..P5 on the side stream)
    _same(_run(axg, mode, [STEPS]), _run(axg, mode, [2, 3, 2, 3, 3, 2, 15]))


def test_count_binning_equals_radix_binning(axg):
    a, b = _run(axg, axg.BIN_COUNT, [STEPS]), _run(axg, axg.BIN_RADIX, [STEPS])
    assert a["counters"]["absorbed"] > 1000 and a["counters"]["emitted"] == STEPS * (4 * 300 + 6)
    _same(a, b)


@pytest.mark.parametrize("sensing", [1, 2])
def test_particle_sensing_is_deterministic(axg, sensing):
    """per-particle sensing (reading A-26): graph replay vs single steps, count vs radix binning, byte for byte; and it
    is not the per-cell rule in disguise (the cones end up elsewhere)."""
    a = _run(axg, axg.BIN_COUNT, [STEPS], sensing=sensing)
    _same(a, _run(axg, axg.BIN_COUNT, [1] * STEPS, sensing=sensing))
    _same(a, _run(axg, axg.BIN_RADIX, [7, 1, 22], sensing=sensing))
    cell = _run(axg, axg.BIN_COUNT, [STEPS])
    assert not np.array_equal(a["CONE_POS"], cell["CONE_POS"])
    assert np.array_equal(a["PART_ID"], cell["PART_ID"])      # the particles do not depend on the cones


def test_count_equals_radix_with_the_fixed_turn_rule(axg):
    st = (1, 8.0, np.pi / 30)
    _same(_run(axg, axg.BIN_COUNT, [STEPS], st), _run(axg, axg.BIN_RADIX, [STEPS], st))


@pytest.mark.parametrize("sensing", [0, 1])   # per-cell rule; per-particle rule (integer sums too: reading A-26)
def test_two_shards_on_one_gpu_equal_the_unsharded_run(axg, sensing):
    """DESIGN.md §8 on the real library: two contexts sharded by source (axg_set_shard, the enqueue / sync calls of the
    multi-GPU loop), the all-reduce replaced by a sum of the two device buffers on the same stream.  The cones must be
    bit-identical to the unsharded run, and the two shards' particles together must be its particles, bit for bit.
    (One process, one GPU, the host drives both shards in turn: no kernel waits on another.)"""
    import torch
    from paper_1405_3331_b200 import sharded as S

    steps = 40
    w = W.small(seed=47, grid=(40, 33, 21), n_cones=200, n_sources=5, rate=150)
    w.max_particles = 1 << 17

    def make():
        g = axg.Axg(w.grid, w.D, w.emission, w.radius, w.speed, w.noise, w.seed)
        g.set_binning(axg.BIN_COUNT)
        g.set_sensing(sensing)
        W.apply(g, w)
        return g

    ref = make()
    ref.step(steps)
    shards = [make() for _ in range(2)]
    for r, g in enumerate(shards):
        g.set_shard(r, 2)
    bufs = []
    for g in shards:
        ptr, nbytes = g.sense_buffer()
        bufs.append(torch.as_tensor(S._DevBuf(ptr, nbytes // 4), device="cuda"))
    for g in shards:
        g.check_capacity(steps)
    for _ in range(steps):
        for g in shards:
            g.enqueue_phase(S.PHASE_DIFFUSE | S.PHASE_BIN | S.PHASE_SENSE)
        total = bufs[0] + bufs[1]          # torch's current stream = the stream of both contexts
        bufs[0].copy_(total)
        bufs[1].copy_(total)
        for g in shards:
            g.enqueue_phase(S.PHASE_ADVANCE | S.PHASE_COMMIT)
    for g in shards:
        g.sync()
    for f in ("CONE_POS", "CONE_HEADING", "CONE_STATE", "POLY_LEN", "POLYLINE", "CONE_GRADIENT"):
        a = ref.read_state(f)
        for g in shards:
            b = g.read_state(f)
            assert np.array_equal(a.view(np.uint8), b.view(np.uint8)), f
    cols = {k: np.concatenate([g.read_state("PART_" + k) for g in shards]) for k in ("ID", "X", "Y", "Z", "SPECIES")}
    order, rorder = np.argsort(cols["ID"], kind="stable"), np.argsort(ref.read_state("PART_ID"), kind="stable")
    assert len(order) == len(rorder) > 5000
    for k in ("ID", "X", "Y", "Z", "SPECIES"):
        a, b = ref.read_state("PART_" + k)[rorder], cols[k][order]
        assert np.array_equal(a.view(np.uint8), b.view(np.uint8)), k
    c = [g.counters() for g in shards]
    assert c[0]["emitted"] + c[1]["emitted"] == ref.counters()["emitted"]
    assert c[0]["next_id"] == c[1]["next_id"] == ref.counters()["next_id"]
    for g in shards + [ref]:
        g.close()


def test_sharded_stepper_with_a_real_nccl_all_reduce(axg):
    """The multi-GPU loop of paper_1405_3331_b200/sharded.py exactly as bench.py --gpus N runs it -- ShardedStepper, the
    NCCL all-reduce on the ctx-owned device buffer wrapped without a copy, no host synchronisation inside -- with a
    process group of ONE rank (the box has one GPU): must equal axg_step bit for bit."""
    import os
    import torch
    import torch.distributed as dist
    from paper_1405_3331_b200 import sharded as S

    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29571")
    own_group = not dist.is_initialized()
    if own_group:
        dist.init_process_group("nccl", rank=0, world_size=1)
    try:
        w = W.small(seed=53, grid=(40, 33, 21), n_cones=200, n_sources=5, rate=150)
        w.max_particles = 1 << 17

        def make():
            g = axg.Axg(w.grid, w.D, w.emission, w.radius, w.speed, w.noise, w.seed)
            g.set_binning(axg.BIN_COUNT)
            W.apply(g, w)
            return g

        ref, g, h = make(), make(), make()
        ref.step(25)
        st = S.ShardedStepper(g, 0, 1, S.nccl_exchange)
        st._exchange = S.nccl_exchange(g)   # with one rank the stepper would skip the exchange: force it
        assert st._overlap                  # the CUDA binding takes the overlapped, graph-captured loop
        st.step(25)                         # first unit eager, 24 replays of the captured unit, last cones eager
        torch.cuda.synchronize()
        for f in FIELDS:
            a, b = ref.read_state(f), g.read_state(f)
            assert np.array_equal(a.view(np.uint8), b.view(np.uint8)), f
        # every call pattern of the loop: plain (n = 1), overlapped without a graph (n = 2, 3), graph (n >= 4), and the
        # same stepper again after the context's parameters changed (the captured unit must be re-captured)
        st2 = S.ShardedStepper(h, 0, 1, S.nccl_exchange)
        st2._exchange = S.nccl_exchange(h)
        for n in (1, 2, 3, 5, 6):
            st2.step(n)
        h.set_capacity(w.max_particles + 4096, w.max_segments)
        st2.step(8)
        torch.cuda.synchronize()
        assert h.counters()["step"] == 25
        for f in FIELDS:
            a, b = ref.read_state(f), h.read_state(f)
            assert np.array_equal(a.view(np.uint8), b.view(np.uint8)), f
        ref.close()
        g.close()
        h.close()
    finally:
        if own_group:
            dist.destroy_process_group()
