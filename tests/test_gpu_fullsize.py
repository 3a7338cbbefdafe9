"""Full-size checks in the launch configuration that bench.py times (C3: 256^3 cells, 16 384 cones, 16 sources, the
measured ~10.8 M live particles): properties that hold at any size, sampled cells and cones recomputed one by one from
the arrays read back, and one whole step phase by phase against the oracle, which receives the library's snapshot as
its input (reading A-23)."""
import numpy as np
import pytest

from oracle import axo
from paper_1405_3331_b200 import workloads as W

import parity_util as pu

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def c3(request):
    from paper_1405_3331_b200 import axg as m
    m.lib()
    w = W.c3()
    w.max_segments = 64
    sim = W.prerun(lambda D, e: m.Axg(w.grid, D, e, w.radius, w.speed, w.noise, w.seed), w, coarse=16, relax=50)
    yield m, w, sim
    sim.close()


def _arrays(sim):
    return {k: sim.read_state("PART_" + k) for k in ("X", "Y", "Z", "SPECIES", "ID")}


@pytest.mark.parametrize("mode", ["count", "radix"])
def test_properties_and_samples(c3, mode):
    m, w, sim = c3
    sim.set_binning(m.BIN_COUNT if mode == "count" else m.BIN_RADIX)
    before = sim.counters()
    sim.step(3)
    c = sim.counters()
    n = c["n_live"]
    assert n > 5_000_000
    assert c["n_live"] == before["n_live"] + (c["emitted"] - before["emitted"]) - (c["absorbed"] - before["absorbed"])
    a = _arrays(sim)
    nx, ny, nz = w.grid
    key = (a["Z"].astype(np.int64) * ny + a["Y"].astype(np.int64)) * nx + a["X"].astype(np.int64)
    ks = sim.read_state("KEYS_SORTED").astype(np.int64)
    assert np.array_equal(key, ks)                              # the reordered SoA is in key order, keys match
    assert (np.diff(ks) >= 0).all()
    perm = sim.read_state("PERM")
    assert len(perm) == n and np.array_equal(np.sort(perm), np.arange(n, dtype=np.uint32))
    same = ks[1:] == ks[:-1]
    assert (perm[1:][same] > perm[:-1][same]).all()             # equal keys keep pre-sort order (stable)
    assert len(np.unique(a["ID"])) == n
    cs, ce = sim.read_state("CELL_START").astype(np.int64), sim.read_state("CELL_END").astype(np.int64)
    assert (ce - cs).sum() == n
    rng = np.random.default_rng(5)
    for cell in np.concatenate([rng.integers(0, w.cells, 200), rng.choice(ks, 200)]):
        lo, hi = np.searchsorted(ks, cell), np.searchsorted(ks, cell, side="right")
        assert (cs[cell], ce[cell]) == ((lo, hi) if hi > lo else (0, 0))
    # sampled cones: counts and moments recomputed from the particle arrays, all pairs
    sim.step_phase(m.PHASE_SENSE)
    counts = sim.read_state("CONE_COUNTS").reshape(-1, 4)
    moment = sim.read_state("CONE_MOMENT").reshape(-1, 4, 3)
    pos = sim.read_state("CONE_POS").reshape(-1, 3)
    state = sim.read_state("CONE_STATE")
    ix, iy, iz = a["X"].astype(np.int64), a["Y"].astype(np.int64), a["Z"].astype(np.int64)
    active = np.flatnonzero(state == 0)
    for cone in rng.choice(active, min(12, len(active)), replace=False):
        d = np.stack([ix - int(pos[cone, 0]), iy - int(pos[cone, 1]), iz - int(pos[cone, 2])], 1)
        near = (d * d).sum(1) <= int(w.radius * w.radius)
        for s in range(4):
            sel = near & (a["SPECIES"] == s)
            assert counts[cone, s] == sel.sum()
            assert np.array_equal(moment[cone, s], d[sel].sum(0) if sel.any() else np.zeros(3, np.int64))


def test_one_step_against_the_oracle(c3):
    m, w, sim = c3
    sim.set_binning(m.BIN_AUTO)
    a = _arrays(sim)
    c = sim.counters()
    o = axo.Oracle(w.grid, w.D, w.emission, w.radius, w.speed, w.noise, w.seed)
    W.apply(o, w)
    o.load_particles(a["X"], a["Y"], a["Z"], a["SPECIES"], a["ID"], next_id=c["next_id"], step=c["step"])
    o.load_cones(sim.read_state("CONE_POS"), sim.read_state("CONE_HEADING"), sim.read_state("CONE_STATE"),
                 sim.read_state("POLY_LEN"))
    sim.step_phase(m.PHASE_DIFFUSE | m.PHASE_BIN)
    o.step_phase(axo.PHASE_DIFFUSE)
    pu.compare_presort(pu.pre_arrays(sim), pu.pre_arrays(o), w.grid, w.emitted_per_step)
    pu.feed_gpu_presort_to_oracle(sim, o, c["step"])
    pu.compare_binning(sim, o)
    sim.step_phase(m.PHASE_SENSE)
    o.step_phase(axo.PHASE_SENSE)
    pu.compare_sense(sim, o, active_only=True)
    sim.step_phase(m.PHASE_ADVANCE | m.PHASE_COMMIT)
    o.step_phase(axo.PHASE_ADVANCE | axo.PHASE_COMMIT)
    for f in ("CONE_STATE", "POLY_LEN"):
        assert np.array_equal(sim.read_state(f), o.read_state(f))
    for f in ("CONE_POS", "CONE_HEADING"):
        assert pu.close(sim.read_state(f), o.read_state(f)).all()
    o.close()


@pytest.mark.parametrize("mode", [1, 2])
def test_particle_sensing_on_sampled_cones(c3, mode):
    """Per-particle sensing (reading A-26) at full size: the oracle's all-pairs loop over the 16 M particles
    for a sample of the active cones (the others are handed to it as frozen), bit for bit."""
    m, w, sim = c3
    sim.set_binning(m.BIN_AUTO)
    sim.step(2)
    a = _arrays(sim)
    c = sim.counters()
    state = sim.read_state("CONE_STATE")
    active = np.flatnonzero(state == 0)
    pick = np.random.default_rng(9 + mode).choice(active, min(10, len(active)), replace=False)
    masked = np.full_like(state, 2)
    masked[pick] = 0
    o = axo.Oracle(w.grid, w.D, w.emission, w.radius, w.speed, w.noise, w.seed)
    W.apply(o, w)
    o.set_sensing(mode)
    o.load_particles(a["X"], a["Y"], a["Z"], a["SPECIES"], a["ID"], next_id=c["next_id"], step=c["step"])
    o.load_cones(sim.read_state("CONE_POS"), sim.read_state("CONE_HEADING"), masked, sim.read_state("POLY_LEN"))
    o.step_phase(axo.PHASE_SENSE)
    try:
        sim.set_sensing(mode)
        sim.step_phase(m.PHASE_SENSE)
        gc = sim.read_state("CONE_COUNTS").reshape(-1, 4)[pick]
        gm = sim.read_state("CONE_MOMENT").reshape(-1, 12)[pick]
    finally:
        sim.set_sensing(m.SENSE_CELL)
    assert np.array_equal(gc, o.read_state("CONE_COUNTS").reshape(-1, 4)[pick])
    assert np.array_equal(gm, o.read_state("CONE_MOMENT").reshape(-1, 12)[pick])
    assert gc.sum() > 0
    o.close()


def test_brick_order_at_full_size():
    """C3 under the bricked cell order (reading A-27), the configuration `bench.py --key-order brick` times:
    properties that hold at any size, the key restated in numpy, sampled cells, and sampled cones recomputed all pairs."""
    from paper_1405_3331_b200 import axg as m
    m.lib()
    w = W.c3()
    w.max_segments = 32

    def make(D, e):
        s = m.Axg(w.grid, D, e, w.radius, w.speed, w.noise, w.seed)
        s.set_key_order(m.KEY_BRICK)
        return s

    sim = W.prerun(make, w, coarse=16, relax=20)
    try:
        sim.step(3)
        n = sim.counters()["n_live"]
        assert n > 5_000_000
        a = _arrays(sim)
        nx, ny, nz = w.grid
        ix, iy, iz = a["X"].astype(np.int64), a["Y"].astype(np.int64), a["Z"].astype(np.int64)
        key = ((iz // 4 * (ny // 4) + iy // 4) * (nx // 8) + ix // 8) * 128 + iz % 4 * 32 + iy % 4 * 8 + ix % 8
        ks = sim.read_state("KEYS_SORTED").astype(np.int64)
        assert np.array_equal(key, ks) and (np.diff(ks) >= 0).all()
        perm = sim.read_state("PERM")
        assert len(perm) == n and np.array_equal(np.sort(perm), np.arange(n, dtype=np.uint32))
        same = ks[1:] == ks[:-1]
        assert (perm[1:][same] > perm[:-1][same]).all()
        assert len(np.unique(a["ID"])) == n
        cs, ce = sim.read_state("CELL_START").astype(np.int64), sim.read_state("CELL_END").astype(np.int64)
        assert len(cs) == nx * ny * nz and (ce - cs).sum() == n
        rng = np.random.default_rng(6)
        for cell in np.concatenate([rng.integers(0, len(cs), 200), rng.choice(ks, 200)]):
            lo, hi = np.searchsorted(ks, cell), np.searchsorted(ks, cell, side="right")
            assert (cs[cell], ce[cell]) == ((lo, hi) if hi > lo else (0, 0))
        sim.step_phase(m.PHASE_SENSE)
        counts = sim.read_state("CONE_COUNTS").reshape(-1, 4)
        moment = sim.read_state("CONE_MOMENT").reshape(-1, 4, 3)
        pos = sim.read_state("CONE_POS").reshape(-1, 3)
        active = np.flatnonzero(sim.read_state("CONE_STATE") == 0)
        for cone in rng.choice(active, min(12, len(active)), replace=False):
            d = np.stack([ix - int(pos[cone, 0]), iy - int(pos[cone, 1]), iz - int(pos[cone, 2])], 1)
            near = (d * d).sum(1) <= int(w.radius * w.radius)
            for s in range(4):
                sel = near & (a["SPECIES"] == s)
                assert counts[cone, s] == sel.sum()
                assert np.array_equal(moment[cone, s], d[sel].sum(0) if sel.any() else np.zeros(3, np.int64))
    finally:
        sim.close()
