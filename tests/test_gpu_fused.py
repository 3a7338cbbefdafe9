"""The fused step loop (include/axg.h axg_set_fusion): inside axg_step(n > 1) with count binning, P2b/P2c
of step t run inside the diffusion kernel of step t+1.  Checked two ways:
  * against the one-kernel-per-phase path of the same library, bit for bit, on every field axg_read_state reports
    (the arithmetic is the same, so nothing may differ) -- sizes around the tile (1024 rows), cells far larger than a
    tile (they straddle tile boundaries), both species modes;
  * against the oracle after several whole steps: integers bit-exact while no boundary flip happened (reading A-19),
    positions and cones within NS's tolerance.
"""
import numpy as np
import pytest

from oracle import axo
from paper_1405_3331_b200 import workloads as W

import parity_util as pu

pytestmark = pytest.mark.gpu

FIELDS = ("PART_X", "PART_Y", "PART_Z", "PART_SPECIES", "PART_ID", "KEYS_SORTED", "PERM", "CELL_START", "CELL_END",
          "CONE_POS", "CONE_HEADING", "CONE_STATE", "CONE_COUNTS", "CONE_MOMENT", "CONE_GRADIENT", "POLY_LEN",
          "POLYLINE", "PRE_X", "PRE_Y", "PRE_Z", "PRE_ID", "PRE_SPECIES", "PRE_KEY")


@pytest.fixture(scope="module")
def axg():
    from paper_1405_3331_b200 import axg as m
    m.lib()
    return m


def _make(axg, w, fuse, n, seed, n_species, crowd=None):
    g = axg.Axg(w.grid, w.D, w.emission, w.radius, w.speed, w.noise, w.seed)
    g.set_binning(axg.BIN_COUNT)
    g.set_fusion(fuse)
    W.apply(g, w)
    x, y, z, sp, ids = W.random_particles(seed, n, w.grid, n_species=n_species)
    if crowd is not None and n:  # most particles inside a few cells: cells of thousands of members
        k = int(n * 0.8)
        for a, c in zip((x, y, z), crowd):
            a[:k] = c + (a[:k] - np.floor(a[:k])) * 1.5
    g.load_particles(x, y, z, sp, ids, next_id=n, step=5)
    return g


def _same(a, b):
    assert a.shape == b.shape
    assert a.dtype == b.dtype
    assert np.array_equal(a.view(np.uint8), b.view(np.uint8))


@pytest.mark.parametrize("n", [0, 1, 31, 1023, 1024, 1025, 3071, 3072, 3073, 40_009])
@pytest.mark.parametrize("fuse", [1, 2])
def test_fused_equals_unfused(axg, n, fuse):
    w = W.small(seed=21 + n % 5, n_cones=17)
    steps = 4
    g0 = _make(axg, w, axg.FUSE_OFF, n, 100 + n, 2)
    g1 = _make(axg, w, fuse, n, 100 + n, 2)
    for _ in range(steps):
        g0.step(1)
    g1.step(steps)
    assert g0.counters() == g1.counters()
    for f in FIELDS:
        _same(g0.read_state(f), g1.read_state(f))
    g0.close()
    g1.close()


@pytest.mark.parametrize("n_species", [1, 2])
def test_fused_crowded_cells_straddle_tiles(axg, n_species):
    """80 % of 20 000 particles start inside a 1.5-cell cube, D small: cells hold thousands of members, far more
    than the 1024 rows of a tile, so most tiles lie inside one cell and every boundary case of the settle phase runs."""
    w = W.small(seed=31, grid=(12, 10, 9), n_cones=12, two_species=(n_species == 2))
    w.D = 0.02
    g0 = _make(axg, w, axg.FUSE_OFF, 20_000, 7, n_species, crowd=(5.0, 4.0, 3.0))
    g1 = _make(axg, w, axg.FUSE_ON, 20_000, 7, n_species, crowd=(5.0, 4.0, 3.0))
    for _ in range(3):
        g0.step(1)
    g1.step(3)
    assert g0.counters() == g1.counters()
    occupancy = g1.read_state("CELL_END").astype(np.int64) - g1.read_state("CELL_START")
    assert occupancy.max() > 2048
    for f in FIELDS:
        _same(g0.read_state(f), g1.read_state(f))
    g0.close()
    g1.close()


def test_fused_split_calls_equal_one_call(axg):
    """axg_step(2) + axg_step(3) == axg_step(5): the closing reorder of a call leaves the state the next call needs."""
    w = W.small(seed=33, n_cones=20)
    g0 = _make(axg, w, axg.FUSE_ON, 30_000, 9, 2)
    g1 = _make(axg, w, axg.FUSE_ON, 30_000, 9, 2)
    g0.step(2)
    g0.step(3)
    g1.step(5)
    for f in FIELDS:
        _same(g0.read_state(f), g1.read_state(f))
    g0.close()
    g1.close()


def test_fused_against_oracle(axg):
    """Three whole steps in one fused call against three oracle steps from the same loaded state."""
    w = W.small(seed=35, n_cones=24)
    n, steps = 25_013, 3
    g = axg.Axg(w.grid, w.D, w.emission, w.radius, w.speed, w.noise, w.seed)
    g.set_binning(axg.BIN_COUNT)
    g.set_fusion(axg.FUSE_ON)
    o = axo.Oracle(w.grid, w.D, w.emission, w.radius, w.speed, w.noise, w.seed)
    W.apply(g, w)
    W.apply(o, w)
    pu.load_same_particles(g, o, 41, n, w.grid, n_species=2, step=0)
    g.step(steps)
    o.step(steps)
    gc, oc = g.counters(), o.counters()
    assert gc["step"] == oc["step"] == steps and gc["next_id"] == oc["next_id"] and gc["emitted"] == oc["emitted"]
    gid, oid = g.read_state("PART_ID"), o.read_state("PART_ID")
    if gid.shape == oid.shape and np.array_equal(gid, oid):   # no boundary flip (A-19) in 75 000 particle-steps
        for f in ("KEYS_SORTED", "PERM", "CELL_START", "CELL_END", "PART_SPECIES"):
            assert np.array_equal(g.read_state(f), o.read_state(f)), f
        for f in ("PART_X", "PART_Y", "PART_Z"):
            a, b = g.read_state(f), o.read_state(f)
            assert pu.close(a, b).all(), (f, np.abs(a - b).max())
        pu.compare_sense(g, o)
        pu.compare_cones(g, o)
    else:  # a flip: the populations still agree up to a handful of particles
        assert abs(len(gid) - len(oid)) <= 4
        assert len(np.setxor1d(gid, oid)) <= 8
    g.close()
    o.close()


@pytest.mark.parametrize("n", [20_000, 90_000])
def test_crowded_cells_binning_against_oracle(axg, n):
    """Cells above AXG_BIG_CELL members take the sorted-slot path (k_sort_big_cells: shared-memory network up to 8192
    members, in-place global network above): binning of a crowded population against std::stable_sort, bit for bit."""
    grid = (12, 10, 9)
    g = axg.Axg(grid, 0.5, 1, 2.0, 0.25, 0.1, 3)
    g.set_binning(axg.BIN_COUNT)
    o = axo.Oracle(grid, 0.5, 1, 2.0, 0.25, 0.1, 3)
    g.set_capacity(n + 16, 4)
    o.set_capacity(n + 16, 4)
    x, y, z, sp, ids = W.random_particles(5, n, grid, n_species=2)
    k = int(n * 0.8)
    for a, c in zip((x, y, z), (5.0, 4.0, 3.0)):
        a[:k] = c + (a[:k] - np.floor(a[:k])) * 1.5
    for s in (g, o):
        s.load_particles(x, y, z, sp, ids, next_id=n, step=0)
    g.step_phase(axg.PHASE_BIN)
    o.step_phase(axo.PHASE_BIN)
    occupancy = o.read_state("CELL_END").astype(np.int64) - o.read_state("CELL_START")
    assert occupancy.max() > (8192 if n > 50_000 else 2048)
    pu.compare_binning(g, o)
    g.close()
    o.close()
