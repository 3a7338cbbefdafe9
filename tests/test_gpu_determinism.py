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


def _run(axg, binning, calls, steering=None):
    w = W.small(seed=41, grid=(40, 33, 21), n_cones=300, n_sources=4, rate=300)
    w.max_particles = 1 << 18
    g = axg.Axg(w.grid, w.D, w.emission, w.radius, w.speed, w.noise, w.seed)
    g.set_binning(binning)
    if steering:
        g.set_steering(*steering)
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


def test_count_binning_equals_radix_binning(axg):
    a, b = _run(axg, axg.BIN_COUNT, [STEPS]), _run(axg, axg.BIN_RADIX, [STEPS])
    assert a["counters"]["absorbed"] > 1000 and a["counters"]["emitted"] == STEPS * (4 * 300 + 6)
    _same(a, b)


def test_count_equals_radix_with_the_fixed_turn_rule(axg):
    st = (1, 8.0, np.pi / 30)
    _same(_run(axg, axg.BIN_COUNT, [STEPS], st), _run(axg, axg.BIN_RADIX, [STEPS], st))
