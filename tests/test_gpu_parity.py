"""GPU-vs-oracle parity of the whole hot path, phase by phase and end to end, through the C-ABI (ctypes binding).

Bars (BASELINE.json north_star): keys, sorted permutation, cellStart / cellEnd, per-cone counts and
moments BIT-EXACT (binning and sensing on identical post-diffusion positions); single-step fp32 positions, gradients,
headings within 1e-5 relative + 1e-6 absolute; multi-step runs statistically (tests/test_gpu_multistep.py).
"""
import numpy as np
import pytest

from oracle import axo
from paper_1405_3331_b200 import workloads as W

import parity_util as pu
from parity_util import (compare_binning, compare_cones, compare_presort, compare_sense, feed_gpu_presort_to_oracle,
                         load_same_particles, make_pair, pre_arrays)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", params=["radix", "count"])
def axg(request):
    """Every test runs under both binning modes (include/axg.h axg_set_binning): the results must be identical."""
    from paper_1405_3331_b200 import axg as m
    m.lib()
    pu.BINNING = m.BIN_RADIX if request.param == "radix" else m.BIN_COUNT
    yield m
    pu.BINNING = None


def _chain(axg, w, n, seed, steps=2, n_species=2, steering=None, sensing=None):
    """load -> [P1 | P2 | P3 | P4+P5] x steps, each phase compared; the oracle is re-fed the GPU's P1 output so that
    integer phases are compared on identical inputs."""
    g, o = make_pair(w, axg)
    if steering is not None:
        g.set_steering(*steering)
        o.set_steering(*steering)
    if sensing is not None:
        g.set_sensing(sensing)
        o.set_sensing(sensing)
    load_same_particles(g, o, seed, n, w.grid, n_species=n_species, step=3)
    flips = 0
    for k in range(steps):
        t = 3 + k
        g.step_phase(axg.PHASE_DIFFUSE | axg.PHASE_BIN)
        o.step_phase(axo.PHASE_DIFFUSE)
        gp, op = pre_arrays(g), pre_arrays(o)
        flips += compare_presort(gp, op, w.grid, w.emitted_per_step)
        gc, oc = g.counters(), o.counters()
        assert gc["next_id"] == oc["next_id"] and gc["step"] == oc["step"] == t
        assert gc["n_live"] == len(gp["ID"])
        assert gc["emitted"] == oc["emitted"]
        feed_gpu_presort_to_oracle(g, o, t)
        compare_binning(g, o)
        g.step_phase(axg.PHASE_SENSE)
        o.step_phase(axo.PHASE_SENSE)
        compare_sense(g, o)
        g.step_phase(axg.PHASE_ADVANCE | axg.PHASE_COMMIT)
        o.step_phase(axo.PHASE_ADVANCE | axo.PHASE_COMMIT)
        compare_cones(g, o)
        if sensing is not None:
            # per-particle sensing takes x - p in fp32: its integers are compared on identical cone positions, as the
            # binning is on identical particle positions (the positions agreed within tolerance just above)
            o.load_cones(g.read_state("CONE_POS"), g.read_state("CONE_HEADING"), g.read_state("CONE_STATE"),
                         g.read_state("POLY_LEN"))
    g.close()
    o.close()
    return flips


def test_chain_small_ragged_two_species(axg):
    w = W.small(seed=7)                      # 24 x 20 x 16 grid, 3 sources of both polarities, 24 cones anywhere
    _chain(axg, w, n=50_037, seed=11, steps=3)


def test_chain_single_species_fast_path(axg):
    w = W.small(seed=8, two_species=False, grid=(40, 33, 21), n_cones=200)
    _chain(axg, w, n=30_011, seed=12, steps=2, n_species=1)


def test_chain_radius3_three_pass_keys(axg):
    # 128 x 128 x 64 = 2^20 cells -> 3 digit passes; R = 3 stencil (123 cells); D = 1
    w = W.small(seed=9, grid=(128, 128, 64), n_cones=300, n_sources=5, radius=3.0)
    w.D = 1.0
    w.max_particles = 1 << 18
    _chain(axg, w, n=200_003, seed=13, steps=2)


@pytest.mark.parametrize("grid", [(64, 64, 40), (8, 8, 8), (512, 512, 512)])
def test_chain_nine_bit_digits(axg, grid):
    """Radix binning takes 9-bit digits where that saves a pass ("9-bit digits would take C4 to 3 passes"):
    18-bit keys (2 passes of 9 instead of 3 of 8), 9-bit keys (one pass) and C4's own 27-bit key space (3 instead of 4) --
    the latter with 3e5 particles around a few sources, so that all three digits are populated.  Bit-exact like every
    other binning case; under count binning these are three more grids."""
    w = W.small(seed=23, grid=grid, n_cones=50, n_sources=4, rate=30)
    if grid[0] == 512:
        w.max_particles = 1 << 19
        _chain(axg, w, n=300_007, seed=29, steps=1)
    else:
        _chain(axg, w, n=40_009, seed=29, steps=2)


@pytest.mark.parametrize("n", [0, 1, 31, 2048, 2049, 6144, 6145])
def test_chain_edge_sizes(axg, n):
    w = W.small(seed=10 + n % 7, n_cones=9)
    _chain(axg, w, n=n, seed=14 + n, steps=2)


def test_empty_everything(axg):
    """No particles, no sources, no cones: a step is a no-op that still commits."""
    g = pu.new_axg(axg, (8, 8, 8), 0.5, 1, 2.0, 0.25, 0.1, 1)
    g.step(3)
    c = g.counters()
    assert c["step"] == 3 and c["n_live"] == 0 and c["emitted"] == 0
    assert g.read_state("CELL_START").sum() == 0 and g.read_state("CELL_END").sum() == 0
    assert g.read_state("PART_X").size == 0
    g.close()


def test_binning_only_on_given_positions(axg):
    """AXG_PHASE_BIN alone: copy + re-key + sort + reorder + ranges, against std::stable_sort binning."""
    for seed, grid, n in ((1, (256, 256, 256), 300_000), (2, (7, 5, 3), 20_000), (3, (1024, 1024, 256), 100_000)):
        g = pu.new_axg(axg, grid, 0.5, 1, 2.0, 0.25, 0.1, seed)
        o = axo.Oracle(grid, 0.5, 1, 2.0, 0.25, 0.1, seed)
        g.set_capacity(n + 16, 8)
        o.set_capacity(n + 16, 8)
        load_same_particles(g, o, seed, n, grid)
        g.step_phase(axg.PHASE_BIN)
        o.step_phase(axo.PHASE_BIN)
        compare_binning(g, o)
        ks = g.read_state("KEYS_SORTED")
        assert (np.diff(ks.astype(np.int64)) >= 0).all()
        g.close()
        o.close()


def test_binning_with_the_wide_reorder_kernel(axg):
    """A particle capacity above 32 M selects the four-slots-per-thread reorder kernel (radix mode): same results."""
    grid, n, seed = (64, 48, 40), 123_457, 5
    g = pu.new_axg(axg, grid, 0.5, 1, 2.0, 0.25, 0.1, seed)
    o = axo.Oracle(grid, 0.5, 1, 2.0, 0.25, 0.1, seed)
    g.set_capacity(34_000_000, 8)
    o.set_capacity(34_000_000, 8)
    load_same_particles(g, o, seed, n, grid)
    g.step_phase(axg.PHASE_BIN)
    o.step_phase(axo.PHASE_BIN)
    compare_binning(g, o)
    g.close()
    o.close()


def test_table1_of_the_paper_on_gpu(axg, golden_dir):
    """PAPER.md:267-276 Table 1 (reading A-17): 6 particles in cells 9 6 6 4 6 4 of a 16-cell row."""
    cells = np.array([9, 6, 6, 4, 6, 4])
    g = pu.new_axg(axg, (16, 1, 1), 0.5, 1, 2.0, 0.25, 0.1, 1)
    x = cells.astype(np.float32) + 0.5
    zeros = np.zeros(6, np.float32)
    g.load_particles(x, zeros, zeros, np.zeros(6, np.uint8), np.arange(6, dtype=np.uint32), 6, 0)
    g.step_phase(axg.PHASE_BIN)
    assert g.read_state("KEYS_SORTED").tolist() == [4, 4, 6, 6, 6, 9]
    assert g.read_state("PERM").tolist() == [3, 5, 1, 2, 4, 0]
    cs, ce = g.read_state("CELL_START"), g.read_state("CELL_END")
    assert (cs[4], ce[4], cs[6], ce[6], cs[9], ce[9]) == (0, 2, 2, 5, 5, 6)
    assert cs[[0, 1, 2, 3, 5, 7, 8, 10, 15]].sum() == 0 and ce[[0, 1, 2, 3, 5, 7, 8, 10, 15]].sum() == 0
    g.close()


def test_whole_steps_c1_from_empty(axg):
    """C1 (32^3, 8 cones, one source, 8 particles / step): the first steps from empty, whole axg_step calls."""
    w = W.c1()
    g, o = make_pair(w, axg)
    g.step(12)
    o.step(12)
    gp = {k: g.read_state("PART_" + k) for k in ("X", "Y", "Z", "ID", "SPECIES")}
    op = {k: o.read_state("PART_" + k) for k in ("X", "Y", "Z", "ID", "SPECIES")}
    gc, oc = g.counters(), o.counters()
    assert gc == oc
    # sorted order can differ only if a key differs; with ~100 particles it does not
    assert np.array_equal(gp["ID"], op["ID"])
    # north_star's bar (1e-5 relative + 1e-6 absolute) is a SINGLE-step bar; a particle that has lived k <= 12 steps
    # carries the rounding differences of k Box-Muller draws and k fp32 additions, so the bound here is 12 x that bar
    # (multi-step agreement proper is statistical: tests/test_gpu_multistep.py)
    for k in ("X", "Y", "Z"):
        d = np.abs(gp[k].astype(np.float64) - op[k].astype(np.float64))
        assert (d <= 12 * (pu.ATOL + pu.RTOL * np.abs(op[k].astype(np.float64)))).all(), (k, d.max())
    compare_cones(g, o)
    g.close()
    o.close()


def test_crowded_cells_and_d_zero(axg):
    """D = 0 piles a source's whole emission into one cell, and a loaded state may hold any number of particles per cell
    (axg_create accepts D = 0).  Count binning ranks the members of a crowded cell as a whole (k_settle: a block-wide
    sort in shared memory up to 4 096 members; above that tile by tile, every member adding up how many entries of each
    sorted tile lie below it), not member by member: cells of 32, 33, 40, 700, 4 096, 4 097, 5 000 and 200 000 members,
    bit-exact against the oracle's std::stable_sort in both binning modes, inside a stated time bound."""
    import time
    grid = (16, 12, 10)
    rng = np.random.default_rng(77)
    sizes = {(3, 3, 3): 200_000, (9, 2, 7): 5_000, (1, 10, 1): 4_097, (12, 5, 5): 4_096, (6, 6, 2): 700, (14, 1, 8): 40,
             (0, 0, 0): 33, (15, 11, 9): 32}
    pos = [np.asarray(c, np.float64) + rng.uniform(0.0, 1.0, (m, 3)) for c, m in sizes.items()]
    pos.append(rng.uniform(0.0, 1.0, (30_000, 3)) * np.asarray(grid))           # a sparse background
    p = np.concatenate(pos, 0).astype(np.float32)
    p = np.minimum(p, np.nextafter(np.asarray(grid, np.float32), np.float32(0)))
    p = p[rng.permutation(len(p))]                                               # members arrive in arbitrary order
    n = len(p)
    sp = rng.integers(0, 2, n).astype(np.uint8)
    ids = rng.permutation(n).astype(np.uint32)
    g = pu.new_axg(axg, grid, 0.0, 50, 2.0, 0.25, 0.1, 9)
    o = axo.Oracle(grid, 0.0, 50, 2.0, 0.25, 0.1, 9)
    for s in (g, o):
        s.set_capacity(n + 4096, 16)
        s.add_source(3.5, 3.5, 3.5, 0, 1, 50)                                    # emits into the 200 000-member cell
        s.add_source(8.25, 8.5, 4.75, 1, -1, 37)
        s.place_neurons(np.array([[3.2, 3.9, 2.1], [9.5, 2.5, 7.5], [0.5, 0.5, 0.5]], np.float32))
        s.load_particles(p[:, 0].copy(), p[:, 1].copy(), p[:, 2].copy(), sp, ids, next_id=n, step=0)
    g.step_phase(axg.PHASE_DIFFUSE | axg.PHASE_BIN)                             # warm: allocations, module load
    t0 = time.perf_counter()
    g.load_particles(p[:, 0].copy(), p[:, 1].copy(), p[:, 2].copy(), sp, ids, next_id=n, step=0)
    g.step_phase(axg.PHASE_DIFFUSE | axg.PHASE_BIN)
    dt = time.perf_counter() - t0
    assert dt < 0.5, "one P1 + P2 over 2.4e5 rows with a 2e5-member cell took %.3f s" % dt
    o.step_phase(axo.PHASE_DIFFUSE | axo.PHASE_BIN)
    assert compare_presort(pre_arrays(g), pre_arrays(o), grid, 87) == 0         # sigma = 0: nothing can differ
    compare_binning(g, o)
    for ph in (axg.PHASE_SENSE, axg.PHASE_ADVANCE | axg.PHASE_COMMIT):
        g.step_phase(ph)
        o.step_phase(ph)
    compare_sense(g, o)
    compare_cones(g, o)
    t0 = time.perf_counter()
    g.step(6)                                                                    # the crowded cells keep growing
    dt = time.perf_counter() - t0
    assert dt < 1.0, "six whole steps took %.3f s" % dt
    o.step(6)
    gc, oc = g.counters(), o.counters()
    gc["emitted"] -= 87                                                          # the untimed warm-up P1 of this side
    assert gc == oc
    for f in ("PART_ID", "PART_SPECIES", "KEYS_SORTED", "PERM", "CELL_START", "CELL_END"):
        assert np.array_equal(g.read_state(f), o.read_state(f)), f
    for f in ("PART_X", "PART_Y", "PART_Z"):
        assert np.array_equal(g.read_state(f).view(np.uint32), o.read_state(f).view(np.uint32)), f
    compare_cones(g, o)
    g.close()
    o.close()


def test_device_error_word_is_reported_once_and_cleared(axg):
    """axg_enqueue_phase checks nothing (include/axg.h): the device-side capacity guard fires, axg_sync reports it as
    AXG_ECAPACITY once and clears the word; after axg_set_capacity + axg_load_particles the context works again."""
    g = pu.new_axg(axg, (8, 8, 8), 0.0, 4, 2.0, 0.25, 0.1, 1)       # D = 0: nothing moves, nothing is absorbed
    g.set_capacity(10, 64)
    g.add_source(4.5, 4.5, 4.5, 0, 1, 4)
    for _ in range(3):                                                # 4, 8, then 12 > 10 particles
        g.enqueue_phase(axg.PHASE_ALL)
    with pytest.raises(axg.AxgError) as e:
        g.sync()
    assert e.value.code == -2
    g.sync()                                                          # reported once
    assert g.counters()["n_live"] == 8                                # the third emission was dropped
    g.set_capacity(1000, 64)
    x = np.full(5, 1.5, np.float32)
    g.load_particles(x, x, x, np.zeros(5, np.uint8), np.arange(5, dtype=np.uint32), next_id=5, step=0)
    g.step(3)
    c = g.counters()
    assert (c["n_live"], c["next_id"], c["step"]) == (17, 17, 3)
    # a loaded row outside the domain has no cell: AXG_PHASE_BIN alone flags it (AXG_EINVAL) and stays in bounds
    bad = np.array([1.5, 9.5], np.float32)
    g.load_particles(bad, bad, bad, np.zeros(2, np.uint8), np.arange(2, dtype=np.uint32), next_id=2, step=0)
    with pytest.raises(axg.AxgError) as e:
        g.step_phase(axg.PHASE_BIN)
    assert e.value.code == -1
    g.load_particles(x, x, x, np.zeros(5, np.uint8), np.arange(5, dtype=np.uint32), next_id=5, step=0)
    g.step_phase(axg.PHASE_BIN)
    assert g.read_state("KEYS_SORTED").tolist() == [73] * 5
    g.close()


def test_errors_and_capacity(axg):
    g = pu.new_axg(axg, (8, 8, 8), 0.5, 4, 2.0, 0.25, 0.1, 1)
    g.set_capacity(10, 2)
    g.add_source(4, 4, 4, 0, 1, 4)
    with pytest.raises(axg.AxgError) as e:
        g.add_source(9, 4, 4, 0, 1, 4)
    assert e.value.code == -1
    with pytest.raises(axg.AxgError) as e:
        g.add_source(4, 4, 4, 0, -1, 4)       # polarity conflict within a species
    assert e.value.code == -1
    with pytest.raises(axg.AxgError) as e:
        g.step(3)                              # 12 > 10 particles
    assert e.value.code == -2
    assert g.counters()["step"] == 0           # a failing call changed nothing
    g.place_neurons(np.array([[1, 1, 1]], np.float32))
    g.step(2)
    with pytest.raises(axg.AxgError) as e:
        g.step(1)                              # particle (and polyline) capacity
    assert e.value.code == -2
    with pytest.raises(axg.AxgError) as e:
        g.place_neurons(np.array([[1, 1, 1]], np.float32))
    assert e.value.code == -3
    g.close()
    with pytest.raises(axg.AxgError):
        axg.Axg((0, 8, 8), 0.5, 4, 2.0, 0.25, 0.1, 1)
    with pytest.raises(axg.AxgError):
        axg.Axg((8, 8, 8), 0.5, 4, 9.0, 0.25, 0.1, 1)


@pytest.mark.parametrize("n", [20_000, 90_000])
def test_binning_crowded_cells(axg, n):
    """80 % of the particles inside a 1.5-cell cube (a source cell holds hundreds to thousands of members in the coarse
    pre-run): cells of several thousand members, i.e. the quadratic rank loop of count binning and long equal-key runs
    in the radix passes, against std::stable_sort, bit for bit."""
    grid = (12, 10, 9)
    g = pu.new_axg(axg, grid, 0.5, 1, 2.0, 0.25, 0.1, 3)
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
    compare_binning(g, o)
    g.close()
    o.close()


@pytest.mark.parametrize("grid", [(24, 20, 16), (6, 5, 4)])
def test_chain_heavy_absorption(axg, grid):
    """sigma = 4 cells on a 24 x 20 x 16 and on a 6 x 5 x 4 grid: a third to nearly all of the particles leave the box
    in one step, so the compaction of P1 is far from the identity (count binning: chunks with few or no survivors, most
    physical rows are holes; radix binning: long look-back sums); on the small grid the newborns are a large part of
    what is left and every cell is crowded.  (sigma stays at 4: the position tolerance of NS is absolute, and an ulp
    of a normal deviate times sigma must stay below it.)"""
    w = W.small(seed=17, grid=grid, n_cones=9)
    w.D = 8.0
    _chain(axg, w, n=30_011, seed=19, steps=2)


def test_chain_snr_steering(axg):
    """the paper's first steering rule (fixed turn pi/30 by the sign of N(SNR, 1), Eq. 5) on both
    sides; the decision is taken in fp32 with the same operations in the same order, so headings agree within NS's
    tolerance unless SNR + xi is within an ulp of zero.  Gains chosen so that turns towards and away both occur."""
    import math
    for gain in (0.0, 8.0):
        w = W.small(seed=23, n_cones=400, grid=(24, 20, 16))
        _chain(axg, w, n=60_013, seed=29, steps=3, steering=(1, gain, math.pi / 30))


@pytest.mark.parametrize("mode", [1, 2])
def test_chain_particle_sensing(axg, mode):
    """SURVEY.md §8(f) NEXT-2 (reading A-26): per-particle sensing, flat and weighted.  Counts
    and fixed-point moments bit-exact against the oracle's all-pairs loop, then P4 / P5 on them within NS's tolerance."""
    w = W.small(seed=31, n_cones=300, grid=(24, 20, 16))
    _chain(axg, w, n=60_013, seed=37, steps=3, sensing=mode)
    w = W.small(seed=32, grid=(40, 33, 21), n_cones=200, two_species=False, radius=3.0)
    _chain(axg, w, n=30_011, seed=38, steps=2, n_species=1, sensing=mode)
    import math
    w = W.small(seed=33, n_cones=100, grid=(24, 20, 16), radius=2.5)
    _chain(axg, w, n=20_001, seed=39, steps=2, sensing=mode, steering=(1, 8.0, math.pi / 30))


@pytest.mark.parametrize("mode", [1, 2])
def test_particle_sensing_on_given_state(axg, mode):
    """P3 alone on identical particles and cones: cones in the corners, on the walls, on cell faces, inside a cell that
    holds thousands of particles (the whole-warp path of k_sense_particles) and in empty space; particles exactly on
    the sphere of a cone (d^2 == R^2: detected).  Bit-exact counts and moments."""
    grid = (12, 10, 9)
    n = 40_000
    for R in (1.0, 2.0, 2.75):
        g = pu.new_axg(axg, grid, 0.5, 1, R, 0.25, 0.1, 3)
        o = axo.Oracle(grid, 0.5, 1, R, 0.25, 0.1, 3)
        x, y, z, sp, ids = W.random_particles(5, n, grid, n_species=2)
        k = int(n * 0.5)
        for a, c in zip((x, y, z), (5.0, 4.0, 3.0)):
            a[:k] = c + (a[:k] - np.floor(a[:k])) * 1.5
        rng = np.random.default_rng(77)
        nx, ny, nz = grid
        hi = [np.nextafter(np.float32(v), np.float32(0)) for v in grid]
        corners = [(a, b, c) for a in (0.0, hi[0]) for b in (0.0, hi[1]) for c in (0.0, hi[2])]
        faces = [(3.0, 4.0, 5.0), (5.0, 4.0, 3.0), (6.5, 5.5, 4.5), (5.75, 4.75, 3.75), (0.25, 5.0, 8.75)]
        rest = np.stack([rng.uniform(0, nx, 200), rng.uniform(0, ny, 200), rng.uniform(0, nz, 200)], 1)
        cones = np.concatenate([np.array(corners), np.array(faces), rest], 0).astype(np.float32)
        # particles exactly R away from the cone at (3, 4, 5) along each axis (R is dyadic: exact in fp32)
        ring = np.array([[3 + R, 4, 5], [3, 4 + R, 5], [3, 4, 5 - R], [3 - R, 4, 5]], np.float32)
        x[-4:], y[-4:], z[-4:] = ring[:, 0], ring[:, 1], ring[:, 2]
        for s in (g, o):
            s.set_capacity(n + 16, 4)
            s.add_source(6.0, 5.0, 4.0, 0, 1, 1)
            s.add_source(2.0, 2.0, 2.0, 1, -1, 1)
            s.set_sensing(mode)
            s.place_neurons(cones)
            s.load_particles(x, y, z, sp, ids, next_id=n, step=0)
        g.step_phase(axg.PHASE_BIN | axg.PHASE_SENSE)
        o.step_phase(axo.PHASE_BIN | axo.PHASE_SENSE)
        compare_binning(g, o)
        compare_sense(g, o)
        cnt = o.read_state("CONE_COUNTS").reshape(-1, 4)
        if R >= 2:
            assert cnt.sum(1).max() > 5000
        assert cnt[8].sum() >= 4          # the four particles on the sphere of cone 8 are detected
        g.close()
        o.close()


@pytest.mark.parametrize("mode,coef", [(1, 4 / 15), (2, 8 / 105)])
def test_particle_sensing_against_the_closed_form(axg, mode, coef):
    """The CUDA path against the mathematics directly (no oracle): a cloud of density rho0 (1 + k . (x - centre)) gives
    E[M] = 256 rho0 k coef pi R^5 (coef = 4/15 flat, 8/105 with the weight 1 - r^2/R^2) and E[n] = rho (4 pi / 3) R^3."""
    grid = (16, 16, 16)
    k = np.array([0.08, -0.04, 0.0])
    n = 4_000_000
    rng = np.random.default_rng(11)
    parts = []
    while sum(len(a) for a in parts) < n:
        x = rng.uniform(0, 16, (n, 3))
        parts.append(x[rng.uniform(0, 1.0 + np.abs(k).sum() * 8, n) < 1.0 + (x - 8.0) @ k])
    pts = np.concatenate(parts)[:n].astype(np.float32)
    pts = np.minimum(pts, np.nextafter(np.float32(16), np.float32(0)))
    rho0 = n / 16.0 ** 3
    c = np.array([[x, y, z] for x in (4.3, 6.6, 8.9, 11.2) for y in (4.1, 6.7, 9.0, 11.4) for z in (4.5, 6.9, 9.2, 11.0)],
                 np.float32)
    for R in (2.0, 3.0):
        g = pu.new_axg(axg, grid, 0.5, 1, R, 0.25, 0.0, 1)
        g.set_capacity(n + 16, 4)
        g.add_source(1.0, 1.0, 1.0, 0, 1, 1)
        g.set_sensing(mode)
        g.place_neurons(c)
        g.load_particles(pts[:, 0], pts[:, 1], pts[:, 2], np.zeros(n, np.uint8), np.arange(n, dtype=np.uint32),
                         next_id=n, step=0)
        g.step_phase(axg.PHASE_BIN | axg.PHASE_SENSE)
        cnt = g.read_state("CONE_COUNTS").reshape(-1, 4)[:, 0]
        M = g.read_state("CONE_MOMENT").reshape(-1, 4, 3)[:, 0, :].mean(0)
        g.close()
        expect = 256 * rho0 * k * coef * np.pi * R ** 5
        assert abs(M[0] - expect[0]) < 0.05 * abs(expect[0]), (R, M, expect)
        assert abs(M[1] - expect[1]) < 0.09 * abs(expect[1]), (R, M, expect)
        assert abs(M[2]) < 0.05 * abs(expect[0]), (R, M, expect)
        np.testing.assert_allclose(cnt, rho0 * (1 + (c.astype(np.float64) - 8.0) @ k) * 4 * np.pi / 3 * R ** 3, rtol=0.03)


@pytest.fixture(params=[1, 2], ids=["brick", "morton"])
def brick_order(request):
    pu.KEY_ORDER = request.param
    yield
    pu.KEY_ORDER = 0


@pytest.mark.parametrize("sensing", [None, 1])
def test_chain_brick_order(axg, brick_order, sensing):
    """SURVEY.md §8(f) NEXT-4 (readings A-27, A-31): the bricked cell order, and the Z-order curve, on both sides.  Grids that are whole bricks
    (24 x 20 x 16), ragged ones (40 x 33 x 21: padded key space 40 x 36 x 24; 6 x 5 x 4: one partial brick) and a 3-pass key
    (128 x 128 x 64); keys, permutation, cellStart / cellEnd (indexed by brick key), sums bit-exact as under the linear order."""
    _chain(axg, W.small(seed=7), n=50_037, seed=11, steps=3, sensing=sensing)
    _chain(axg, W.small(seed=8, two_species=False, grid=(40, 33, 21), n_cones=200), n=30_011, seed=12, steps=2,
           n_species=1, sensing=sensing)
    w = W.small(seed=17, grid=(6, 5, 4), n_cones=9)
    w.D = 8.0
    _chain(axg, w, n=30_011, seed=19, steps=2, sensing=sensing)
    w = W.small(seed=9, grid=(128, 128, 64), n_cones=300, n_sources=5, radius=3.0)
    w.D = 1.0
    w.max_particles = 1 << 18
    _chain(axg, w, n=200_003, seed=13, steps=2, sensing=sensing)


def test_brick_order_changes_only_the_order(axg):
    """30 whole steps under either cell order: the same particles (by id, bit for bit), the same cones and polylines; and
    the order can no longer be changed once the context holds anything."""
    w = W.small(seed=41, grid=(40, 33, 21), n_cones=300, n_sources=4, rate=300)
    w.max_particles = 1 << 18
    out = []
    for order in (axg.KEY_LINEAR, axg.KEY_BRICK, axg.KEY_MORTON):
        g = axg.Axg(w.grid, w.D, w.emission, w.radius, w.speed, w.noise, w.seed)
        g.set_key_order(order)
        if pu.BINNING is not None:
            g.set_binning(pu.BINNING)
        W.apply(g, w)
        x, y, z, sp, ids = W.random_particles(43, 120_007, w.grid, n_species=2)
        g.load_particles(x, y, z, sp, ids, next_id=len(ids), step=0)
        g.step(30)
        with pytest.raises(axg.AxgError):
            g.set_key_order((order + 1) % 3)
        srt = np.argsort(g.read_state("PART_ID"))
        out.append([g.read_state("PART_" + k)[srt] for k in ("ID", "X", "Y", "Z", "SPECIES")] +
                   [g.read_state(k) for k in ("CONE_POS", "CONE_HEADING", "CONE_STATE", "POLYLINE", "CONE_MOMENT")])
        ks = g.read_state("KEYS_SORTED")
        assert (np.diff(ks.astype(np.int64)) >= 0).all()
        g.close()
    for other in out[1:]:
        for a, b in zip(out[0], other):
            assert np.array_equal(a.view(np.uint8), b.view(np.uint8))
