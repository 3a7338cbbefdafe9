"""Helpers of the GPU-vs-oracle parity tests (no arithmetic of the method: comparison and bookkeeping only)."""
import numpy as np

from oracle import axo
from paper_1405_3331_b200 import workloads as W

RTOL, ATOL = 1e-5, 1e-6   # BASELINE.json north_star: single-step fp32 positions, gradients, headings
BINNING = None            # axg.BIN_RADIX / axg.BIN_COUNT: set by the parametrised fixture of the GPU tests
KEY_ORDER = 0             # 1: both sides use the bricked cell order (include/axg.h axg_set_key_order)
# Reading A-19: a GPU position within rounding of a wall may be absorbed on one side only.  Expected rate
# with the accurate Box-Muller of both sides: ~5e-7 per particle-step; accepted: 4x that, and
# never fewer than 4 (small cases).  Every comparison appends what it saw to REPORT (printed by conftest.py at the end
# of the run): flips and the largest fraction of the position tolerance that was used.
FLIP_RATE_MAX = 2e-6
REPORT = []


def new_axg(axg_mod, *args):
    g = axg_mod.Axg(*args)
    if KEY_ORDER:
        g.set_key_order(KEY_ORDER)
    if BINNING is not None:
        g.set_binning(BINNING)
    return g


def make_pair(w, axg_mod, place=True):
    """The same workload applied to a CUDA context and an oracle context."""
    g = new_axg(axg_mod, w.grid, w.D, w.emission, w.radius, w.speed, w.noise, w.seed)
    o = axo.Oracle(w.grid, w.D, w.emission, w.radius, w.speed, w.noise, w.seed)
    if KEY_ORDER:
        o.set_key_order(KEY_ORDER)
    W.apply(g, w, place=place)
    W.apply(o, w, place=place)
    return g, o


def pre_arrays(sim):
    return {k: sim.read_state("PRE_" + k) for k in ("X", "Y", "Z", "SPECIES", "ID", "KEY")}


def part_arrays(sim):
    return {k: sim.read_state("PART_" + k) for k in ("X", "Y", "Z", "SPECIES", "ID")}


def close(a, b):
    return np.abs(a.astype(np.float64) - b.astype(np.float64)) <= ATOL + RTOL * np.abs(b.astype(np.float64))


def near_wall(x, y, z, grid, tol_scale=1.0):
    """True where a coordinate is within the comparison tolerance of a domain wall (reading A-19)."""
    out = np.zeros(x.shape, dtype=bool)
    for v, n in ((x, grid[0]), (y, grid[1]), (z, grid[2])):
        v = v.astype(np.float64)
        tol = tol_scale * (ATOL + RTOL * np.maximum(np.abs(v), 1.0))
        out |= (np.abs(v) <= tol) | (np.abs(v - n) <= tol)
    return out


def compare_presort(gp, op, grid, n_newborn, label=None):
    """P1 parity (reading A-19): ids and their order equal except for particles that one side absorbed and the other
    kept within tolerance of a wall; positions of the common ids within tolerance.  Returns the number of flips."""
    gid, oid = gp["ID"], op["ID"]
    if gid.shape == oid.shape and np.array_equal(gid, oid):
        common_g = common_o = slice(None)
        flips = 0
    else:
        only_g = np.setdiff1d(gid, oid)
        only_o = np.setdiff1d(oid, gid)
        flips = len(only_g) + len(only_o)
        assert flips <= max(4, int(FLIP_RATE_MAX * len(oid))), "too many survivor mismatches: %d of %d" % (flips, len(oid))
        mg = np.isin(gid, only_g)
        mo = np.isin(oid, only_o)
        assert near_wall(gp["X"][mg], gp["Y"][mg], gp["Z"][mg], grid).all()
        assert near_wall(op["X"][mo], op["Y"][mo], op["Z"][mo], grid).all()
        common_g, common_o = ~mg, ~mo
        assert np.array_equal(gid[common_g], oid[common_o]), "order of the common survivors differs"
    used = 0.0
    for k in ("X", "Y", "Z"):
        a, b = gp[k][common_g].astype(np.float64), op[k][common_o].astype(np.float64)
        frac = np.abs(a - b) / (ATOL + RTOL * np.abs(b))
        bad = frac > 1.0
        assert not bad.any(), "%s: %d positions out of tolerance, worst %g" % (k, bad.sum(), np.abs(a - b).max())
        used = max(used, float(frac.max()) if frac.size else 0.0)
    assert np.array_equal(gp["SPECIES"][common_g], op["SPECIES"][common_o])
    if n_newborn and flips == 0:
        # newborns sit exactly at their source on both sides: bit-equal
        for k in ("X", "Y", "Z"):
            assert np.array_equal(gp[k][-n_newborn:], op[k][-n_newborn:])
    REPORT.append("P1 %-28s n=%-10d flips=%-3d (accepted %d)  worst |dx| = %.3f of the tolerance" % (
        label or "", len(oid), flips, max(4, int(FLIP_RATE_MAX * len(oid))), used))
    return flips


def compare_binning(g, o):
    """P2 parity on identical inputs: everything is integer / a pure permutation, so bit-exact."""
    for f in ("PRE_KEY", "KEYS_SORTED", "PERM", "CELL_START", "CELL_END", "PART_ID", "PART_SPECIES"):
        a, b = g.read_state(f), o.read_state(f)
        assert a.shape == b.shape, f
        assert np.array_equal(a, b), "%s differs at %d places" % (f, int((a != b).sum()))
    for f in ("PART_X", "PART_Y", "PART_Z"):
        a, b = g.read_state(f), o.read_state(f)
        assert np.array_equal(a.view(np.uint32), b.view(np.uint32)), f


def compare_sense(g, o, active_only=False):
    """active_only: the fields hold the sums of the last P3 in which a cone was ACTIVE; an oracle that was handed a
    snapshot has no history for the frozen ones, so only the active cones are comparable."""
    gc, oc = g.read_state("CONE_COUNTS").reshape(-1, 4), o.read_state("CONE_COUNTS").reshape(-1, 4)
    gm, om = g.read_state("CONE_MOMENT").reshape(-1, 12), o.read_state("CONE_MOMENT").reshape(-1, 12)
    gg, og = g.read_state("CONE_GRADIENT").reshape(-1, 3), o.read_state("CONE_GRADIENT").reshape(-1, 3)
    if active_only:
        act = o.read_state("CONE_STATE") == 0
        assert np.array_equal(act, g.read_state("CONE_STATE") == 0)
        gc, oc, gm, om, gg, og = gc[act], oc[act], gm[act], om[act], gg[act], og[act]
    assert np.array_equal(gc, oc), "per-cone counts differ"
    assert np.array_equal(gm, om), "per-cone moments differ"
    assert close(gg, og).all()


def compare_cones(g, o):
    assert np.array_equal(g.read_state("CONE_STATE"), o.read_state("CONE_STATE"))
    assert np.array_equal(g.read_state("POLY_LEN"), o.read_state("POLY_LEN"))
    for f in ("CONE_POS", "CONE_HEADING", "POLYLINE"):
        a, b = g.read_state(f), o.read_state(f)
        assert a.shape == b.shape, f
        bad = ~close(a, b)
        assert not bad.any(), "%s: %d out of tolerance, worst %g" % (f, bad.sum(), np.abs(a - b).max())


def load_same_particles(g, o, seed, n, grid, n_species=2, step=3):
    x, y, z, sp, ids = W.random_particles(seed, n, grid, n_species=n_species)
    g.load_particles(x, y, z, sp, ids, next_id=n, step=step)
    o.load_particles(x, y, z, sp, ids, next_id=n, step=step)
    return x, y, z, sp, ids


def feed_gpu_presort_to_oracle(g, o, step):
    """NS: 'binning checked on identical post-diffusion positions' -- the oracle bins the GPU's own P1 output."""
    gp = pre_arrays(g)
    c = g.counters()
    o.load_particles(gp["X"], gp["Y"], gp["Z"], gp["SPECIES"], gp["ID"], next_id=c["next_id"], step=step)
    o.step_phase(axo.PHASE_BIN)
    return gp
