"""Pin T14: per-particle sensing (section 5.3; reading A-26) of the oracle.

 (a) a worked example with hand-computed integers (boundary inclusion, fixed-point units, weights),
 (b) the special case that reduces to the per-cell rule (pinned by T9): particles and cones at cell centres,
 (c) closed forms for a planted linear density: E[M] = 256 k (4 pi / 15) R^5 (flat), 256 k (8 pi / 105) R^5 (weighted),
 (d) invariants: mirror symmetry, translation, independence of the particle order, polarity, frozen cones.
"""
import numpy as np

from oracle import axo
from paper_1405_3331_b200 import workloads as W

FLAT, WEIGHTED = 1, 2


def _oracle(grid, R, cones, pts, species=None, mode=FLAT, sources=((1.0, 1.0, 1.0, 0, 1),)):
    o = axo.Oracle(grid, 0.5, 0, R, 0.25, 0.0, 1)
    o.set_capacity(max(len(pts), 1), 4)
    for s in sources:
        o.add_source(*s, 1)
    o.set_sensing(mode)
    o.place_neurons(np.asarray(cones, np.float32))
    pts = np.asarray(pts, np.float32).reshape(-1, 3)
    sp = np.zeros(len(pts), np.uint8) if species is None else species
    o.load_particles(pts[:, 0], pts[:, 1], pts[:, 2], sp, np.arange(len(pts), dtype=np.uint32), next_id=len(pts), step=0)
    o.step_phase(axo.PHASE_BIN | axo.PHASE_SENSE)
    return o


def _nm(o):
    return o.read_state("CONE_COUNTS").reshape(-1, 4), o.read_state("CONE_MOMENT").reshape(-1, 4, 3)


def test_T14a_worked_example():
    # cone at (4.5, 4.5, 4.5), R = 2.  Offsets: (1.25, 0, 0) in; (0, -2, 0) exactly on the sphere: in (d^2 <= R^2);
    # (0, 0, 2.0078125) out; (1.5, 1.5, 0) out (d^2 = 4.5, although its cell is inside the per-cell stencil); (1, 1, 1) in.
    off = np.array([[1.25, 0, 0], [0, -2, 0], [0, 0, 2.0078125], [1.5, 1.5, 0], [1, 1, 1]])
    o = _oracle((9, 9, 9), 2.0, [[4.5, 4.5, 4.5]], off + 4.5)
    n, M = _nm(o)
    assert n[0, 0] == 3
    assert tuple(M[0, 0]) == (256 + 320, -512 + 256, 256)        # 256 * (1.25 + 1, -2 + 1, 1)
    g = o.read_state("CONE_GRADIENT")
    assert np.array_equal(g, np.array([576, -256, 256], np.float32) / np.float32(256 * 26))   # S2(R = 2) = 26
    # weights 1 - d^2 / 4: d^2 = 1.5625 -> 0.609375 -> rint(9.75) = 10; d^2 = 4 -> 0; d^2 = 3 -> 0.25 -> 4
    o = _oracle((9, 9, 9), 2.0, [[4.5, 4.5, 4.5]], off + 4.5, mode=WEIGHTED)
    n, M = _nm(o)
    assert n[0, 0] == 3
    assert tuple(M[0, 0]) == (10 * 20 + 4 * 16, 0 * -32 + 4 * 16, 4 * 16)
    # round to nearest, ties to even: 256 * 0.001953125 = 0.5 -> 0, 256 * 0.005859375 = 1.5 -> 2
    o = _oracle((9, 9, 9), 2.0, [[4.5, 4.5, 4.5]], np.array([[0.001953125, 0.005859375, -0.005859375]]) + 4.5)
    assert tuple(_nm(o)[1][0, 0]) == (0, 2, -2)


def test_T14b_reduces_to_the_per_cell_rule_at_cell_centres():
    """Particles and cones at cell centres, integer R: the Euclidean ball picks exactly the cells of the index-space
    ball N_R (|d|^2 <= R^2 on integers), so counts are equal and M(particle) = 256 * M(cell) -- the rule pinned by T9."""
    rng = np.random.default_rng(5)
    for grid, R in (((10, 8, 7), 2.0), ((9, 9, 9), 3.0)):
        n = 4000
        cells = np.stack([rng.integers(0, grid[a], n) for a in range(3)], 1)
        pts = cells + 0.5
        sp = rng.integers(0, 2, n).astype(np.uint8)
        cones = np.stack([rng.integers(0, grid[a], 40) for a in range(3)], 1) + 0.5
        src = ((1.0, 1.0, 1.0, 0, 1), (2.0, 2.0, 2.0, 1, -1))
        cell_rule = _nm(_oracle(grid, R, cones, pts, sp, mode=0, sources=src))
        part_rule = _nm(_oracle(grid, R, cones, pts, sp, mode=FLAT, sources=src))
        assert cell_rule[0].sum() > 0
        assert np.array_equal(cell_rule[0], part_rule[0])
        assert np.array_equal(256 * cell_rule[1], part_rule[1])


def _linear_density_cloud(rng, n, grid, k):
    """n points with density proportional to 1 + k . (x - centre), by rejection from the uniform density"""
    g = np.array(grid, np.float64)
    out = []
    top = 1.0 + np.abs(k) @ (g / 2)
    while sum(len(a) for a in out) < n:
        x = rng.uniform(0, 1, (n, 3)) * g
        keep = rng.uniform(0, top, n) < 1.0 + (x - g / 2) @ k
        out.append(x[keep])
    return np.concatenate(out)[:n]


def test_T14c_planted_linear_density_closed_form():
    """density rho(x) = rho0 (1 + k . (x - centre)): E[sum of offsets in the ball] = rho0 k int_ball x^2 dV
    = rho0 k (4 pi / 15) R^5; with the weight 1 - r^2/R^2 the integral is (8 pi / 105) R^5."""
    grid = (16, 16, 16)
    k = np.array([0.08, -0.04, 0.0])
    n = 4_000_000
    rng = np.random.default_rng(11)
    pts = _linear_density_cloud(rng, n, grid, k)
    rho0 = n / 16.0 ** 3
    c = np.array([[x, y, z] for x in (4.3, 6.6, 8.9, 11.2) for y in (4.1, 6.7, 9.0, 11.4) for z in (4.5, 6.9, 9.2, 11.0)])
    for R in (2.0, 3.0):
        for mode, integral in ((FLAT, 4 * np.pi / 15 * R ** 5), (WEIGHTED, 8 * np.pi / 105 * R ** 5)):
            cnt, M = _nm(_oracle(grid, R, c, pts, mode=mode))
            # the local density at cone p is rho0 (1 + k . (p - centre)); the first moment only sees rho0 k
            expect = 256 * rho0 * k * integral
            got = M[:, 0, :].mean(0)
            assert abs(got[0] - expect[0]) < 0.05 * abs(expect[0]), (R, mode, got, expect)
            assert abs(got[1] - expect[1]) < 0.09 * abs(expect[1]), (R, mode, got, expect)
            assert abs(got[2]) < 0.05 * abs(expect[0]), (R, mode, got, expect)
            vol = 4 * np.pi / 3 * R ** 3
            dens = rho0 * (1 + (c - 8.0) @ k)
            np.testing.assert_allclose(cnt[:, 0], dens * vol, rtol=0.03)


def test_T14d_invariants():
    rng = np.random.default_rng(3)
    grid = (12, 10, 9)
    x, y, z, sp, _ = W.random_particles(21, 5000, grid)
    pts = np.stack([x, y, z], 1)
    cones = np.stack([rng.uniform(2, 10, 30), rng.uniform(2, 8, 30), rng.uniform(2, 7, 30)], 1).astype(np.float32)
    src = ((1.0, 1.0, 1.0, 0, 1), (2.0, 2.0, 2.0, 1, -1))
    for mode in (FLAT, WEIGHTED):
        o = _oracle(grid, 2.5, cones, pts, sp, mode=mode, sources=src)
        n0, M0 = _nm(o)
        assert n0[:, :2].min() > 0
        # independent of the particle order (integer sums)
        p = rng.permutation(len(pts))
        n1, M1 = _nm(_oracle(grid, 2.5, cones, pts[p], sp[p], mode=mode, sources=src))
        assert np.array_equal(n0, n1) and np.array_equal(M0, M1)
        # G = M_0 - M_1 (species 1 repels)
        g = o.read_state("CONE_GRADIENT").reshape(-1, 3)
        np.testing.assert_allclose(g, (M0[:, 0] - M0[:, 1]) / (256.0 * axo.stencil_S2(2.5)), rtol=1e-6)
    # a particle on a dyadic lattice and a cone on it: translation by whole cells changes nothing
    lat = rng.integers(0, 4 * 64, (3000, 3)) / 64.0 + 3.0
    cl = rng.integers(0, 2 * 64, (10, 3)) / 64.0 + 4.0
    a = _nm(_oracle((12, 12, 12), 2.0, cl, lat, mode=FLAT))
    b = _nm(_oracle((12, 12, 12), 2.0, cl + 1.0, lat + 1.0, mode=FLAT))
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and a[0].sum() > 0
    # mirror image in y about the plane y = 6 (exact on the lattice): My flips, Mx / Mz and the counts stay
    for mode in (FLAT, WEIGHTED):
        a = _nm(_oracle((12, 12, 12), 2.0, cl, lat, mode=mode))
        b = _nm(_oracle((12, 12, 12), 2.0, cl * [1, -1, 1] + [0, 12, 0], lat * [1, -1, 1] + [0, 12, 0], mode=mode))
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1] * np.array([1, -1, 1]), b[1]) and np.abs(a[1]).sum() > 0


def test_T14d_frozen_cones_and_the_numpy_restatement():
    grid = (11, 9, 8)
    x, y, z, sp, _ = W.random_particles(33, 3000, grid)
    pts = np.stack([x, y, z], 1)
    rng = np.random.default_rng(8)
    cones = np.stack([rng.uniform(0, 11, 20), rng.uniform(0, 9, 20), rng.uniform(0, 8, 20)], 1).astype(np.float32)
    for mode in (FLAT, WEIGHTED):
        o = axo.Oracle(grid, 0.5, 0, 2.0, 0.25, 0.0, 1)
        o.add_source(1.0, 1.0, 1.0, 0, 1, 1)
        o.add_source(2.0, 2.0, 2.0, 1, -1, 1)
        o.set_sensing(mode)
        o.place_neurons(cones)
        state = np.zeros(20, np.uint8); state[3] = 1; state[7] = 2
        o.load_cones(cones, np.tile(np.array([0, 0, 1], np.float32), (20, 1)), state, np.ones(20, np.uint32))
        o.load_particles(x, y, z, sp, np.arange(3000, dtype=np.uint32), next_id=3000, step=0)
        o.step_phase(axo.PHASE_BIN | axo.PHASE_SENSE)
        n, M = _nm(o)
        assert n[3].sum() == 0 and n[7].sum() == 0 and not M[3].any() and not M[7].any()
        # fp32 restatement (numpy evaluates every operation in fp32, one rounding each)
        for c in (0, 5, 11, 19):
            d = pts.astype(np.float32) - cones[c]
            d2 = (d[:, 0] * d[:, 0] + d[:, 1] * d[:, 1]) + d[:, 2] * d[:, 2]
            inr = d2 <= np.float32(4.0)
            for s in range(2):
                m = inr & (sp == s)
                assert n[c, s] == m.sum()
                if mode == FLAT:
                    q = np.rint(d[m] * np.float32(256)).astype(np.int64).sum(0)
                else:
                    w = np.rint((np.float32(1) - d2[m] / np.float32(4)) * np.float32(16)).astype(np.int64)
                    q = (w[:, None] * np.rint(d[m] * np.float32(16)).astype(np.int64)).sum(0)
                assert tuple(M[c, s]) == tuple(q)
