"""Pin T9: sensing (O7).  Grid form == brute-force all-pairs form, exact integers; a planted linear density returns
its gradient exactly; stencil sizes."""
import itertools

import numpy as np

from oracle import axo
from paper_1405_3331_b200 import workloads as W


def _stencil(r2):
    R = int(np.floor(np.sqrt(r2)))
    return [d for d in itertools.product(range(-R, R + 1), repeat=3) if d[0] ** 2 + d[1] ** 2 + d[2] ** 2 <= r2]


def test_T9_stencil_sizes_and_S2():
    # |N_R| = 7 / 33 / 123 (81 at floor(R^2)=6: 1+6+12+8+6+24+24), S2 = 2 / 26 / 236 for R = 1 / 2 / 3 (A-11, A-12): lattice-point counts of a ball
    for R, ncell, s2 in ((1.0, 7, 2), (2.0, 33, 26), (3.0, 123, 236), (2.5, 81, None)):
        st = _stencil(int(np.floor(R * R)))
        assert len(st) == ncell
        if s2 is not None:
            assert sum(d[0] ** 2 for d in st) == s2 == axo.stencil_S2(R)
        assert tuple(np.sum(st, 0)) == (0, 0, 0)


def test_T9_grid_equals_brute_force():
    for seed, grid, R in ((1, (12, 9, 7), 2.0), (2, (6, 6, 6), 3.0), (3, (16, 4, 5), 1.0), (4, (9, 9, 9), 2.5)):
        rng = np.random.default_rng(seed)
        n = 2000
        x, y, z, sp, ids = W.random_particles(seed, n, grid)
        o = axo.Oracle(grid, 0.5, 0, R, 0.25, 0.1, seed)
        o.add_source(grid[0] / 2, grid[1] / 2, grid[2] / 2, 0, 1, 1)
        o.add_source(1.5, 1.5, 1.5, 1, -1, 1)
        # cones: all 8 corners, wall cells, the source cell, the rest random
        nx, ny, nz = grid
        corners = [(a, b, c) for a in (0.5, nx - 0.5) for b in (0.5, ny - 0.5) for c in (0.5, nz - 0.5)]
        rest = np.stack([rng.uniform(0, nx, 48), rng.uniform(0, ny, 48), rng.uniform(0, nz, 48)], 1)
        cones = np.concatenate([np.array(corners), [[nx / 2, ny / 2, nz / 2]], rest], 0).astype(np.float32)
        o.place_neurons(cones)
        o.load_particles(x, y, z, sp, ids, next_id=n, step=0)
        o.step_phase(axo.PHASE_BIN | axo.PHASE_SENSE)
        cnt = o.read_state("CONE_COUNTS").reshape(-1, 4)
        mom = o.read_state("CONE_MOMENT").reshape(-1, 4, 3)
        bc, bm = o.sense_brute()
        assert np.array_equal(cnt, bc) and np.array_equal(mom, bm)
        assert cnt.sum() > 0 and np.abs(mom).sum() > 0
        # and against a numpy restatement of the definition (neither of the oracle's two loops)
        cell = np.stack([np.floor(x), np.floor(y), np.floor(z)], 1).astype(np.int64)
        r2 = int(np.floor(R * R))
        for c in range(0, len(cones), 7):
            d = cell - np.floor(cones[c]).astype(np.int64)
            inr = (d ** 2).sum(1) <= r2
            for s in range(2):
                m = inr & (sp == s)
                assert cnt[c, s] == m.sum()
                assert tuple(mom[c, s]) == tuple(d[m].sum(0))
        # gradient = sum_s polarity_s M_s / S2
        G = mom[:, 0, :] - mom[:, 1, :]
        g = o.read_state("CONE_GRADIENT").reshape(-1, 3)
        np.testing.assert_allclose(g, G / float(axo.stencil_S2(R)), rtol=1e-6)


def test_T9_planted_linear_density_returns_its_gradient():
    """k_x particles more per cell per unit x (and k_y, k_z): count(cell) = c0 + k.cell  =>  M = k * S2 exactly."""
    grid = (16, 16, 16)
    kx, ky, kz, c0 = 2, -1, 3, 50
    pts = []
    for cx, cy, cz in itertools.product(range(16), repeat=3):
        cnt = c0 + kx * (cx - 8) + ky * (cy - 8) + kz * (cz - 8)
        assert cnt >= 0
        pts += [(cx + 0.5, cy + 0.25, cz + 0.75)] * cnt
    pts = np.array(pts, np.float32)
    rng = np.random.default_rng(0)
    pts = pts[rng.permutation(len(pts))]
    for R in (2.0, 3.0):
        o = axo.Oracle(grid, 0.5, 0, R, 0.25, 0.1, 1)
        o.set_capacity(len(pts), 4)
        o.add_source(1.0, 1.0, 1.0, 0, 1, 1)
        o.place_neurons(np.array([[8.5, 8.5, 8.5], [5.2, 9.9, 6.1]], np.float32))
        o.load_particles(pts[:, 0], pts[:, 1], pts[:, 2], np.zeros(len(pts), np.uint8),
                         np.arange(len(pts), dtype=np.uint32), next_id=len(pts), step=0)
        o.step_phase(axo.PHASE_BIN | axo.PHASE_SENSE)
        g = o.read_state("CONE_GRADIENT").reshape(-1, 3)
        assert np.array_equal(g, np.array([[kx, ky, kz]] * 2, np.float32))
        S2 = axo.stencil_S2(R)
        M = o.read_state("CONE_MOMENT").reshape(-1, 4, 3)
        assert np.array_equal(M[:, 0, :], np.array([[kx * S2, ky * S2, kz * S2]] * 2))


def test_T9_repulsive_species_flips_sign_and_frozen_cones_are_skipped():
    o = axo.Oracle((8, 8, 8), 0.5, 0, 2.0, 0.25, 0.0, 1)
    o.add_source(1.0, 1.0, 1.0, 0, -1, 1)       # species 0 repels
    o.place_neurons(np.array([[4.5, 4.5, 4.5], [4.5, 4.5, 4.5]], np.float32))
    o.load_cones(np.array([[4.5, 4.5, 4.5]] * 2, np.float32), np.array([[0, 0, 1.0]] * 2, np.float32),
                 np.array([0, 2], np.uint8), np.array([1, 1], np.uint32))
    o.load_particles([5.5], [4.5], [4.5], [0], [0], next_id=1, step=0)
    o.step_phase(axo.PHASE_BIN | axo.PHASE_SENSE)
    g = o.read_state("CONE_GRADIENT").reshape(-1, 3)
    assert g[0, 0] < 0 and g[0, 1] == 0 and g[0, 2] == 0
    assert np.all(g[1] == 0) and o.read_state("CONE_COUNTS").reshape(-1, 4)[1].sum() == 0
