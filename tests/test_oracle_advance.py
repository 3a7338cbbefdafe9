"""Pins T10, T11: cone advance (O8) and segment append / arrival / exit (O9)."""
import math

import numpy as np

from oracle import axo


def _mk(noise, speed=0.25, grid=(32, 32, 32), seed=5, R=2.0):
    return axo.Oracle(grid, 0.5, 0, R, speed, noise, seed)


def test_T10_noise_free_heading_is_the_unit_vector_to_the_cluster():
    o = _mk(0.0)
    o.add_source(30.0, 30.0, 30.0, 0, 1, 1)
    o.place_neurons(np.array([[10.5, 10.5, 10.5]], np.float32), np.array([[1.0, 0, 0]], np.float32))
    # a cluster in the cell at offset (1, -1, 1) (inside the R=2 ball): G = n * (1, -1, 1)
    n = 17
    o.load_particles(np.full(n, 11.3, np.float32), np.full(n, 9.7, np.float32), np.full(n, 11.1, np.float32),
                     np.zeros(n, np.uint8), np.arange(n, dtype=np.uint32), next_id=n, step=0)
    o.step_phase(axo.PHASE_BIN | axo.PHASE_SENSE | axo.PHASE_ADVANCE)
    h = o.read_state("CONE_HEADING")
    np.testing.assert_allclose(h, np.array([1, -1, 1]) / math.sqrt(3), rtol=1e-6, atol=1e-7)
    p = o.read_state("CONE_POS")
    np.testing.assert_allclose(p, np.array([10.5, 10.5, 10.5]) + 0.25 * np.array([1, -1, 1]) / math.sqrt(3), rtol=1e-6)


def test_T10_no_particles_keeps_heading():
    o = _mk(0.0)
    o.add_source(30.0, 30.0, 30.0, 0, 1, 1)
    h0 = np.array([[0.6, 0.0, 0.8], [0.0, 1.0, 0.0]], np.float32)
    o.place_neurons(np.array([[10.5, 10.5, 10.5], [3.0, 3.0, 3.0]], np.float32), h0)
    o.step_phase(axo.PHASE_BIN | axo.PHASE_SENSE | axo.PHASE_ADVANCE | axo.PHASE_COMMIT)
    np.testing.assert_allclose(o.read_state("CONE_HEADING").reshape(-1, 3), h0, rtol=1e-6, atol=1e-7)
    # symmetric surroundings (G = 0 with particles present) behave the same (A-14)
    o.load_particles([9.5, 11.5], [10.5, 10.5], [10.5, 10.5], [0, 0], [0, 1], next_id=2, step=1)
    o.step_phase(axo.PHASE_BIN | axo.PHASE_SENSE | axo.PHASE_ADVANCE)
    assert o.read_state("CONE_COUNTS").reshape(-1, 4)[0, 0] == 2
    np.testing.assert_allclose(o.read_state("CONE_HEADING").reshape(-1, 3), h0, rtol=1e-6, atol=1e-7)


def test_T10_unit_heading_fixed_step_and_angular_noise_law():
    C = 120_000
    for noise in (0.05, 0.1):
        o = _mk(noise, speed=0.25, grid=(64, 64, 64), seed=77)
        o.add_source(60.0, 60.0, 60.0, 0, 1, 1)
        rng = np.random.default_rng(1)
        pos = rng.uniform(8, 56, (C, 3)).astype(np.float32)
        h0 = rng.normal(size=(C, 3))
        h0 /= np.linalg.norm(h0, axis=1, keepdims=True)
        o.set_capacity(16, 2)
        o.place_neurons(pos, h0.astype(np.float32))
        o.step_phase(axo.PHASE_SENSE | axo.PHASE_ADVANCE)     # empty grid: G = 0 => ghat = old heading
        h1 = o.read_state("CONE_HEADING").reshape(-1, 3).astype(np.float64)
        p1 = o.read_state("CONE_POS").reshape(-1, 3).astype(np.float64)
        assert np.abs(np.linalg.norm(h1, axis=1) - 1).max() < 1e-6
        assert np.abs(np.linalg.norm(p1 - pos, axis=1) - 0.25).max() < 1e-5   # ulp(56) = 3.8e-6 on the difference
        cosang = np.clip((h1 * (h0.astype(np.float32).astype(np.float64))).sum(1), -1, 1)
        # angle via the cross product (acos loses precision at small angles)
        s = np.linalg.norm(np.cross(h0.astype(np.float32).astype(np.float64), h1), axis=1)
        theta = np.arctan2(s, cosang)
        # tangential components ~ N(0, noise^2) each: E[theta^2] = 2 noise^2 (1 + O(noise^2)), E[theta] = noise sqrt(pi/2)
        assert abs(np.mean(theta ** 2) / (2 * noise ** 2) - 1) < 0.02
        assert abs(np.mean(theta) / (noise * math.sqrt(math.pi / 2)) - 1) < 0.02
        # isotropy about the old heading: the deflection has no preferred lab direction
        dv = h1 - h0
        assert np.abs(dv.mean(0)).max() < 5 * noise / math.sqrt(C)


def test_T11_append_lengths_exit_and_arrival():
    speed = 0.5
    o = _mk(0.0, speed=speed, grid=(16, 16, 16))
    o.add_source(8.0, 8.0, 8.0, 0, 1, 1)          # attractive: a target
    o.add_source(3.0, 3.0, 14.0, 1, -1, 1)        # repulsive: never a target
    o.set_capacity(1 << 12, 40)
    start = np.array([[8.0, 8.0, 5.2],      # heads +z into the target: arrives
                      [1.0, 1.0, 14.9],     # heads +z out of the box: exits
                      [3.0, 3.0, 12.0],     # heads +z through the repulsive source: must not "arrive"
                      [12.0, 2.0, 2.0]],    # heads +x, stays inside for a while
                     np.float32)
    head = np.array([[0, 0, 1], [0, 0, 1], [0, 0, 1], [1, 0, 0]], np.float32)
    o.place_neurons(start, head)
    states, lens = [], []
    for t in range(12):
        o.step_phase(axo.PHASE_ADVANCE | axo.PHASE_COMMIT)   # no particles binned: G = 0, straight lines
        states.append(o.read_state("CONE_STATE").copy())
        lens.append(o.read_state("POLY_LEN").copy())
    poly = o.read_state("POLYLINE").reshape(4, 41, 3)
    st = states[-1]
    assert list(st) == [1, 2, 2, 2]
    # cone 0: |z - 8| <= 1 first holds at z = 7.2 after 4 steps (5.7, 6.2, 6.7, 7.2)
    assert lens[-1][0] == 1 + 4 and abs(poly[0, 4, 2] - 7.2) < 1e-5
    # cone 1: 14.9 -> 15.4 -> 15.9 -> 16.4 (outside): the exit point is recorded, then frozen
    assert lens[-1][1] == 1 + 3 and poly[1, 3, 2] > 16.0
    # cone 2 passes through the repulsive source untouched and exits the top later
    assert lens[-1][2] == 1 + 8  # 12.0 + 8 * 0.5 = 16.0 is outside the half-open box
    # cone 3 exits through x = 16 after 8 steps
    assert lens[-1][3] == 1 + 8
    for c in range(4):
        L = lens[-1][c]
        assert np.array_equal(poly[c, 0], start[c])
        seg = np.linalg.norm(np.diff(poly[c, :L].astype(np.float64), axis=0), axis=1)
        assert np.abs(seg - speed).max() < 1e-5
        assert np.all(poly[c, L:] == 0)
        assert np.array_equal(poly[c, L - 1], o.read_state("CONE_POS").reshape(-1, 3)[c])
    # len = 1 + number of steps the cone was active at the start of
    for c in range(4):
        active_steps = sum(1 for t in range(12) if (t == 0 or states[t - 1][c] == 0))
        assert lens[-1][c] == 1 + active_steps
    cn = o.counters()
    assert (cn["active"], cn["arrived"], cn["exited"]) == (0, 1, 3)


def test_T11_capacity_is_checked_before_anything_changes():
    o = _mk(0.0)
    o.add_source(8.0, 8.0, 8.0, 0, 1, 100)
    o.set_capacity(250, 3)
    o.place_neurons(np.array([[8.0, 8.0, 2.0]], np.float32))
    o.step(2)
    before = o.counters()
    try:
        o.step(1)   # 200 + 100 > 250
        assert False
    except axo.OracleError as e:
        assert e.code == -2
    assert o.counters() == before
    try:
        o.set_capacity(1000, 3)
        o.step(2)   # poly_len 3 + 2 > 4
        assert False
    except axo.OracleError as e:
        assert e.code == -2
