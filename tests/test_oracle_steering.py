"""Pins T13: the paper's first steering rule (Eq. 5; reading A-25) in the oracle.

  SNR = gain * mu * sqrt(gamma / (1 + gamma)^3) * sin(phi),  draw s ~ N(SNR, 1),  turn by delta = pi/30 towards the
  gradient direction if s > 0, away from it otherwise.

What fixes it without an implementation to compare against: the geometry of a rotation (angle exactly delta, in the
plane of heading and gradient, unit length, fixed step), the Gaussian law of the decision (fraction of turns towards
the gradient = Phi(SNR), which exposes every factor of Eq. 5 separately), and the degenerate cases of P:282-286.
"""
import math

import numpy as np

from oracle import axo

DELTA = math.pi / 30
N_R2 = 33      # cells of the radius-2 stencil
S2_R2 = 26     # sum of dx^2 over it


def _phi(x):
    return 0.5 * (1.0 + math.erf(x / math.sqrt(2.0)))


def _cones(C, seed, gain, n_all, G, heading=None):
    """C cones in an empty 64^3 box with planted sensing sums: n_all particles in range, integer moment G."""
    o = axo.Oracle((64, 64, 64), 0.5, 0, 2.0, 0.25, 0.1, seed)
    o.add_source(60.0, 60.0, 60.0, 0, 1, 1)
    rng = np.random.default_rng(seed)
    pos = rng.uniform(8, 56, (C, 3)).astype(np.float32)
    if heading is None:
        h0 = rng.normal(size=(C, 3))
        h0 /= np.linalg.norm(h0, axis=1, keepdims=True)
    else:
        h0 = np.tile(np.asarray(heading, dtype=np.float64), (C, 1))
    o.set_capacity(16, 2)
    o.place_neurons(pos, h0.astype(np.float32))
    o.set_steering(1, gain, DELTA)
    counts = np.zeros((C, 4), np.int64)
    counts[:, 0] = n_all
    moment = np.zeros((C, 4, 3), np.int64)
    moment[:, 0, :] = G
    o.load_sense(counts, moment)
    o.step_phase(axo.PHASE_ADVANCE)
    h1 = o.read_state("CONE_HEADING").reshape(-1, 3).astype(np.float64)
    p1 = o.read_state("CONE_POS").reshape(-1, 3).astype(np.float64)
    return pos.astype(np.float64), h0.astype(np.float32).astype(np.float64), h1, p1


def _expected_snr(gain, n_all, G, sinphi):
    gamma = n_all / N_R2
    mu = (np.linalg.norm(G) / S2_R2) / gamma
    return gain * mu * math.sqrt(gamma / (1 + gamma) ** 3) * sinphi


def test_T13_turn_is_a_rotation_by_delta_in_the_plane_of_heading_and_gradient():
    G = np.array([3, -1, 2])
    pos, h0, h1, p1 = _cones(50_000, 3, 1.0, 40, G)
    ghat = G / np.linalg.norm(G)
    assert np.abs(np.linalg.norm(h1, axis=1) - 1).max() < 1e-6
    assert np.abs(np.linalg.norm(p1 - pos, axis=1) - 0.25).max() < 1e-5
    ang = np.arctan2(np.linalg.norm(np.cross(h0, h1), axis=1), (h0 * h1).sum(1))
    assert np.abs(ang - DELTA).max() < 2e-6                       # every cone turns, by exactly delta
    normal = np.cross(h0, ghat)
    normal /= np.linalg.norm(normal, axis=1, keepdims=True)
    assert np.abs((h1 * normal).sum(1)).max() < 2e-6              # ... inside the plane spanned by h and g
    # towards the gradient <=> the angle to the gradient shrinks by delta; away <=> grows by delta
    a0 = np.arccos(np.clip(h0 @ ghat, -1, 1))
    a1 = np.arccos(np.clip(h1 @ ghat, -1, 1))
    mid = (a0 > 2 * DELTA) & (a0 < math.pi - 2 * DELTA)
    d = (a1 - a0)[mid]
    assert np.abs(np.abs(d) - DELTA).max() < 1e-5
    assert 0.3 < (d < 0).mean() < 0.99                            # both outcomes occur


def test_T13_decision_follows_the_gaussian_law_of_eq5():
    """Heading orthogonal to the gradient (sin phi = 1): P(turn towards) = Phi(SNR); every factor of Eq. 5 is varied."""
    C = 40_000
    h = (0.0, 0.0, 1.0)
    cases = [  # gain, particles in range, integer moment (orthogonal to the heading)
        (0.0, 40, (5, 0, 0)),          # no signal: a fair coin
        (10.0, 40, (5, 0, 0)),
        (20.0, 40, (5, 0, 0)),         # gain doubles the SNR
        (10.0, 40, (3, 4, 0)),         # |G| = 5 again, another direction: same SNR
        (10.0, 40, (10, 0, 0)),        # mu doubles
        (10.0, 160, (20, 0, 0)),       # same mu, four times the background: sqrt(gamma / (1 + gamma)^3) at work
    ]
    for gain, n_all, G in cases:
        G = np.array(G)
        _, h0, h1, _ = _cones(C, 11, gain, n_all, G, heading=h)
        ghat = G / np.linalg.norm(G)
        towards = ((h1 - h0) @ ghat) > 0
        snr = _expected_snr(gain, n_all, G, 1.0)
        p = _phi(snr)
        se = math.sqrt(p * (1 - p) / C)
        assert abs(towards.mean() - p) < 4 * se + 1e-4, (gain, n_all, tuple(G), towards.mean(), p)
    # the cases were chosen to be informative: not saturated, and different from one another
    snrs = [_expected_snr(g, n, np.array(G), 1.0) for g, n, G in cases]
    assert 0.2 < snrs[1] < 1.0 and abs(snrs[2] - 2 * snrs[1]) < 1e-12 and abs(snrs[3] - snrs[1]) < 1e-12
    assert abs(snrs[4] - 2 * snrs[1]) < 1e-12 and abs(snrs[5] - snrs[1]) > 0.05


def test_T13_sin_phi_scales_the_snr():
    """Heading at 30 degrees to the gradient: the SNR is half of the orthogonal case."""
    C = 40_000
    G = np.array([5, 0, 0])
    h = (math.cos(math.pi / 6), 0.0, math.sin(math.pi / 6))
    _, h0, h1, _ = _cones(C, 13, 20.0, 40, G, heading=h)
    towards = ((h1 - h0) @ (G / 5.0)) > 0
    p = _phi(_expected_snr(20.0, 40, G, 0.5))
    assert abs(towards.mean() - p) < 4 * math.sqrt(p * (1 - p) / C) + 1e-4
    assert abs(p - _phi(_expected_snr(20.0, 40, G, 1.0))) > 0.05   # distinguishable from sin phi = 1


def test_T13_degenerate_cases_keep_the_direction():
    # nothing in range, G = 0 with particles present, heading parallel / antiparallel to the gradient
    for n_all, G, h in ((0, (0, 0, 0), (0.6, 0.0, 0.8)), (12, (0, 0, 0), (0.6, 0.0, 0.8)),
                        (12, (0, 0, 7), (0.0, 0.0, 1.0)), (12, (0, 0, 7), (0.0, 0.0, -1.0))):
        pos, h0, h1, p1 = _cones(64, 17, 5.0, n_all, np.array(G), heading=h)
        np.testing.assert_allclose(h1, h0, rtol=0, atol=1e-7)
        np.testing.assert_allclose(p1, pos + 0.25 * h0, rtol=0, atol=1e-5)


def test_T13_default_mode_is_the_vector_rule():
    """axg_set_steering(0, ...) / never calling it: the north_star rule (noise-free: heading = gradient direction)."""
    o = axo.Oracle((32, 32, 32), 0.5, 0, 2.0, 0.25, 0.0, 5)
    o.add_source(30.0, 30.0, 30.0, 0, 1, 1)
    o.place_neurons(np.array([[10.5, 10.5, 10.5]], np.float32), np.array([[1.0, 0, 0]], np.float32))
    o.set_steering(1, 1.0, DELTA)
    o.set_steering(0, 1.0, DELTA)
    counts = np.zeros((1, 4), np.int64); counts[0, 0] = 9
    moment = np.zeros((1, 4, 3), np.int64); moment[0, 0] = (2, -2, 1)
    o.load_sense(counts, moment)
    o.step_phase(axo.PHASE_ADVANCE)
    np.testing.assert_allclose(o.read_state("CONE_HEADING"), np.array([2, -2, 1]) / 3.0, rtol=1e-6, atol=1e-7)
