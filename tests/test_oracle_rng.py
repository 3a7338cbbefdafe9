"""Pins T1, T1b, T2: the oracle's Philox, uniform mapping and Box-Muller against known answers and moments."""
import math
import os

import numpy as np

from oracle import axo


def _lines(path, kind=None):
    for ln in open(path):
        ln = ln.strip()
        if not ln or ln.startswith("#"):
            continue
        if kind is None or ln.split()[0] == kind:
            yield ln


def test_T1_philox_known_answers(golden_dir):
    n = 0
    for ln in _lines(os.path.join(golden_dir, "philox_kat.txt")):
        w = [int(v, 16) for v in ln.split()]
        out = axo.philox4x32_10(w[0:4], w[4:6])
        assert [int(v) for v in out] == w[6:10], ln
        n += 1
    assert n == 3


def test_T1_philox_round_structure_bruteforce():
    """Independent restatement with Python big ints (not the oracle's code path): 200 random counters/keys."""
    rng = np.random.default_rng(5)
    M0, M1, W0, W1, MASK = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85, 0xFFFFFFFF
    for _ in range(200):
        c = [int(v) for v in rng.integers(0, 2**32, 4)]
        k = [int(v) for v in rng.integers(0, 2**32, 2)]
        cc, kk = list(c), list(k)
        for rnd in range(10):
            p0, p1 = M0 * cc[0], M1 * cc[2]
            cc = [(p1 >> 32) ^ cc[1] ^ kk[0], p1 & MASK, (p0 >> 32) ^ cc[3] ^ kk[1], p0 & MASK]
            kk = [(kk[0] + W0) & MASK, (kk[1] + W1) & MASK]
        assert [int(v) for v in axo.philox4x32_10(c, k)] == cc


def test_T1b_worked_examples(golden_dir):
    path = os.path.join(golden_dir, "worked_examples.txt")
    n = 0
    for ln in _lines(path, "normals"):
        head, rhex, zdec = [p.split() for p in ln.split("|")]
        seed, ent, t, stream = int(head[1], 16), int(head[2]), int(head[3]), int(head[4])
        r, u, z = axo.normals(seed, ent, 1, t, stream)
        assert [int(v) for v in r[0]] == [int(v, 16) for v in rhex]
        np.testing.assert_allclose(z[0], [float(v) for v in zdec], rtol=2e-7, atol=1e-9)
        n += 1
    assert n == 4
    for ln in _lines(path, "uniforms"):
        head, udec = [p.split() for p in ln.split("|")]
        r, u, z = axo.normals(int(head[1], 16), int(head[2]), 1, int(head[3]), int(head[4]))
        np.testing.assert_allclose(u[0], [float(v) for v in udec], rtol=1e-7)
    for ln in _lines(path, "zbits"):
        head, zb = [p.split() for p in ln.split("|")]
        r, u, z = axo.normals(int(head[1], 16), int(head[2]), 1, int(head[3]), int(head[4]))
        assert [int(v) for v in z[0].view(np.uint32)] == [int(v, 16) for v in zb]


def test_T1b_particle_move_and_key(golden_dir):
    for ln in _lines(os.path.join(golden_dir, "worked_examples.txt"), "move"):
        head, pos, pos1, pos1hex, grid, key = [p.split() for p in ln.split("|")]
        seed, pid, t, D = int(head[1], 16), int(head[2]), int(head[3]), float(head[4])
        g = [int(v) for v in grid]
        o = axo.Oracle(g, D, 0, 2.0, 0.25, 0.1, seed)
        p = [np.array([float(v)], dtype=np.float32) for v in pos]
        o.load_particles(p[0], p[1], p[2], np.zeros(1, np.uint8), np.array([pid], np.uint32), next_id=100, step=t)
        o.step_phase(axo.PHASE_DIFFUSE)
        got = np.array([o.read_state("PRE_X")[0], o.read_state("PRE_Y")[0], o.read_state("PRE_Z")[0]], np.float32)
        assert [int(v) for v in got.view(np.uint32)] == [int(v, 16) for v in pos1hex]
        np.testing.assert_allclose(got, [float(v) for v in pos1], rtol=1e-7)
        assert int(o.read_state("PRE_KEY")[0]) == int(key[0])


def test_T1b_cone_advance(golden_dir):
    for ln in _lines(os.path.join(golden_dir, "worked_examples.txt"), "advance"):
        head, G, ns, pos, hd1, pos1, defl = [p.split() for p in ln.split("|")]
        seed, cone, t = int(head[1], 16), int(head[2]), int(head[3])
        G = [int(v) for v in G]
        noise, speed = float(ns[0]), float(ns[1])
        o = axo.Oracle((16, 16, 16), 0.5, 0, 2.0, speed, noise, seed)
        o.add_source(12.0, 12.0, 12.0, 0, 1, 1)
        # cone index `cone` must carry the example; pad with frozen cones before it
        xyz = np.tile(np.array([float(v) for v in pos], np.float32), (cone + 1, 1))
        o.place_neurons(xyz)
        # plant particles so that M = G exactly: one particle per unit of each component, in cells cone_cell + e_axis*sign
        ci = xyz[cone].astype(np.int32)
        pts = []
        for axis in range(3):
            for _ in range(abs(G[axis])):
                d = np.zeros(3)
                d[axis] = 1 if G[axis] > 0 else -1
                pts.append(ci + d + 0.5)
        pts = np.array(pts, np.float32)
        o.load_particles(pts[:, 0], pts[:, 1], pts[:, 2], np.zeros(len(pts), np.uint8),
                         np.arange(len(pts), dtype=np.uint32), next_id=len(pts), step=t)
        o.step_phase(axo.PHASE_BIN | axo.PHASE_SENSE)
        M = o.read_state("CONE_MOMENT").reshape(-1, 4, 3)
        assert [int(v) for v in M[cone, 0]] == G
        o.step_phase(axo.PHASE_ADVANCE)
        h = o.read_state("CONE_HEADING").reshape(-1, 3)[cone]
        p = o.read_state("CONE_POS").reshape(-1, 3)[cone]
        np.testing.assert_allclose(h, [float(v) for v in hd1], rtol=2e-6, atol=2e-7)
        np.testing.assert_allclose(p, [float(v) for v in pos1], rtol=2e-6, atol=2e-7)
        g = np.array(G, float) / np.linalg.norm(G)
        ang = math.acos(min(1.0, float(np.dot(g, h.astype(float)))))
        assert abs(ang - float(defl[0])) < 5e-5


def test_T2_uniform_and_normal_moments():
    n = 3_400_000  # blocks -> 1.02e7 normals
    r, u, z = axo.normals(12345, 0, n, 3, 0)
    assert u.min() >= 2.0**-24 and u.max() <= 1.0 - 2.0**-24
    # the mapping is exact: u * 2^24 is an odd integer
    k = (u.astype(np.float64) * 2**24)
    assert np.all(k == np.floor(k)) and np.all(k.astype(np.int64) % 2 == 1)
    assert abs(u.astype(np.float64).mean() - 0.5) < 3 * math.sqrt(1 / 12 / u.size) + 1e-7
    zz = z.astype(np.float64).ravel()
    assert np.all(np.isfinite(zz))
    N = zz.size
    assert abs(zz.mean()) < 1e-3
    assert abs(zz.var() - 1.0) < 2e-3
    kurt = np.mean(zz**4) / zz.var() ** 2 - 3.0
    assert abs(kurt) < 5e-3
    assert np.abs(zz).max() <= 5.769
    # largest value the mapping allows: sqrt(-2 ln 2^-24)
    assert np.abs(zz).max() <= math.sqrt(-2 * math.log(2.0**-24)) + 1e-6
    c = np.corrcoef(z.astype(np.float64).T)
    assert abs(c[0, 1]) < 3e-3 and abs(c[0, 2]) < 3e-3 and abs(c[1, 2]) < 3e-3
    # z0^2 + z1^2 = -2 ln u0 exactly (pairing): catches a swapped sine/cosine radius
    rho2 = -2 * np.log(u[:, 0].astype(np.float64))
    np.testing.assert_allclose(z[:, 0].astype(np.float64) ** 2 + z[:, 1].astype(np.float64) ** 2, rho2, rtol=3e-6,
                               atol=1e-9)
    # angle of (z0, z1) is 2 pi u1
    ang = np.mod(np.arctan2(z[:, 1].astype(np.float64), z[:, 0].astype(np.float64)), 2 * np.pi)
    d = np.abs(ang - 2 * np.pi * u[:, 1].astype(np.float64))
    d = np.minimum(d, 2 * np.pi - d)
    big = rho2 > 1e-3
    assert d[big].max() < 1e-4
    # streams differ, steps differ
    _, _, z_s1 = axo.normals(12345, 0, 1000, 3, 1)
    _, _, z_t4 = axo.normals(12345, 0, 1000, 4, 0)
    assert not np.array_equal(z_s1, z[:1000]) and not np.array_equal(z_t4, z[:1000])


def test_uniform_built_without_int_to_float_is_the_same_number():
    """Reading A-3: the kernel forms u as asfloat(0x3f800000 | r >> 9) - (1 - 2^-24); that must be THE value
    ((r >> 9) * 2 + 1) * 2^-24 for every 23-bit mantissa (all 2^23 of them), else both sides would draw differently."""
    m = np.arange(1 << 23, dtype=np.uint32)
    spec = ((m << np.uint32(1)) | np.uint32(1)).astype(np.float32) * np.float32(2.0 ** -24)
    built = (m | np.uint32(0x3F800000)).view(np.float32) + np.float32(-float.fromhex("0x1.fffffep-1"))
    assert built.dtype == np.float32 and np.array_equal(spec.view(np.uint32), built.view(np.uint32))
    assert spec.min() == np.float32(2.0 ** -24) and spec.max() == np.float32(1 - 2.0 ** -24)
