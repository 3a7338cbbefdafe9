"""Host-side check of the branch-free Box-Muller helpers of csrc/axg_dev.cuh: the polynomial coefficients in the header
are the ones csrc/gen_math_coeffs.py derives (Chebyshev interpolants computed in double precision), and evaluated in
float32 they meet the error bounds DESIGN.md reading A-4 states.  No GPU, no oracle: numpy against libm in double."""
import importlib.util
import os
import re

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_1405_3331_b200", "csrc")


def _gen():
    spec = importlib.util.spec_from_file_location("gen_math_coeffs", os.path.join(CSRC, "gen_math_coeffs.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def _header_coeffs(func, var):
    """The constants of `var`'s Horner chain inside device function `func`, lowest degree first."""
    src = open(os.path.join(CSRC, "axg_dev.cuh")).read()
    body = src[src.index(func):]
    body = body[:body.index("\n}\n")]
    first = re.search(r"float %s = (-?[0-9.e+-]+)f;" % var, body).group(1)
    rest = re.findall(r"%s = fmaf\(%s, \w+, (-?[0-9.e+-]+)f\);" % (var, var), body)
    return [float(c) for c in reversed([first] + rest)]


def test_header_coefficients_are_the_generated_ones():
    g = _gen()
    a, b = np.sqrt(0.5) - 1.0, np.sqrt(2.0) - 1.0
    q = (np.pi / 4) ** 2
    for func, var, want in (("axg_neg2log(", "l", g.cheb_fit(g.L, a, b, 8)),
                            ("axg_sincos_turns(", "ps", g.cheb_fit(g.S, 0.0, q, 3)),
                            ("axg_sincos_turns(", "pc", g.cheb_fit(g.C, 0.0, q, 3))):
        have = _header_coeffs(func, var)
        assert len(have) == len(want)
        np.testing.assert_allclose(have, want, rtol=2e-9, atol=0)     # printed with 10 significant digits


def test_float32_error_bounds():
    g = _gen()
    f32 = np.float32
    cl = _header_coeffs("axg_neg2log(", "l")
    k = np.arange(0, 1 << 23, 8, dtype=np.int64) + 3
    u = ((2 * k + 1).astype(np.float64) * 2.0 ** -24).astype(f32)
    ix = u.view(np.int32).astype(np.int64)
    e = (ix - 0x3f3504f3) >> 23
    f = ((ix - (e << 23)).astype(np.int32).view(f32) - f32(1.0)).astype(f32)
    z = (f * f).astype(f32)
    y = ((f * z).astype(f32) * g.horner32(cl, f)).astype(f32)
    y = (y - f32(0.5) * z).astype(f32)
    ln = ((f + y).astype(f32) + (e.astype(f32) * f32(0.693147181))).astype(f32)
    t = (f32(-2.0) * ln).astype(np.float64)
    ref = -2.0 * np.log(u.astype(np.float64))
    assert (np.abs(t - ref) / ref).max() < 2.4e-7                      # < 2 ulp of fp32
    assert np.abs(np.sqrt(t) - np.sqrt(ref)).max() < 5e-7              # rho, whose largest value is 5.77
    cs, cc = _header_coeffs("axg_sincos_turns(", "ps"), _header_coeffs("axg_sincos_turns(", "pc")
    r = np.arange(-(1 << 21), 1 << 21, 4, dtype=np.int64)
    th = (r.astype(f32) * f32(3.74507039e-07)).astype(f32)
    w = (th * th).astype(f32)
    s = (th + ((th * w).astype(f32) * g.horner32(cs, w)).astype(f32)).astype(f32)
    c = ((f32(1.0) - f32(0.5) * w).astype(f32) + ((w * w).astype(f32) * g.horner32(cc, w)).astype(f32)).astype(f32)
    ang = r.astype(np.float64) * (2.0 * np.pi * 2.0 ** -24)
    assert np.abs(s - np.sin(ang)).max() < 1.5e-7 and np.abs(c - np.cos(ang)).max() < 1.5e-7
