"""Derives the polynomial coefficients of the branch-free fp32 Box-Muller helpers in axg_dev.cuh (axg_neg2log,
axg_sincos_turns) and checks their error against double precision.  Run:  python gen_math_coeffs.py

The polynomials are Chebyshev interpolants (near-minimax) computed here in double precision; nothing is copied from a
math library.  The check emulates the kernel's evaluation order in numpy float32 (numpy has no fused multiply-add, so
the emulation rounds twice where the kernel rounds once: the printed errors are upper estimates).

  ln(1+f)   = f - f^2/2 + f^3 * L(f)          f in [sqrt(1/2) - 1, sqrt(2) - 1],  L of degree 8
  sin(t)    = t + t^3 * S(t^2)                 t in [-pi/4, pi/4],                 S of degree 3 in t^2
  cos(t)    = 1 - t^2/2 + t^4 * C(t^2)         t in [-pi/4, pi/4],                 C of degree 3 in t^2
"""
import numpy as np
from numpy.polynomial import chebyshev as Ch
from numpy.polynomial import polynomial as P


def cheb_fit(fn, a, b, deg):
    """Power-basis coefficients (in x) of the Chebyshev interpolant of fn on [a, b]."""
    c = Ch.chebinterpolate(lambda s: fn(0.5 * (b - a) * s + 0.5 * (b + a)), deg)
    p = Ch.cheb2poly(c)                       # polynomial in s
    # substitute s = (2 x - (a + b)) / (b - a)
    lin = np.array([-(a + b) / (b - a), 2.0 / (b - a)])
    out = np.zeros(1)
    for k in range(len(p) - 1, -1, -1):
        out = P.polyadd(P.polymul(out, lin), [p[k]])
    return out


def L(f):
    f = np.asarray(f, dtype=np.float64)
    small = np.abs(f) < 1e-3
    fs = np.where(small, 0.1, f)
    exact = (np.log1p(fs) - fs + 0.5 * fs * fs) / fs ** 3
    series = 1.0 / 3 - f / 4 + f * f / 5 - f ** 3 / 6 + f ** 4 / 7
    return np.where(small, series, exact)


def S(w):   # (sin t - t) / t^3 with w = t^2
    w = np.asarray(w, dtype=np.float64)
    t = np.sqrt(np.maximum(w, 1e-300))
    small = w < 1e-4
    ts = np.where(small, 0.1, t)
    exact = (np.sin(ts) - ts) / ts ** 3
    series = -1.0 / 6 + w / 120 - w * w / 5040
    return np.where(small, series, exact)


def C(w):   # (cos t - 1 + t^2/2) / t^4
    w = np.asarray(w, dtype=np.float64)
    t = np.sqrt(np.maximum(w, 1e-300))
    small = w < 1e-3
    ts = np.where(small, 0.1, t)
    exact = (np.cos(ts) - 1.0 + 0.5 * ts * ts) / ts ** 4
    series = 1.0 / 24 - w / 720 + w * w / 40320
    return np.where(small, series, exact)


def horner32(coef, x):
    acc = np.full(x.shape, np.float32(coef[-1]), dtype=np.float32)
    for c in coef[-2::-1]:
        acc = (acc * x + np.float32(c)).astype(np.float32)
    return acc


def main():
    f32 = np.float32
    a, b = np.sqrt(0.5) - 1.0, np.sqrt(2.0) - 1.0
    cl = cheb_fit(L, a, b, 8)
    q = (np.pi / 4) ** 2
    cs = cheb_fit(S, 0.0, q, 3)
    cc = cheb_fit(C, 0.0, q, 3)
    for name, c in (("LOG", cl), ("SIN", cs), ("COS", cc)):
        print("// %s: " % name + ", ".join("%.9ef" % v for v in c))

    # ---- check -2 ln u and rho = sqrt(-2 ln u) over every 2^23 uniform of reading A-3 (strided sample of 2^21) -----
    k = np.arange(0, 1 << 23, 4, dtype=np.int64) + 1
    u = ((2 * k + 1).astype(np.float64) * 2.0 ** -24)
    u32 = u.astype(f32)
    ix = u32.view(np.int32).astype(np.int64)
    e = (ix - 0x3f3504f3) >> 23
    m = (ix - (e << 23)).astype(np.int32).view(f32)
    f = (m - f32(1.0)).astype(f32)
    z = (f * f).astype(f32)
    pl = horner32(cl, f)
    y = ((f * z).astype(f32) * pl).astype(f32)
    y = (y - f32(0.5) * z).astype(f32)
    fe = e.astype(f32)
    ln = ((f + y).astype(f32) + (fe * f32(0.693147180559945))).astype(f32)   # kernel: two-part ln 2, fused
    t = (f32(-2.0) * ln).astype(f32)
    ref_t = -2.0 * np.log(u)
    rel = np.abs(t.astype(np.float64) - ref_t) / ref_t
    rho = np.sqrt(t.astype(np.float64))
    print("-2 ln u: max rel err %.3g (fp32 eps = 6e-8); rho: max abs err %.3g" % (rel.max(), np.abs(rho - np.sqrt(ref_t)).max()))

    # ---- check sin / cos on [-pi/4, pi/4] ---------------------------------------------------------------------
    r = np.arange(-(1 << 21), 1 << 21, 2, dtype=np.int64)
    th = (r.astype(f32) * f32(2.0 * np.pi * 2.0 ** -24)).astype(f32)
    w = (th * th).astype(f32)
    s = (th + ((th * w).astype(f32) * horner32(cs, w)).astype(f32)).astype(f32)
    c = ((f32(1.0) - f32(0.5) * w).astype(f32) + ((w * w).astype(f32) * horner32(cc, w)).astype(f32)).astype(f32)
    ang = r.astype(np.float64) * (2.0 * np.pi * 2.0 ** -24)
    print("sin: max abs err %.3g   cos: max abs err %.3g" % (np.abs(s - np.sin(ang)).max(), np.abs(c - np.cos(ang)).max()))


if __name__ == "__main__":
    main()
