"""Pins for the oracle's invariant mappings (Eq. 15-20): what Eq. 15 demands of any (G, g) pair,
checked independently of the printed formulas -- g integrates to 1 over [x_min, x_max] (quadrature), G maps 0 -> x_min,
1 -> x_max monotonically, g(G(r)) dG/dr = 1 (high-order finite differences in 50-digit arithmetic on the same G),
G^-1(G(r)) = r, the cumulative of g equals G^-1; plus the limits the text states: nu = 0 is the flat map, nu -> 1 tends
to the logarithmic map (Eq. 19), and the Breit-Wigner map puts the fraction (atan-weighted) of points below the pole."""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy import integrate

from oracle import invariant_maps as im

CASES = [("FLAT", 3.0, 50.0, 0.0, 0.0), ("POWER", 4.0, 1e4, 0.0, 0.8), ("POWER", 0.0, 1e4, -1e-3, 0.8),
         ("POWER", 10.0, 500.0, 2.0, 2.0), ("POWER", 1.0, 100.0, 0.0, 1.0), ("POWER", 0.0, 1e6, -0.5, 1.0),
         ("POWER", 5.0, 7.0, 1.0, 0.3), ("BW", 50.0 ** 2, 130.0 ** 2, 91.2 ** 2, 91.2 * 2.5), ("BW", 0.0, 400.0 ** 2, 173.0 ** 2, 173.0 * 1.4)]


@pytest.mark.parametrize("kind,x_min,x_max,m2,par", CASES)
def test_eq15_properties(kind, x_min, x_max, m2, par):
    rs = np.random.Generator(np.random.Philox(key=12))
    r = np.sort(np.concatenate((rs.random(2000), [0.0, 1.0])))
    x, g = im.forward(kind, r, x_min, x_max, m2, par)
    assert abs(x[0] - x_min) <= 1e-9 * max(abs(x_max), 1) and abs(x[-1] - x_max) <= 1e-9 * abs(x_max)
    assert np.all(np.diff(x) > 0) and np.all(g > 0)
    r2, g2 = im.inverse(kind, x, x_min, x_max, m2, par)
    assert np.max(np.abs(r2 - r)) <= 1e-9 and np.allclose(g2, g, rtol=1e-12)
    # normalisation and cumulative of g by quadrature
    gfun = lambda t: float(im.inverse(kind, np.array([t]), x_min, x_max, m2, par)[1][0])

    def integral(lo, hi):
        if kind == "POWER":                      # integrate in t = ln(x - m2): the integrand g e^t is smooth there
            f = lambda t: gfun(m2 + math.exp(t)) * math.exp(t)
            return integrate.quad(f, math.log(lo - m2), math.log(hi - m2), epsabs=0, epsrel=1e-11, limit=400)[0]
        pts = [m2] if (kind == "BW" and lo < m2 < hi) else None
        return integrate.quad(gfun, lo, hi, points=pts, epsabs=0, epsrel=1e-11, limit=400)[0]
    assert abs(integral(x_min, x_max) - 1.0) < 1e-8
    for q in (0.1, 0.5, 0.9):
        xq = float(im.forward(kind, np.array([q]), x_min, x_max, m2, par)[0][0])
        assert abs(integral(x_min, xq) - q) < 1e-8
    # g(G(r)) dG/dr = 1 with dG/dr from 50-digit central differences of the printed G
    mp.mp.dps = 50

    def G(t):
        t = mp.mpf(t)
        if kind == "FLAT":
            return x_min + (x_max - x_min) * t
        if kind == "BW":
            u1, u2 = mp.atan((mp.mpf(x_min) - m2) / par), mp.atan((mp.mpf(x_max) - m2) / par)
            return par * mp.tan(u1 + (u2 - u1) * t) + m2
        a, b = mp.mpf(x_min) - m2, mp.mpf(x_max) - m2
        if par == 1.0:
            return mp.exp(t * mp.log(b) + (1 - t) * mp.log(a)) + m2
        p = 1 - mp.mpf(par)
        return (t * b ** p + (1 - t) * a ** p) ** (1 / p) + m2
    for q in (0.05, 0.37, 0.93):
        dG = mp.diff(G, q)
        gq = float(im.forward(kind, np.array([q]), x_min, x_max, m2, par)[1][0])
        assert abs(gq * float(dG) - 1.0) < 1e-10


def test_stated_limits():
    r = np.linspace(0.0, 1.0, 101)
    xf, gf = im.forward("FLAT", r, 3.0, 50.0)
    x0, g0 = im.forward("POWER", r, 3.0, 50.0, 0.0, 0.0)                 # nu = 0 "reduces to" Eq. 20
    assert np.allclose(x0, xf, rtol=1e-14) and np.allclose(g0, gf, rtol=1e-14)
    xl, gl = im.forward("POWER", r, 2.0, 900.0, 0.5, 1.0)
    for eps in (1e-6, -1e-6):
        xn, gn = im.forward("POWER", r, 2.0, 900.0, 0.5, 1.0 + eps)      # smooth limit nu -> 1
        assert np.allclose(xn, xl, rtol=1e-4) and np.allclose(gn, gl, rtol=1e-4)
    # Breit-Wigner: fraction of points below the pole = -u1 / (u2 - u1)
    m, gam = 91.2, 2.5
    u1, u2 = math.atan((50.0 ** 2 - m * m) / (m * gam)), math.atan((130.0 ** 2 - m * m) / (m * gam))
    rr = np.random.Generator(np.random.Philox(key=13)).random(400000)
    x, _ = im.forward("BW", rr, 50.0 ** 2, 130.0 ** 2, m * m, m * gam)
    frac = np.mean(x < m * m)
    assert abs(frac - (-u1 / (u2 - u1))) < 4 * math.sqrt(0.25 / len(rr))
