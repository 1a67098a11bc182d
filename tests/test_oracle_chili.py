"""Pins for the oracle's Chili mapping (Eq. 70-77; readings C-1..C-5).  SURVEY.md section 8(f) NEXT-4.

What fixes it other than its own code:
  * the volume: sum w / N -> int dx1 dx2 Phi_n(x1 x2 s) = Phi_n(1) s^(n-2) / (n-1)^2 (Eq. 81 integrated with
    int_0^1 dtau tau^(n-2) ln(1/tau) = 1/(n-1)^2), which fixes every factor of reading C-4 (the per-particle measure,
    the delta-function Jacobians 1/2 and 2/s, (2 pi)^(4-3n)) and the Jacobians of Eq. 73, 74, 75;
  * the pT-cut branch (Eq. 72): n = 2 with pT > pT_min has the closed form
    int dtau ln(1/tau) sqrt(1 - 4 pT_min^2/(tau s)) / (8 pi), evaluated here by quadrature;
  * massive n = 2: int dtau ln(1/tau) sqrt(lambda(tau s, m1^2, m2^2)) / (8 pi tau s) by quadrature;
  * every event: p_i^2 = m_i^2, sum p = p_a + p_b exactly as constructed (Eq. 76-77), p_a, p_b light-like along z,
    the technical cut E+- <= sqrt(s) decides w > 0, x1 x2 s = (sum p)^2;
  * Eq. 72/73 end points and monotonicity; phi is measured from the recoil direction (Eq. 75).
"""
import math

import numpy as np
import pytest
from scipy import integrate

from oracle.chili import chili


def phi_n_unit(n):
    return 1.0 / (math.gamma(n) * math.gamma(n - 1) * math.pi ** (2 * n - 3) * 2.0 ** (4 * n - 5))     # Eq. 81 at E = 1


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


@pytest.mark.parametrize("n,rs,N", [(2, 10.0, 1 << 20), (3, 10.0, 1 << 21), (4, 10.0, 1 << 21)])
def test_massless_volume(orc, n, rs, N):
    s = rs * rs
    x = orc.fill_uniforms(N, 3 * n - 2, 5)
    p, w, x1x2 = chili(n, x, s)
    ref = phi_n_unit(n) * s ** (n - 2) / (n - 1) ** 2
    err = w.std() / math.sqrt(N)
    assert abs(w.mean() - ref) < 4.5 * err and err / ref < 6e-3
    out = [p[4 * (j + 2):4 * (j + 2) + 4] for j in range(n)]
    assert np.max(np.abs(sum(out) - p[0:4] - p[4:8])) <= 4e-15 * rs
    for q in out:
        assert np.max(np.abs(mdot(q, q))) <= 4e-15 * s
    assert np.all(p[1] == 0) and np.all(p[2] == 0) and np.all(p[0] == p[3]) and np.all(p[4] == -p[7])
    inside = (x1x2[0] <= 1.0) & (x1x2[1] <= 1.0)
    assert np.array_equal(w > 0, inside)
    tot = sum(out)
    assert np.max(np.abs(mdot(tot, tot) - x1x2[0] * x1x2[1] * s)) <= 1e-13 * s


def test_pt_cut_branch_closed_form(orc):
    rs, ptmin, N = 20.0, 3.0, 1 << 21
    s = rs * rs
    x = orc.fill_uniforms(N, 4, 6)
    p, w, _ = chili(2, x, s, pt_min=(ptmin, 0.0))
    pt = np.hypot(p[9], p[10])
    assert pt.min() >= ptmin * (1 - 1e-14) and pt.max() <= rs / 2 * (1 + 1e-14)
    f = lambda tau: math.log(1 / tau) * math.sqrt(max(1 - 4 * ptmin ** 2 / (tau * s), 0.0)) / (8 * math.pi)
    ref = integrate.quad(f, 4 * ptmin ** 2 / s, 1.0, epsabs=0, epsrel=1e-10)[0]
    err = w.std() / math.sqrt(N)
    assert abs(w.mean() - ref) < 4.5 * err and err / ref < 3e-3


def test_massive_two_body_closed_form(orc):
    rs, m, N = 30.0, (5.0, 3.0), 1 << 21
    s = rs * rs
    x = orc.fill_uniforms(N, 4, 7)
    p, w, _ = chili(2, x, s, masses=m)
    lam = lambda a, b, c: a * a + b * b + c * c - 2 * a * b - 2 * a * c - 2 * b * c
    f = lambda tau: math.log(1 / tau) * math.sqrt(max(lam(tau * s, m[0] ** 2, m[1] ** 2), 0.0)) / (8 * math.pi * tau * s)
    ref = integrate.quad(f, (m[0] + m[1]) ** 2 / s, 1.0, epsabs=0, epsrel=1e-10)[0]
    err = w.std() / math.sqrt(N)
    assert abs(w.mean() - ref) < 4.5 * err and err / ref < 5e-3
    for j in range(2):
        q = p[4 * (j + 2):4 * (j + 2) + 4]
        assert np.max(np.abs(mdot(q, q) - m[j] ** 2)) <= 1e-14 * s


def test_pt_maps_end_points_and_recoil_azimuth(orc):
    s = 100.0 ** 2
    r = np.array([2.0 ** -53, 0.25, 0.5, 0.75, 1 - 2.0 ** -53])
    x = np.zeros((4, 5))
    x[0], x[1], x[2], x[3] = r, 0.5, 0.0, 0.5
    p, _, _ = chili(2, x, s, pt_min=(10.0, 0.0))                    # Eq. 72: pT^2 from pT_min^2 (r=0) to pT_max^2 (r=1)
    pt = np.hypot(p[9], p[10])
    assert abs(pt[0] - 10.0) < 1e-12 and abs(pt[-1] - 50.0) < 1e-11 and np.all(np.diff(pt) > 0)
    assert np.allclose(1 / pt ** 2, r / 50.0 ** 2 + (1 - r) / 10.0 ** 2, rtol=1e-14)
    p, _, _ = chili(2, x, s)                                        # Eq. 73 with lambda_C = 1: 0 (r=0) .. pT_max (r=1)
    pt = np.hypot(p[9], p[10])
    assert pt[0] < 1e-13 and abs(pt[-1] - 50.0) < 1e-11 and np.all(np.diff(pt) > 0)
    assert np.allclose(pt, 2 * 50.0 * r / (2 + 50.0 * (1 - r)), rtol=1e-14)
    # n = 3: the second particle's azimuth is r_phi * 2 pi measured from the recoil of the first (Eq. 75)
    x3 = orc.fill_uniforms(1000, 7, 8)
    p3, _, _ = chili(3, x3, s)
    phi1 = np.arctan2(p3[10], p3[9])
    phi2 = np.arctan2(p3[14], p3[13])
    d = np.mod(phi2 - (phi1 + np.pi) - 2 * np.pi * x3[5] + np.pi, 2 * np.pi) - np.pi
    assert np.max(np.abs(d)) < 1e-12
    assert np.max(np.abs(np.mod(phi1, 2 * np.pi) - 2 * np.pi * x3[2])) < 1e-12      # first particle: phi_rec = 0
