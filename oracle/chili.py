"""oracle.chili -- TEST INFRASTRUCTURE: the Chili phase-space mapping (Eq. 70-77) in plain numpy fp64,
step by step in the paper's order.  SURVEY.md section 8(f) NEXT-4 (mapping only; observables and cuts on arbitrary
observables are out of scope).

Readings where the paper is silent (C-1..C-5):
  C-1 uniforms per event, 3n-2 of them: for i = 1..n-1 the triple (r_pT, r_y, r_phi) at rows 3(i-1)..3(i-1)+2,
      then r_y of the last particle at row 3n-3.
  C-2 Eq. 72 is used for a particle with a lower cut pT_min > 0, Eq. 73 otherwise with lambda_C = m (massive) or 1 GeV
      (massless) "as default"; pT_max = sqrt(s_lab)/2 (Eq. 71).
  C-3 the last particle's rapidity is sampled uniformly in |y_n| <= y_max(m_T,n) of Eq. 74 -- "the kinematic range
      implied by the already generated subsystem" is not spelled out; any range is correct as long as the weight carries
      its length, and the technical cut E+- <= sqrt(s_lab) removes what is unphysical.
  C-4 weight: the paper prints only the densities g of the pT maps.  From Eq. 70 with the delta functions integrated out
      (d^3p/2E = dpT^2 dy dphi/4 per generated particle; the last particle's d^2pT is eaten by delta^2 leaving dy_n/2;
      int dx1 dx2 delta(E) delta(pz) = 2/s_lab):
        w = (2 pi)^(4-3n) * prod_{i<n} [ (dpT^2/dr)_i * 2 y_max,i * 2 pi / 4 ] * [ 2 y_max,n / 2 ] * [ 2 / s_lab ],
      i.e. the density of  dPhi_n dx1 dx2  (no flux factor, no PDFs); 0 outside the technical cut or when Eq. 74 has
      no solution (s_lab < 4 m_T^2).
  C-5 phi_rec of the first particle is 0; afterwards the azimuth of -(sum of the transverse momenta generated so far).
"""
from __future__ import annotations

import numpy as np


def chili(n, x, s_lab, masses=None, pt_min=None, y_cut=None):
    """x: [3n-2][N] uniforms.  Returns (p [4(n+2)][N], w [N], x1x2 [2][N]).  Row layout as everywhere:
    particles 0,1 incoming (Eq. 77), 2..n+1 outgoing; component order (E, px, py, pz)."""
    x = np.asarray(x, dtype=np.float64)
    N = x.shape[1]
    assert x.shape[0] == 3 * n - 2
    m = np.zeros(n) if masses is None else np.asarray(masses, dtype=np.float64)
    ptmin = np.zeros(n) if pt_min is None else np.asarray(pt_min, dtype=np.float64)
    ycut = np.zeros(n) if y_cut is None else np.asarray(y_cut, dtype=np.float64)
    rs = np.sqrt(s_lab)
    pt_max = rs / 2.0                                                      # Eq. 71
    p = np.zeros((4 * (n + 2), N))
    w = np.full(N, (2.0 * np.pi) ** (4 - 3 * n) * 2.0 / s_lab)
    ok = np.ones(N, dtype=bool)
    sum_x, sum_y = np.zeros(N), np.zeros(N)
    e_plus, e_minus = np.zeros(N), np.zeros(N)

    def y_max_of(mt2, i):
        a = s_lab / (4.0 * mt2)
        good = a >= 1.0
        a = np.where(good, a, 1.0)
        ym = np.log(np.sqrt(a) + np.sqrt(a - 1.0))                         # Eq. 74
        if ycut[i] > 0.0:
            ym = np.minimum(ym, ycut[i])
        return ym, good

    for i in range(n - 1):
        r_pt, r_y, r_phi = x[3 * i], x[3 * i + 1], x[3 * i + 2]
        if ptmin[i] > 0.0:                                                 # Eq. 72
            pt2 = 1.0 / (r_pt / pt_max ** 2 + (1.0 - r_pt) / ptmin[i] ** 2)
            dpt2_dr = pt2 * pt2 * (1.0 / ptmin[i] ** 2 - 1.0 / pt_max ** 2)
            pt = np.sqrt(pt2)
        else:                                                              # Eq. 73
            lam = m[i] if m[i] > 0.0 else 1.0
            den = 2.0 * lam + pt_max * (1.0 - r_pt)
            pt = 2.0 * lam * pt_max * r_pt / den
            dpt_dr = 2.0 * lam * pt_max * (2.0 * lam + pt_max) / den ** 2
            pt2 = pt * pt
            dpt2_dr = 2.0 * pt * dpt_dr
        mt2 = pt2 + m[i] ** 2
        ym, good = y_max_of(mt2, i)
        ok &= good
        y = ym * (2.0 * r_y - 1.0)                                         # Eq. 75
        phi_rec = np.arctan2(-sum_y, -sum_x) if i > 0 else np.zeros(N)
        phi = 2.0 * np.pi * r_phi + phi_rec                                # Eq. 75
        mt = np.sqrt(mt2)
        e, px, py, pz = mt * np.cosh(y), pt * np.cos(phi), pt * np.sin(phi), mt * np.sinh(y)
        p[4 * (i + 2):4 * (i + 2) + 4] = (e, px, py, pz)
        sum_x += px
        sum_y += py
        e_plus += e + pz
        e_minus += e - pz
        w *= dpt2_dr * (2.0 * ym) * (2.0 * np.pi) / 4.0
    # last particle: Eq. 76 and its rapidity (reading C-3)
    i = n - 1
    px, py = -sum_x, -sum_y
    mt2 = px * px + py * py + m[i] ** 2
    ym, good = y_max_of(mt2, i)
    ok &= good
    y = ym * (2.0 * x[3 * n - 3] - 1.0)
    mt = np.sqrt(mt2)
    e, pz = mt * np.cosh(y), mt * np.sinh(y)
    p[4 * (i + 2):4 * (i + 2) + 4] = (e, px, py, pz)
    e_plus += e + pz
    e_minus += e - pz
    w *= (2.0 * ym) / 2.0
    # Eq. 77 and the technical cut
    p[0], p[3] = e_plus / 2.0, e_plus / 2.0
    p[4], p[7] = e_minus / 2.0, -e_minus / 2.0
    ok &= (e_plus <= rs) & (e_minus <= rs)
    w = np.where(ok, w, 0.0)
    return p, w, np.stack((e_plus / rs, e_minus / rs))
