"""Pins for the oracle's massive phase space by REWEIGHTING (strategy (ii), Eq. 68-69 -- the one
MadSpace adopts), SURVEY.md section 8(f) NEXT-1.

What fixes it independently of the oracle's own code:
  * n = 2: every weight equals the closed-form massive two-body volume sqrt(lambda)/(8 pi s); this also settles the
    prefactor of Eq. 68 (the printed 1/8 gives 1/8 of it: reading K-4b) -- checked explicitly;
  * n = 3, 4: <w> -> the massive volume from nested two-body quadrature typed out here (scipy), the same number the
    Newton-rescale strategy (i) reproduces (4-body: BASELINE.md's 1500880.28692 GeV^4), and the two strategies agree
    with each other within their Monte Carlo errors;
  * every event: p_i^2 = m_i^2, sum p = Q, positive energies;
  * massless limit: all m = 0 reproduces orc.fastrambo bit for bit in the weights' leading digits (1e-14);
  * Eq. 69 reading K-4a: M_i - M_{i+1} >= m_i for every i (the theta functions of Eq. 53), which the printed sum
    j = 1..n would violate;
  * the exact-Rambo variant has a weight that depends only on the masses M_i (flat in the angles).
"""
import math

import numpy as np
import pytest
from scipy import integrate


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def outgoing(p, n):
    return [p[4 * (j + 2):4 * (j + 2) + 4] for j in range(n)]


def lam(a, b, c):
    return a * a + b * b + c * c - 2 * a * b - 2 * a * c - 2 * b * c


def phi2(s, a2, b2):
    return math.sqrt(max(lam(s, a2, b2), 0.0)) / (8 * math.pi * s)


def check_kinematics(p, n, W, masses, tol=5e-15):
    out = outgoing(p, n)
    inc = p[0:4] + p[4:8]
    assert np.max(np.abs(sum(out) - inc)) <= tol * W
    for j, q in enumerate(out):
        assert np.max(np.abs(mdot(q, q) - masses[j] ** 2)) / W ** 2 <= tol
        assert np.all(q[0] >= masses[j])


def test_n2_closed_form_and_prefactor(orc):
    N, W, m = 2048, 500.0, (173.0, 80.4)
    x = orc.fill_uniforms(N, 2, 1)
    p, w, nbad = orc.rambo_massive_reweight(2, x, W, m)
    assert nbad == 0
    ref = phi2(W * W, m[0] ** 2, m[1] ** 2)
    assert np.max(np.abs(w / ref - 1)) < 1e-14          # prefactor 1 (reading K-4b); 1/8 would give ref / 8
    kabs = np.sqrt(sum(p[8 + i] ** 2 for i in (1, 2, 3)))
    assert np.max(np.abs(kabs / (math.sqrt(lam(W * W, m[0] ** 2, m[1] ** 2)) / (2 * W)) - 1)) < 1e-14
    check_kinematics(p, 2, W, m)


def phi3(q2, m1, m2, m3):
    """Massive three-body volume by one quadrature over s_23."""
    f = lambda s23: phi2(q2, m1 * m1, s23) * phi2(s23, m2 * m2, m3 * m3) / (2 * math.pi)
    return integrate.quad(f, (m2 + m3) ** 2, (math.sqrt(q2) - m1) ** 2, epsabs=0, epsrel=1e-11)[0]


def test_n3_volume(orc):
    W, m = 2000.0, (173.0, 173.0, 50.0)
    ref = phi3(W * W, *m)
    assert abs(ref / 426.196008 - 1) < 1e-8               # SURVEY.md section 8c K-pins (nested quadrature)
    N = 1 << 19
    x = orc.fill_uniforms(N, 5, 7)
    p, w, nbad = orc.rambo_massive_reweight(3, x, W, m)
    assert nbad == 0
    check_kinematics(p, 3, W, m)
    err = w.std() / math.sqrt(N)
    assert abs(w.mean() - ref) < 5 * err and err / ref < 2e-3


def test_cfg4_volume_agrees_with_quadrature_and_with_strategy_i(orc):
    W, m = 2000.0, (173.0, 173.0, 0.0, 0.0)
    f4 = lambda s234: phi2(W * W, m[0] ** 2, s234) * phi3(s234, m[1], 0.0, 0.0) / (2 * math.pi)
    ref = integrate.quad(f4, m[1] ** 2, (W - m[0]) ** 2, epsabs=0, epsrel=1e-10)[0]
    assert abs(ref / 1500880.28692 - 1) < 1e-8
    N = 1 << 20
    x = orc.fill_uniforms(N, 8, 1)
    p, w, nbad = orc.rambo_massive_reweight(4, x, W, m)
    assert nbad == 0
    check_kinematics(p, 4, W, m)
    err = w.std() / math.sqrt(N)
    assert abs(w.mean() - ref) < 5 * err and err / ref < 1e-3
    # strategy (i) on the same uniforms integrates to the same volume
    p0, w0 = orc.fastrambo(4, x, W)
    _, w1, nf = orc.massive_rescale(4, W, m, p0, w0)
    assert nf == 0
    err1 = w1.std() / math.sqrt(N)
    assert abs(w.mean() - w1.mean()) < 5 * math.hypot(err, err1)
    # Eq. 53 theta functions / Eq. 69 reading K-4a: M_{i-1} - M_i >= m_{i-1}, M_i >= sum_{j>=i} m_j
    out = outgoing(p, 4)
    Q = out[3].copy()
    M = [np.sqrt(np.maximum(mdot(Q, Q), 0))]              # M_4 = m_4
    for i in (2, 1, 0):
        Q = Q + out[i]
        M.append(np.sqrt(np.maximum(mdot(Q, Q), 0)))
    M = M[::-1]                                           # M_1 .. M_4
    for i in range(3):
        assert np.all(M[i] - M[i + 1] >= m[i] * (1 - 1e-12) - 1e-9)
        assert np.all(M[i] >= sum(m[i:]) * (1 - 1e-12))


def test_massless_limit_is_fastrambo(orc):
    for n in (3, 5, 8):
        x = orc.fill_uniforms(4096, 3 * n - 4, 3)
        p0, w0 = orc.fastrambo(n, x, 1000.0)
        p1, w1, _ = orc.rambo_massive_reweight(n, x, 1000.0, (0.0,) * n)
        assert np.max(np.abs(p1 - p0)) <= 2e-15 * 1000.0 and np.max(np.abs(w1 / w0 - 1)) < 1e-13


def test_exact_variant_weight_is_flat_in_the_angles(orc):
    """With the exact Rambo u_i the massless part is flat, so the weight is a function of the mass uniforms only."""
    n, W, m = 4, 1000.0, (100.0, 50.0, 20.0, 5.0)
    x = orc.fill_uniforms(2048, 8, 5)
    x[:2] = np.array([[0.3], [0.7]])                      # same masses for every event, angles vary
    _, w, nbad = orc.rambo_massive_reweight(n, np.ascontiguousarray(x), W, m, exact=True)
    assert nbad == 0 and np.max(np.abs(w / w[0] - 1)) < 1e-13


def test_threshold_is_reported(orc):
    x = orc.fill_uniforms(64, 2, 1)
    _, w, nbad = orc.rambo_massive_reweight(2, x, 100.0, (60.0, 50.0))
    assert nbad == 64 and np.all(w == 0.0)


def _condition(p, n, masses):
    """min over the chain of K_i / K_{i-1} (massless-equivalent mass ratios) and of q_i / sqrt_s (rest-frame momenta)."""
    out = outgoing(p, n)
    msum = np.cumsum(np.asarray(masses)[::-1])[::-1]
    Q = out[n - 1].copy()
    Ks, Ms = [], []
    for i in range(n - 1, 0, -1):
        Q = Q + out[i - 1]
        M = np.sqrt(np.maximum(mdot(Q, Q), 0))
        Ms.append(M)
        Ks.append(M - msum[i - 1])
    Ks = Ks[::-1]                                          # K_1 .. K_{n-1}
    umin = np.ones(p.shape[1])
    for i in range(1, len(Ks)):
        umin = np.minimum(umin, Ks[i] / Ks[i - 1])
    return umin, Ks


@pytest.mark.parametrize("n,masses,W", [(4, (173.0, 173.0, 0.0, 0.0), 2000.0), (3, (173.0, 173.0, 50.0), 2000.0),
                                        (6, (0.0, 4.7, 0.0, 173.0, 1.0, 80.4), 1000.0), (2, (173.0, 80.4), 500.0)])
def test_massive_inverse_round_trip(orc, n, masses, W):
    """F^-1 o F = id for the massive map (the paper's own validation protocol, uses massive
    gg -> t tbar g g kinematics): median deviation at the rounding level, tail governed by the condition of the
    event (smallest K_i/K_{i-1}, i.e. invariants close to threshold -- "power-law tail ... invariants close to zero")."""
    N = 1 << 16
    x = orc.fill_uniforms(N, 3 * n - 4, 29)
    p, w, nbad = orc.rambo_massive_reweight(n, x, W, masses)
    assert nbad == 0
    x2, w2 = orc.rambo_massive_reweight_inverse(n, p, masses)
    dev = np.abs(x2 - x)
    for a in range(n - 1):
        row = n - 1 + 2 * a
        dev[row] = np.minimum(dev[row], 1 - dev[row])      # phi is periodic
    umin, Ks = _condition(p, n, masses)
    kmin = np.min(np.stack(Ks), axis=0) / W if Ks else np.ones(N)
    # errors of the stored momenta (eps * W) are divided by the smallest massless-equivalent mass K_i and, for the
    # angles, by the rest-frame momentum ~ K_i (1 - u^2)
    tol = 1e-10 * np.maximum(1.0, (1e-3 / np.minimum(umin, kmin)) ** 2)
    assert np.all(dev.max(axis=0) <= tol)
    assert np.median(dev) < 2e-15
    assert np.median(np.abs(w2 / w - 1)) < 1e-13 and np.quantile(np.abs(w2 / w - 1), 0.99) < 1e-9
