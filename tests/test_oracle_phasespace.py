"""Pins for the oracle's phase-space maps: FastRambo, exact Rambo, inverse, massive rescale,
Bjorken-x sampling + boost, toy integrand, unweighting, and the literal __float128 evaluator.

Expected values: closed forms of the paper (Eq. 81, Eq. 63 flat weight, PAPER.md:506 n=3 flatness),
textbook closed forms (two-body phase space, Beta(2,n-2) energy spectrum of flat massless phase
space), invariants (momentum conservation, on-shell conditions), and brute force typed here.
"""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy import integrate

import ms_inputs


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def outgoing(p, n):
    return [p[4 * (j + 2):4 * (j + 2) + 4] for j in range(n)]


def check_kinematics(p, n, sqrt_s, masses=None, tol=4e-15):
    out = outgoing(p, n)
    tot = sum(out)
    inc = p[0:4] + p[4:8]
    assert np.max(np.abs(tot - inc)) <= tol * np.max(sqrt_s)
    for j, q in enumerate(out):
        m2 = 0.0 if masses is None else masses[j] ** 2
        # absolute error of a boosted component is eps * sqrt_s, so p^2 is off by ~eps * s (not eps * E^2)
        assert np.max(np.abs(mdot(q, q) - m2) / np.max(sqrt_s) ** 2) <= tol
        assert np.all(q[0] > 0)


# ------------------------------------------------------------ n = 2, 3: brute force / flatness

def test_n2_two_body(orc):
    """M-4: n=2 has no mass dims; isotropic back-to-back decay, weight = Phi_2 = 1/(8 pi) (Eq. 81)."""
    x = orc.fill_uniforms(4096, 2, 1)
    p, w = orc.fastrambo(2, x, 500.0)
    assert np.allclose(w, 1 / (8 * math.pi), rtol=1e-15, atol=0)
    p1, p2 = outgoing(p, 2)
    assert np.max(np.abs(p1[1:] + p2[1:])) == 0.0
    assert np.allclose(p1[0], 250.0, rtol=1e-15) and np.allclose(p2[0], 250.0, rtol=1e-15)
    # Eq. 25 typed here: cos theta = 2 x0 - 1, phi = 2 pi x1
    cth, phi = 2 * x[0] - 1, 2 * math.pi * x[1]
    sth = np.sqrt(1 - cth ** 2)
    assert np.max(np.abs(p1[3] - 250 * cth)) < 1e-12
    assert np.max(np.abs(p1[1] - 250 * sth * np.cos(phi))) < 1e-11
    assert np.max(np.abs(p1[2] - 250 * sth * np.sin(phi))) < 1e-11
    pe, we = orc.rambo_massless(2, x, 500.0)
    assert np.array_equal(pe, p) and np.array_equal(we, w)


def test_cfg1_n3_weights_are_the_volume(orc):
    """cfg 1 / PAPER.md:506: k=1, c=2 => FastRambo n=3 is exactly flat: every weight = Phi_3(1000)."""
    wl = ms_inputs.WORKLOADS["cfg1"]
    r = orc.fill_uniforms(wl.N, wl.d, ms_inputs.SEED_EVENTS)
    x, jac = orc.vegas_forward(wl.grid(), r)
    p, w = orc.fastrambo(3, x, wl.sqrt_s)
    w = w * jac
    assert np.max(np.abs(w / 125.982556379686 - 1)) < 3e-14
    check_kinematics(p, 3, 1000.0)
    # n=3 brute force: first decay in the CM frame, |p_1| = sqrt_s (1-u^2)/2, u^2 = 1 - sqrt(1-r) (Eq. 62, k=1)
    v = 1 - np.sqrt(1 - x[0])
    assert np.max(np.abs(p[8] - 500.0 * (1 - v))) < 1e-10
    m23 = np.sqrt(mdot(p[12:16] + p[16:20], p[12:16] + p[16:20]))
    assert np.max(np.abs(m23 - 1000.0 * np.sqrt(v))) < 1e-9
    # flat Dalitz plot: x_i = 2E_i/sqrt_s in the triangle, uniform => E[x_1] = 2/3, var = 1/18
    x1 = 2 * p[8] / 1000.0
    assert abs(x1.mean() - 2 / 3) < 6 * math.sqrt(1 / 18 / wl.N)


# ------------------------------------------------------------ volumes by Monte Carlo (Eq. 81)

@pytest.mark.parametrize("n,sqrt_s,N", [(4, 1000.0, 1 << 20), (5, 700.0, 1 << 19), (8, 3000.0, 1 << 19)])
def test_fastrambo_volume_and_invariants(orc, n, sqrt_s, N):
    """<w> -> Phi_n (Eq. 81; paper's own check PAPER.md:724-738), conservation, p^2 = 0,
    weighted Beta(2, n-2) energy fractions."""
    x = orc.fill_uniforms(N, 3 * n - 4, 1)
    p, w = orc.fastrambo(n, x, sqrt_s)
    phi = orc.phi_n(n, sqrt_s)
    err = w.std() / math.sqrt(N)
    assert abs(w.mean() - phi) < 5 * err
    assert err / phi < 2e-3
    check_kinematics(p, n, sqrt_s)
    for j in range(n):
        xe = 2 * p[4 * (j + 2)] / sqrt_s
        mean = np.sum(w * xe) / np.sum(w)
        var = np.sum(w * (xe - 2 / n) ** 2) / np.sum(w)
        assert abs(mean - 2 / n) < 4e-3
        assert abs(var / (2 * (n - 2) / (n * n * (n + 1))) - 1) < 3e-2


@pytest.mark.parametrize("n", [3, 4, 5, 6, 9])
def test_exact_rambo_flat_weight_and_beta(orc, n):
    """Eq. 63: RamboOnDiet weight is constant = Phi_n; energies ~ Beta(2, n-2) unweighted;
    pair-invariant mean of flat massless phase space E[s_ij] = s * 2/(n(n-1))."""
    N, sqrt_s = 1 << 17, 91.1876
    x = orc.fill_uniforms(N, 3 * n - 4, 1)
    p, w = orc.rambo_massless(n, x, sqrt_s)
    assert np.max(np.abs(w / orc.phi_n(n, sqrt_s) - 1)) < 1e-14
    check_kinematics(p, n, sqrt_s)
    var_ref = 2 * (n - 2) / (n * n * (n + 1))
    for j in range(n):
        xe = 2 * p[4 * (j + 2)] / sqrt_s
        assert abs(xe.mean() - 2 / n) < 6 * math.sqrt(var_ref / N) + 1e-12
        if n > 3:
            assert abs(xe.var() / var_ref - 1) < 0.03
    out = outgoing(p, n)
    s01 = mdot(out[0] + out[1], out[0] + out[1])
    s_last = mdot(out[n - 2] + out[n - 1], out[n - 2] + out[n - 1])
    ref = sqrt_s ** 2 * 2 / (n * (n - 1))
    assert abs(s01.mean() / ref - 1) < 0.02 and abs(s_last.mean() / ref - 1) < 0.02


def test_fastrambo_weight_range_fig3(orc):
    """Fig. 3 right: w_n/Phi_n is O(1) and not flat for n >= 4; SURVEY §8c M-2 ranges."""
    x = orc.fill_uniforms(1 << 18, 8, 1)
    _, w = orc.fastrambo(4, x, 1000.0)
    wn = w / orc.phi_n(4, 1000.0)
    assert 0.74 < wn.min() < 0.76 and 1.09 < wn.max() < 1.12


# ------------------------------------------------------------ literal quad evaluator

@pytest.mark.parametrize("n,exact", [(3, False), (4, False), (8, False), (5, True), (4, True)])
def test_fp64_forms_agree_with_literal_float128(orc, n, exact):
    """The printed equations (Eq. 25, 54-55, 60, 62/65, 67, 81) evaluated literally in __float128
    (ms_oracle_lit.c) vs the well-conditioned fp64 forms of ms_oracle.c."""
    N, sqrt_s = 3000, 1000.0
    x = orc.fill_uniforms(N, 3 * n - 4, 1)
    # adversarial corners for the mass dims
    x[0, :8] = [2.0 ** -53, 1e-12, 1e-6, 0.5, np.nextafter(0.5, 1), 1 - 1e-6, 1 - 1e-12, 1 - 2.0 ** -53]
    pl, wl = orc.lit_rambo(n, x, sqrt_s, exact=exact)
    p, w = (orc.rambo_massless if exact else orc.fastrambo)(n, x, sqrt_s)
    assert np.max(np.abs(p - pl)) < 2e-14 * sqrt_s
    assert np.max(np.abs(w / wl - 1)) < 2e-14


# ------------------------------------------------------------ inverse

@pytest.mark.parametrize("n", [3, 4, 8])
def test_fastrambo_inverse_roundtrip(orc, n):
    """F-6 / PAPER.md:740: F^-1 o F = id up to the condition of the last pair (reading F-7)."""
    N, sqrt_s = 1 << 16, 3000.0
    x = orc.fill_uniforms(N, 3 * n - 4, 1)
    p, w = orc.fastrambo(n, x, sqrt_s)
    x2, w2 = orc.fastrambo_inverse(n, p)
    dev = np.abs(x2 - x)
    # phi is periodic: r_phi ~ 0 and ~ 1 are the same point
    for a in range(n - 1):
        row = n - 1 + 2 * a
        dev[row] = np.minimum(dev[row], 1 - dev[row])
    # u_min per event from the true masses
    out = outgoing(p, n)
    Q = out[n - 1].copy()
    umin = np.ones(N)
    M = []                                   # M_{n-1}, ..., M_1 with Q_i = sum_{j>=i} p_j
    for i in range(n - 1, 0, -1):
        Q = Q + out[i - 1]
        M.append(np.sqrt(np.maximum(mdot(Q, Q), 0)))
    M = M[::-1]                              # M_1 .. M_{n-1}
    for i in range(1, len(M)):
        umin = np.minimum(umin, M[i] / M[i - 1])
    tol = 1e-10 * np.maximum(1.0, (1e-3 / umin) ** 2)
    assert np.all(dev.max(axis=0) <= tol)
    assert np.median(dev) < 1e-15
    assert np.max(np.abs(w2 / w - 1)) < 1e-9


# ------------------------------------------------------------ massive rescale (cfg 4)

def lam(a, b, c):
    return a * a + b * b + c * c - 2 * a * b - 2 * a * c - 2 * b * c


def test_massive_n2_closed_form_per_event(orc):
    """K-pin: n=2: w = Phi_2(massive) = sqrt(lambda(s,m1^2,m2^2))/(8 pi s) for every event; |k| = sqrt(lambda)/(2 sqrt_s)."""
    N, W, m = 2048, 500.0, (173.0, 80.4)
    x = orc.fill_uniforms(N, 2, 1)
    p, w = orc.fastrambo(2, x, W)
    k, wk, nf = orc.massive_rescale(2, W, m, p, w)
    assert nf == 0
    ref = math.sqrt(lam(W * W, m[0] ** 2, m[1] ** 2)) / (8 * math.pi * W * W)
    assert np.max(np.abs(wk / ref - 1)) < 1e-13
    kabs = np.sqrt(k[9] ** 2 + k[10] ** 2 + k[11] ** 2)
    assert np.max(np.abs(kabs / (math.sqrt(lam(W * W, m[0] ** 2, m[1] ** 2)) / (2 * W)) - 1)) < 1e-13
    check_kinematics(k, 2, W, m, tol=2e-14)


def phi3_massless_m(s):  # Eq. 81, n=3
    return s / (256 * math.pi ** 3)


def test_massive_cfg4_volume_and_onshell(orc):
    """cfg 4: p^2 = m^2, sum k = Q, F(xi) <= 1e-14 W; <w> -> Phi_4(2000; 173,173,0,0).
    The reference volume is recomputed here by nested quadrature
    Phi_4 = int ds_234/(2 pi) Phi_2(s; m1, sqrt(s_234)) Phi_3(s_234; m2, 0, 0),
    Phi_3(q2; m,0,0) = int ds_34/(2 pi) Phi_2(q2; m, sqrt(s_34)) Phi_2(s_34;0,0), Phi_2 = sqrt(lambda)/(8 pi s)."""
    W, m = 2000.0, (173.0, 173.0, 0.0, 0.0)

    def phi2(s, a2, b2):
        return math.sqrt(max(lam(s, a2, b2), 0.0)) / (8 * math.pi * s)

    def phi3_m00(q2, mm):
        f = lambda s34: phi2(q2, mm * mm, s34) * phi2(s34, 0, 0) / (2 * math.pi)
        return integrate.quad(f, 0, (math.sqrt(q2) - mm) ** 2, epsabs=0, epsrel=1e-11)[0]

    f4 = lambda s234: phi2(W * W, m[0] ** 2, s234) * phi3_m00(s234, m[1]) / (2 * math.pi)
    ref = integrate.quad(f4, m[1] ** 2, (W - m[0]) ** 2, epsabs=0, epsrel=1e-10)[0]
    assert abs(ref / 1500880.28692 - 1) < 1e-8
    N = 1 << 20
    x = orc.fill_uniforms(N, 8, 1)
    p, w = orc.fastrambo(4, x, W)
    k, wk, nf = orc.massive_rescale(4, W, m, p, w)
    assert nf == 0
    check_kinematics(k, 4, W, m, tol=1.2e-14)   # Newton stop: |F| <= 1e-14 W (+ rounding of the sum)
    assert np.max(np.abs(sum(k[4 * (j + 2)] for j in range(4)) - W)) <= 1.2e-14 * W
    err = wk.std() / math.sqrt(N)
    assert abs(wk.mean() - ref) < 5 * err and err / ref < 5e-4
    # massless limit: masses 0 => xi = 1, w_m = 1
    k0, w0, _ = orc.massive_rescale(4, W, (0, 0, 0, 0), p, w)
    assert np.max(np.abs(k0 - p)) <= 1e-12 and np.max(np.abs(w0 / w - 1)) < 1e-14
    # literal quad (bisection) evaluator
    kl, wl = orc.lit_massive_rescale(4, W, m, p[:, :2000].copy(), w[:2000].copy())
    assert np.max(np.abs(kl - k[:, :2000])) < 1e-13 * W
    assert np.max(np.abs(wl / wk[:2000] - 1)) < 1e-13


# ------------------------------------------------------------ Bjorken-x sampling + boost (cfg 3)

def test_pdf_x_sampling_closed_forms(orc):
    """Eq. 19 (nu=1, m^2=0), Eq. 22-23: tau in [tau_min,1] with density 1/(tau ln(1/tau_min)); rapidity uniform;
    x1 x2 = tau; E[J_x] = int dx1 dx2 theta(x1 x2 > tau_min) = 1 - tau_min + tau_min ln tau_min."""
    wl = ms_inputs.WORKLOADS["cfg3"]
    N, tmin, s_had = 1 << 18, wl.tau_min, wl.sqrt_s ** 2
    r = orc.fill_uniforms(N, 2, 1)
    x1x2, rs, jac = orc.pdf_x_sample(s_had, tmin, r)
    tau = x1x2[0] * x1x2[1]
    assert np.max(np.abs(tau / tmin ** (1 - r[0]) - 1)) < 1e-13
    assert np.max(np.abs(rs / np.sqrt(tau * s_had) - 1)) < 1e-14
    assert tau.min() >= tmin * (1 - 1e-14) and tau.max() <= 1.0 and x1x2.max() <= 1.0
    # ln tau uniform on [ln tau_min, 0]
    lt = np.log(tau) / math.log(tmin)
    assert abs(lt.mean() - 0.5) < 6 * math.sqrt(1 / 12 / N)
    # rapidity y = 0.5 ln(x1/x2) uniform on +- 0.5 ln(1/tau): 2y/ln(1/tau) ~ U(-1,1), var 1/3
    yy = np.log(x1x2[0] / x1x2[1]) / np.log(1 / tau)
    assert abs(yy.mean()) < 6 * math.sqrt(1 / 3 / N) and abs(yy.var() - 1 / 3) < 5e-3
    area = 1 - tmin + tmin * math.log(tmin)
    assert abs(jac.mean() - area) < 5 * jac.std() / math.sqrt(N)
    xl, rl, jl = orc.lit_pdf_x_sample(s_had, tmin, r[:, :4000].copy())
    assert np.max(np.abs(xl / x1x2[:, :4000] - 1)) < 1e-14
    assert np.max(np.abs(jl / jac[:4000] - 1)) < 1e-14 and np.max(np.abs(rl / rs[:4000] - 1)) < 1e-14


def test_cfg3_pipeline_closed_form_integral(orc):
    """X-pin: sum w / N -> I = Phi_5(1) s_had^3 [(1-tmin^4)/16 + tmin^4 ln(tmin)/4];
    lab-frame conservation; incoming momenta x_{1,2} sqrt(s_had)/2 (1,0,0,+-1); massless after the boost."""
    wl = ms_inputs.WORKLOADS["cfg3"]
    n, N, s_had, tmin = wl.n, 1 << 19, wl.sqrt_s ** 2, wl.tau_min
    r = orc.fill_uniforms(N, wl.d, 1)
    x, jv = orc.vegas_forward(wl.grid(), r)
    assert np.all(jv == 1.0)
    x1x2, rs, jx = orc.pdf_x_sample(s_had, tmin, np.ascontiguousarray(x[0:2]))
    p, w = orc.rambo_massless(n, np.ascontiguousarray(x[2:2 + 3 * n - 4]), rs)
    assert np.max(np.abs(w / (orc.phi_n(n, 1.0) * rs ** (2 * n - 4)) - 1)) < 1e-13
    plab = orc.pdf_boost(n, s_had, x1x2, p)
    wt = w * jx * jv
    a = n - 1
    I = orc.phi_n(5, 1.0) * s_had ** 3 * ((1 - tmin ** a) / a ** 2 + tmin ** a * math.log(tmin) / a)
    assert abs(I / 2.77492935789908e13 - 1) < 1e-12
    assert abs(wt.mean() - I) < 5 * wt.std() / math.sqrt(N)
    assert wt.std() / math.sqrt(N) / I < 5e-3
    Eb = wl.sqrt_s / 2
    assert np.array_equal(plab[0], x1x2[0] * Eb) and np.array_equal(plab[3], x1x2[0] * Eb)
    assert np.array_equal(plab[4], x1x2[1] * Eb) and np.array_equal(plab[7], -x1x2[1] * Eb)
    tot = sum(outgoing(plab, n))
    assert np.max(np.abs(tot - plab[0:4] - plab[4:8])) < 4e-15 * wl.sqrt_s
    Elab = plab[0] + plab[4]                      # boosted components carry eps * (total lab energy)
    for q in outgoing(plab, n):
        assert np.max(np.abs(mdot(q, q)) / Elab ** 2) < 4e-15
    # boost = textbook Lorentz boost with beta = (x1-x2)/(x1+x2)
    beta = (x1x2[0] - x1x2[1]) / (x1x2[0] + x1x2[1])
    gam = 1 / np.sqrt(1 - beta ** 2)
    q, ql = outgoing(p, n)[2], outgoing(plab, n)[2]
    assert np.max(np.abs(ql[0] - gam * (q[0] + beta * q[3])) / ql[0]) < 1e-12
    assert np.array_equal(ql[1], q[1]) and np.array_equal(ql[2], q[2])


# ------------------------------------------------------------ toy integrand (not from the paper)

def test_toy_integrand_bruteforce(orc):
    """Reading T: f = prod_{i} 1/(s_{i,i+1} + 100), s_ij = (p_i+p_j)^2 over the open chain; typed here with the
    plain Minkowski square (massless momenta => equal up to the off-shellness of fp64 momenta)."""
    for n in (2, 3, 4, 8):
        x = orc.fill_uniforms(20000, 3 * n - 4, 1)
        p, _ = orc.fastrambo(n, x, 1000.0)
        f = orc.toy_integrand(n, p, ms_inputs.TOY_REG)
        out = outgoing(p, n)
        ref = np.ones(p.shape[1])
        for i in range(n - 1):
            ref /= mdot(out[i] + out[i + 1], out[i] + out[i + 1]) + 100.0
        assert np.max(np.abs(f / ref - 1)) < 1e-9
        if n == 2:
            assert np.allclose(f, 1 / (1000.0 ** 2 + 100.0), rtol=1e-14)
    # rotation invariance: swap x <-> y components of all momenta
    p2 = p.copy()
    for j in range(n + 2):
        p2[4 * j + 1], p2[4 * j + 2] = p[4 * j + 2].copy(), p[4 * j + 1].copy()
    assert np.max(np.abs(orc.toy_integrand(n, p2) / f - 1)) < 1e-14


def test_toy_cross_section_three_body_dalitz(orc):
    """Absolute normalisation of the weighted toy integrand at n = 3, against a number the oracle has no part in:
    for massless particles s_ij = 2 p_i.p_j, and the three-body phase space in Dalitz variables is
    dPhi_3 = ds_12 ds_23 / (128 pi^3 s) on the triangle s_12 + s_23 <= s (PDG kinematics; its area s^2/2 reproduces
    Eq. 81's Phi_3 = s / (256 pi^3)), so
        int dPhi_3 f = 1/(128 pi^3 s) int_0^s dx ln((s - x + a)/a) / (x + a),     f = 1/((s_12+a)(s_23+a)),
    a one-dimensional quadrature typed out here.  <w f> from FastRambo and from the exact Rambo chain must both hit it."""
    W = 1000.0
    s = W * W
    assert abs(orc.phi_n(3, W) / (s / (256 * math.pi ** 3)) - 1) < 1e-14
    N = 1 << 22
    x = orc.fill_uniforms(N, 5, 17)
    # a = (250 GeV)^2: smooth integrand, per-mille Monte Carlo error -- a wrong factor 2, pi or pair cannot hide;
    # a = TOY_REG = (10 GeV)^2, the benchmark's regulator: peaked (f spans 10^8), the same check at its 5 % error
    for a, max_rel_err in ((62500.0, 1.5e-3), (ms_inputs.TOY_REG, 8e-2)):
        inner = lambda t: math.log((s - t + a) / a) / (t + a)
        ref = integrate.quad(inner, 0.0, s, epsabs=0, epsrel=1e-12, points=[10 * a, min(1000 * a, 0.5 * s)], limit=400)[0]
        ref /= 128 * math.pi ** 3 * s
        for fn in (orc.fastrambo, orc.rambo_massless):
            p, w = fn(3, x, W)
            wf = w * orc.toy_integrand(3, p, a)
            err = wf.std() / math.sqrt(N)
            assert err / ref < max_rel_err, (a, err / ref)
            assert abs(wf.mean() - ref) < 5 * err, (a, wf.mean(), ref, err)


# ------------------------------------------------------------ unweighting

def test_unweight_bruteforce_and_sum_identity(orc):
    """Reading U: accept <=> u w_max < w, stable order, w_out = max(1, w/w_max);
    E[sum w_out] = sum w / w_max."""
    N = 1 << 17
    x = orc.fill_uniforms(N, 8, 1)
    p, w = orc.fastrambo(4, x, 1000.0)
    w = w * orc.toy_integrand(4, p)
    w_max = orc.wmax(w[:4096])
    assert w_max == w[:4096].max()
    idx, wout, n_acc = orc.unweight(w, w_max, ms_inputs.SEED_UNWEIGHT, ms_inputs.STREAM_UNWEIGHT)
    u = orc.fill_uniforms(N, 1, ms_inputs.SEED_UNWEIGHT, stream=ms_inputs.STREAM_UNWEIGHT)[0]
    ref_idx = [e for e in range(N) if u[e] * w_max < w[e]]
    assert n_acc == len(ref_idx) and list(idx) == ref_idx
    assert np.array_equal(wout, np.maximum(1.0, w[idx] / w_max))
    assert np.any(wout > 1.0)                      # overweights are not a corner case (SURVEY U)
    expect = w.sum() / w_max
    pacc = np.minimum(1.0, w / w_max)
    sigma = math.sqrt(np.sum(pacc * (1 - pacc)))
    assert abs(wout.sum() - expect) < 6 * sigma + 1e-9
    # cap: first `cap` accepted are written, the true count is still returned
    idx2, wout2, n2 = orc.unweight(w, w_max, ms_inputs.SEED_UNWEIGHT, ms_inputs.STREAM_UNWEIGHT, cap=5)
    assert n2 == n_acc and list(idx2) == ref_idx[:5]
    # degenerate: w_max tiny => all accepted; w = 0 => none
    assert orc.unweight(w, 1e-300, 3)[2] == N
    assert orc.unweight(np.zeros(100), 1.0, 3)[2] == 0
