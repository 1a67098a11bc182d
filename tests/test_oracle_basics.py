"""Pins for the oracle's building blocks: Philox, uniforms, VEGAS map, Eq. 81, RQF map, Table 1.

Every expected value here comes from the paper (cited), from the generator's published
test vectors, from mpmath at 40 digits, or from an independent brute-force definition
typed in this file -- never from the CUDA path and never from the oracle itself.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest
from scipy import integrate, optimize

import ms_inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLD, name)) as fh:
        return [ln.split() for ln in fh if ln.strip() and not ln.startswith("#")]


# ---------------------------------------------------------------- R: Philox -----------------

def test_philox_known_answers(orc):
    """Published Philox4x32-10 test vectors (SC'11), tests/golden/philox_kat.txt."""
    for row in _rows("philox_kat.txt"):
        v = [int(t, 16) for t in row]
        assert orc.philox4x32_10(v[0:4], v[4:6]) == v[6:10]


def test_philox_python_bigint_restatement(orc):
    """Brute force: the round function typed with Python big ints, random counters."""
    rng = np.random.default_rng(7)
    for _ in range(50):
        ctr = [int(t) for t in rng.integers(0, 2 ** 32, 4)]
        key = [int(t) for t in rng.integers(0, 2 ** 32, 2)]
        c, k = list(ctr), list(key)
        for _r in range(10):
            p0 = 0xD2511F53 * c[0]
            p1 = 0xCD9E8D57 * c[2]
            c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & 0xFFFFFFFF, (p0 >> 32) ^ c[3] ^ k[1], p0 & 0xFFFFFFFF]
            k = [(k[0] + 0x9E3779B9) & 0xFFFFFFFF, (k[1] + 0xBB67AE85) & 0xFFFFFFFF]
        assert orc.philox4x32_10(ctr, key) == c


def test_uniform_seed1_event0(orc):
    """SURVEY.md §8(c) R-3 / BASELINE.md §2: seed 1, event 0, stream 0."""
    assert orc.philox4x32_10([0, 0, 0, 0], [1, 0]) == [0xE3E80670, 0xE50A0EBC, 0x95F222C0, 0xB615AA27]
    assert orc.uniform(1, 0, 0, 0) == 0.8902591729757107
    assert orc.uniform(1, 0, 0, 1) == 0.5857259483801359


def test_uniform_layout_and_open_interval(orc):
    """Reading R-2/R-3 retyped with Python ints: ctr=(e_lo,e_hi,j>>1,stream), u=(2m+1)/2^53."""
    for seed, stream, ev, j in [(1, 0, 5, 0), (1, 0, 5, 3), (3, 1, (1 << 33) + 17, 0), ((7 << 32) | 9, 2, 123456789, 19)]:
        w = orc.philox4x32_10([ev & 0xFFFFFFFF, ev >> 32, j >> 1, stream], [seed & 0xFFFFFFFF, seed >> 32])
        W = (w[2] << 32 | w[3]) if j & 1 else (w[0] << 32 | w[1])
        m = W >> 12
        from fractions import Fraction
        assert Fraction(orc.uniform(seed, stream, ev, j)) == Fraction(2 * m + 1, 2 ** 53)
    r = orc.fill_uniforms(1 << 16, 6, 1)
    assert r.min() >= 2.0 ** -53 and r.max() <= 1.0 - 2.0 ** -53
    # moments of U(0,1): mean 1/2, var 1/12 (6 sigma)
    n = r.size
    assert abs(r.mean() - 0.5) < 6 * math.sqrt(1 / 12 / n)
    assert abs(r.var() - 1 / 12) < 6 * math.sqrt(1 / 180 / n)
    # independence of offsets: event_offset shifts the stream
    r2 = orc.fill_uniforms(100, 6, 1, event_offset=1000)
    assert np.array_equal(r2, r[:, 1000:1100])


# ---------------------------------------------------------------- V: VEGAS ------------------

def test_vegas_uniform_grid_is_identity(orc):
    """V-pin (i): power-of-two uniform grid => x == r bit-exact, jac == 1 exactly."""
    for d, nb in [(5, 64), (15, 64), (8, 128)]:
        r = orc.fill_uniforms(4099, d, 1)
        x, jac = orc.vegas_forward(ms_inputs.uniform_grid(d, nb), r)
        assert np.array_equal(x, r)
        assert np.all(jac == 1.0)


def test_vegas_forward_bruteforce(orc):
    """Lepage's piecewise-linear map typed with numpy searchsorted-free logic on a seeded grid."""
    d, nb = 8, 128
    edges = ms_inputs.seeded_grid(d, nb)
    r = orc.fill_uniforms(5000, d, 1)
    x, jac = orc.vegas_forward(edges, r)
    J = np.ones(r.shape[1])
    for dim in range(d):
        t = r[dim] * nb
        j = np.minimum(np.floor(t).astype(int), nb - 1)
        lo, hi = edges[dim][j], edges[dim][j + 1]
        assert np.array_equal(x[dim], lo + (t - j) * (hi - lo))
        assert np.all((x[dim] >= lo) & (x[dim] <= hi))
        J *= nb * (hi - lo)
    assert np.array_equal(jac, J)


def test_vegas_jacobian_mean_and_occupancy(orc):
    """V-pins (ii), (iv): E[jac] = 1 and each bin receives N/n_bins events."""
    d, nb, N = 8, 128, 1 << 18
    edges = ms_inputs.seeded_grid(d, nb)
    r = orc.fill_uniforms(N, d, 1)
    x, jac = orc.vegas_forward(edges, r)
    # per-dimension Jacobian: exact expectation sum_j (1/nb) nb dx_j = 1
    for dim in range(d):
        jd = nb * np.diff(edges[dim])[np.minimum((r[dim] * nb).astype(int), nb - 1)]
        assert abs(jd.mean() - 1.0) < 6 * jd.std() / math.sqrt(N)
        occ = np.histogram(x[dim], bins=edges[dim])[0]
        assert occ.sum() == N
        assert np.all(np.abs(occ - N / nb) < 6 * math.sqrt(N / nb))
    assert abs(jac.mean() - 1.0) < 6 * jac.std() / math.sqrt(N)


def test_vegas_inverse_roundtrip_and_edges(orc):
    """V-pin (iii): V^-1 o V = id; an x on an interior edge belongs to the bin on its right."""
    d, nb = 20, 128
    edges = ms_inputs.seeded_grid(d, nb)
    r = orc.fill_uniforms(20000, d, 1)
    x, jac = orc.vegas_forward(edges, r)
    r2, jinv = orc.vegas_inverse(edges, x)
    assert np.max(np.abs(r2 - r)) < 1e-11
    assert np.max(np.abs(jinv * jac - 1.0)) < 1e-13
    # inverse against numpy searchsorted (independent bin search)
    for dim in range(d):
        j = np.clip(np.searchsorted(edges[dim], x[dim], side="right") - 1, 0, nb - 1)
        ref = (j + (x[dim] - edges[dim][j]) / (edges[dim][j + 1] - edges[dim][j])) / nb
        assert np.array_equal(r2[dim], ref)
    # exactly on interior edges
    xe = np.ascontiguousarray(np.tile(edges[0][1:-1], (d, 1)))
    e1 = np.ascontiguousarray(np.tile(edges[0], (d, 1)))
    re, _ = orc.vegas_inverse(e1, xe)
    assert np.array_equal(re[0], np.arange(1, nb) / nb)


# ---------------------------------------------------------------- W: Eq. 81 -----------------

def test_phi_n_closed_form(orc):
    """Eq. 81 and BASELINE.json's equivalent form, mpmath 40 digits vs golden values."""
    mp.mp.dps = 40
    for n, E, val in _rows("volumes.txt"):
        n, E, val = int(n), mp.mpf(E), float(val)
        eq81 = E ** (2 * n - 4) / (mp.gamma(n) * mp.gamma(n - 1) * mp.pi ** (2 * n - 3) * mp.mpf(2) ** (4 * n - 5))
        s = E * E
        ns = (2 * mp.pi) ** (4 - 3 * n) * (mp.pi / 2) ** (n - 1) * s ** (n - 2) / (mp.gamma(n) * mp.gamma(n - 1))
        assert abs(eq81 / ns - 1) < mp.mpf(10) ** -35
        assert abs(float(eq81) / val - 1) < 2e-14
        assert abs(orc.phi_n(n, float(E)) / float(eq81) - 1) < 1e-14
    assert abs(orc.phi_n(2, 123.0) - 1 / (8 * math.pi)) < 1e-17


# ---------------------------------------------------------------- M: RQF --------------------

def test_table1_values(orc):
    for k, c in _rows("table1_ck.txt"):
        assert orc.ck(int(k)) == float(c)


def test_table1_refit_from_eq66():
    """Eq. 66: c_k* = argmin int_0^1 [G_RQF(y,c) - G_diet(y,k)]^2 dy, typed here with scipy."""
    for k, c_paper in _rows("table1_ck.txt"):
        k, c_paper = int(k), float(c_paper)

        def loss(c):
            f = lambda y: ((y * y + c * y * (1 - y)) / (1 + (c - 2) * y * (1 - y))
                           - ((k + 1) * y - k * y ** (1 + 1.0 / k))) ** 2
            return integrate.quad(f, 0, 1, epsabs=1e-15, epsrel=1e-13)[0]
        res = optimize.minimize_scalar(loss, bounds=(1.0, 6.0), method="bounded", options={"xatol": 1e-9})
        assert abs(res.x - c_paper) < 2e-5, (k, res.x, c_paper)


def test_rqf_forward_inverse_and_density(orc):
    """G(G^-1(x)) = x (Eq. 64/65); g = dG/dy (central difference); G(0)=0, G(1)=1, G'(0)=c, G'(1)=0."""
    xs = np.concatenate([np.linspace(1e-9, 1 - 1e-9, 2001), 10.0 ** -np.arange(3, 16), 1 - 10.0 ** -np.arange(3, 16)])
    for k in range(1, 8):
        c = orc.ck(k)
        for x in xs:
            y = orc.rqf_inverse(x, c)
            assert 0.0 <= y <= 1.0
            assert abs(orc.rqf_forward(y, c) - x) < 4e-15
        for y in np.linspace(0.01, 0.99, 99):
            h = 1e-6
            num = (orc.rqf_forward(y + h, c) - orc.rqf_forward(y - h, c)) / (2 * h)
            assert abs(num - orc.rqf_density(y, c)) < 1e-8
        assert orc.rqf_forward(0.0, c) == 0.0 and orc.rqf_forward(1.0, c) == 1.0
        assert orc.rqf_density(0.0, c) == c and orc.rqf_density(1.0, c) == 0.0


def test_rqf_inverse_vs_mpmath_literal_eq65(orc):
    """Eq. 65 typed literally at 50 digits, including the r -> 0 and r -> 1 corners (1 - y must stay accurate)."""
    mp.mp.dps = 50
    xs = list(np.linspace(0.001, 0.999, 101)) + [2.0 ** -53, 1e-12, 1 - 1e-12, 1 - 2.0 ** -53, 0.5, np.nextafter(0.5, 1)]
    for k in (1, 2, 4, 7):
        c = orc.ck(k)
        for x in xs:
            r, cm = mp.mpf(float(x)), mp.mpf(c)
            b = cm - (cm - 2) * r
            y_ref = 2 * r / (b + mp.sqrt(b * b + 4 * r * (1 - b)))
            y = orc.rqf_inverse(float(x), c)
            assert abs(mp.mpf(y) - y_ref) <= mp.mpf(2) ** -52 * 2


def test_k1_c2_coincides_with_rambo_on_diet(orc):
    """for k=1, c=2 the RQF is G_diet(y,1) = 2y - y^2."""
    for y in np.linspace(0, 1, 101):
        assert abs(orc.rqf_forward(y, 2.0) - (2 * y - y * y)) < 1e-15
        assert abs(orc.rqf_density(y, 2.0) - 2 * (1 - y)) < 1e-15


def test_exact_rambo_mass_step_solves_eq62(orc):
    """Eq. 62 residual at 50 digits: r = (k+1) v^k - k v^(k+1), v = u^2; and 1-u^2 relative accuracy."""
    mp.mp.dps = 50
    rs = list(np.linspace(1e-6, 1 - 1e-6, 301)) + [2.0 ** -53, 1e-14, 1e-9, 1 - 1e-9, 1 - 1e-14, 1 - 2.0 ** -53]
    for k in range(1, 8):
        for r in rs:
            u, t, it = orc.rambo_mass_step(float(r), k)
            assert it < 60
            rr = mp.mpf(float(r))
            v_ref = mp.findroot(lambda v: (k + 1) * v ** k - k * v ** (k + 1) - rr, mp.mpf(u) ** 2, tol=1e-45,
                                maxsteps=200) if 1e-3 < r < 1 - 1e-3 else None
            if v_ref is None:  # bisection in high precision near the ends
                lo, hi = mp.mpf(0), mp.mpf(1)
                for _ in range(200):
                    mid = (lo + hi) / 2
                    if (k + 1) * mid ** k - k * mid ** (k + 1) < rr:
                        lo = mid
                    else:
                        hi = mid
                v_ref = (lo + hi) / 2
            assert abs(mp.mpf(u) - mp.sqrt(v_ref)) <= 4e-16 * mp.sqrt(v_ref) + mp.mpf(10) ** -300
            assert abs(mp.mpf(t) - (1 - v_ref)) <= 2e-15 * (1 - v_ref)
