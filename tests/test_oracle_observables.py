"""Pins for the oracle's observables, cuts, scales and histograms (reading O-1).  The definitions are
named, not printed, in the paper, so they are pinned by what the mathematics fixes rather than by retyping them:
  * Lorentz structure: pT, phi, dphi, deta-of-massless... are invariant under boosts along z; y shifts by exactly the
    boost rapidity (so y differences are invariant); the pair mass and sqrt(s-hat) are invariant under any boost and
    rotation; for a massless momentum eta == y; theta and eta are tied by eta = -ln tan(theta/2);
  * dR^2 = deta^2 + dphi^2; dphi is symmetric, in [0, pi], and invariant under a common rotation about z, including
    across the +-pi branch cut;
  * on the generator's own events: sqrt(s-hat) = sqrt(x1 x2 s); for massless events E_T^tot = H_T = sum pT and
    H_T with masses = sum sqrt(m^2 + pT^2) from the known masses;
  * cuts: complementary windows partition the sample; histograms: all slots sum to sum w and sum w^2, brute force
    against an explicit loop, under/overflow placement.
"""
import math

import numpy as np

import ms_inputs
from oracle import observables as ob
from oracle.chain import oracle_chain
from oracle.chili import chili


def boost_z(p, rap):
    out = p.copy()
    ch, sh = math.cosh(rap), math.sinh(rap)
    for i in range(p.shape[0] // 4):
        e, pz = p[4 * i], p[4 * i + 3]
        out[4 * i], out[4 * i + 3] = e * ch + pz * sh, pz * ch + e * sh
    return out


def rotate_z(p, ang):
    out = p.copy()
    c, s = math.cos(ang), math.sin(ang)
    for i in range(p.shape[0] // 4):
        x, y = p[4 * i + 1], p[4 * i + 2]
        out[4 * i + 1], out[4 * i + 2] = c * x - s * y, s * x + c * y
    return out


def events(orc, name="cfg4rw", N=4096):
    wl = ms_inputs.WORKLOADS[name]
    return oracle_chain(orc, wl, np.arange(N))["p"], wl


def test_lorentz_structure(orc):
    p, wl = events(orc)                                              # massive 2 -> 4 (173, 173, 0, 0) at 2 TeV
    pb = boost_z(p, 0.7)
    for i in range(2, 6):
        for kind in ("PT", "PHI", "PX", "PY"):
            assert np.allclose(ob.observable(kind, pb, i), ob.observable(kind, p, i), rtol=0, atol=1e-9)
        assert np.allclose(ob.observable("Y", pb, i) - ob.observable("Y", p, i), 0.7, rtol=0, atol=1e-11)
    for (a, b) in ((2, 3), (3, 5), (4, 5)):
        assert np.allclose(ob.observable("MASS", pb, a, b), ob.observable("MASS", p, a, b), rtol=1e-11)
        assert np.allclose(ob.observable("DPHI", pb, a, b), ob.observable("DPHI", p, a, b), rtol=0, atol=1e-11)
    assert np.allclose(ob.observable("SQRT_SHAT", pb), 2000.0, rtol=1e-12)
    # massless particles (4, 5): eta == y; eta and theta: eta = -ln tan(theta/2)
    for i in (4, 5):
        assert np.allclose(ob.observable("ETA", p, i), ob.observable("Y", p, i), rtol=0, atol=1e-9)
        th = ob.observable("THETA", p, i)
        assert np.all((th >= 0) & (th <= math.pi))
        assert np.allclose(ob.observable("ETA", p, i), -np.log(np.tan(th / 2)), rtol=0, atol=1e-9)
        assert np.allclose(ob.observable("ABSETA", p, i), np.abs(ob.observable("ETA", p, i)))
    # the two tops are massive: |y| < |eta|
    assert np.all(ob.observable("ABSY", p, 2) < ob.observable("ABSETA", p, 2))
    assert np.allclose(ob.observable("PABS", p, 2) ** 2, ob.observable("E", p, 2) ** 2 - 173.0 ** 2, rtol=1e-10)


def test_pair_observables(orc):
    p, _ = events(orc)
    for (a, b) in ((2, 3), (4, 5), (2, 5)):
        dphi, deta, dr = (ob.observable(k, p, a, b) for k in ("DPHI", "DETA", "DR"))
        assert np.all((dphi >= 0) & (dphi <= math.pi)) and np.all(deta >= 0)
        assert np.allclose(dr ** 2, deta ** 2 + dphi ** 2, rtol=1e-13)
        assert np.array_equal(dphi, ob.observable("DPHI", p, b, a)) and np.array_equal(dr, ob.observable("DR", p, b, a))
        for ang in (0.3, 2.9, -3.1):                                 # rotations push pairs across the +-pi branch cut
            pr = rotate_z(p, ang)
            assert np.allclose(ob.observable("DPHI", pr, a, b), dphi, rtol=0, atol=1e-11)
            assert np.allclose(ob.observable("DR", pr, a, b), dr, rtol=0, atol=1e-10)
            assert np.allclose(ob.observable("MASS", pr, a, b), ob.observable("MASS", p, a, b), rtol=1e-12)


def test_event_level_on_generated_events(orc):
    x = orc.fill_uniforms(4096, 7, 3)
    p, w, x1x2 = chili(3, x, 100.0 ** 2)
    assert np.allclose(ob.observable("SQRT_SHAT", p), np.sqrt(x1x2[0] * x1x2[1]) * 100.0, rtol=1e-12)
    sum_pt = sum(ob.observable("PT", p, i) for i in (2, 3, 4))
    assert np.allclose(ob.observable("ET_TOT", p, n_out=3), sum_pt, rtol=1e-12)     # massless: E = |p|
    assert np.allclose(ob.observable("HT", p, n_out=3), sum_pt, rtol=0, atol=1e-5)  # m^2 = E^2 - p^2 cancels to ~1e-12 E^2
    pm, _ = events(orc)
    masses = (173.0, 173.0, 0.0, 0.0)
    ht = sum(np.sqrt(m * m + ob.observable("PT", pm, i + 2) ** 2) for i, m in enumerate(masses))
    assert np.allclose(ob.observable("HT", pm, n_out=4), ht, rtol=1e-9, atol=1e-4)
    et = ob.observable("ET_TOT", pm, n_out=4)
    assert np.all(et >= sum(ob.observable("PT", pm, i) for i in range(2, 6)) * (1 - 1e-12))


def test_cuts_and_histograms():
    rs = np.random.Generator(np.random.Philox(key=9))
    obs = rs.normal(0.0, 2.0, 20000)
    obs[:3] = [np.nan, -1.0, 1.0]
    w = rs.random(20000)
    inside, below, above = ob.cut(w, obs, -1.0, 1.0), ob.cut(w, obs, hi=np.nextafter(-1.0, -2)), ob.cut(w, obs, lo=np.nextafter(1.0, 2))
    assert inside[0] == 0.0 and inside[1] == w[1] and inside[2] == w[2]
    assert np.allclose((inside + below + above)[1:], w[1:]) and np.all((inside > 0).astype(int) + (below > 0) + (above > 0) <= 1)
    sw, sw2 = ob.histogram(obs, w, -3.0, 3.0, 12)
    ok = ~np.isnan(obs)
    assert abs(sw.sum() - w[ok].sum()) < 1e-9 and abs(sw2.sum() - (w[ok] ** 2).sum()) < 1e-9
    ref = np.zeros(14)
    for o, ww in zip(obs, w):
        if math.isnan(o):
            continue
        k = 0 if o < -3.0 else (13 if o >= 3.0 else int(math.floor((o + 3.0) * 2.0)) + 1)
        ref[k] += ww
    assert np.allclose(sw, ref, rtol=1e-12)
    assert np.allclose(sw[1:13], np.histogram(obs[ok], bins=12, range=(-3.0, 3.0), weights=w[ok])[0] - np.eye(12)[11] * w[ok][obs[ok] == 3.0].sum(), rtol=1e-12)
