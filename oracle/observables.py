"""oracle.observables -- TEST INFRASTRUCTURE: the kinematic observables, cuts, scales and weighted histograms of
PAPER.md:613-648 (Sec. 3.2.4-3.2.6, Eq. 78-80) in plain numpy fp64.  SURVEY.md section 8(f) NEXT-4 ("the observable
kernels it needs").

The paper lists the observables by name only; the definitions are the textbook collider ones (reading O-1):
  single momentum (E, px, py, pz):  pT = sqrt(px^2 + py^2);  |p| = sqrt(px^2 + py^2 + pz^2);  phi = atan2(py, px) in
      (-pi, pi];  theta = atan2(pT, pz) in [0, pi];  y = 1/2 ln((E + pz)/(E - pz));  eta = 1/2 ln((|p| + pz)/(|p| - pz));
  pair:  dphi = |phi_a - phi_b| folded into [0, pi];  deta = |eta_a - eta_b|;  dR = sqrt(deta^2 + dphi^2);
      m = sqrt(max((p_a + p_b)^2, 0));
  event:  sqrt(s-hat) = sqrt((p_in,a + p_in,b)^2);  E_T^tot = sum_i E_i pT_i / |p_i| (Eq. 79);
      H_T = sum_i sqrt(m_i^2 + pT_i^2) (Eq. 80) with m_i^2 = max(E_i^2 - |p_i|^2, 0), over the outgoing particles.
A cut keeps an event if lo <= observable <= hi, else sets its weight to 0 ("minimum and/or maximum values").
Histograms: fixed uniform binning over [lo, hi), under- and overflow kept in the first and last of n_bins + 2 slots,
sum of w and sum of w^2 per bin.
Momentum rows: row = 4 * particle + mu, particles 0, 1 incoming, 2.. outgoing (the layout used everywhere).
"""
from __future__ import annotations

import numpy as np

KINDS = ("E", "PX", "PY", "PZ", "PT", "PABS", "PHI", "THETA", "Y", "ABSY", "ETA", "ABSETA",      # single momentum
         "DPHI", "DETA", "DR", "MASS",                                                            # pair
         "SQRT_SHAT", "ET_TOT", "HT")                                                             # event level


def _vec(p, i):
    return p[4 * i], p[4 * i + 1], p[4 * i + 2], p[4 * i + 3]


def _eta(px, py, pz):
    pabs = np.sqrt(px * px + py * py + pz * pz)
    return 0.5 * np.log((pabs + pz) / (pabs - pz))


def observable(kind, p, a=0, b=0, n_out=0):
    """kind in KINDS; a, b = particle indices (as row blocks: 0, 1 incoming, 2.. outgoing); n_out for the event sums."""
    e, px, py, pz = _vec(p, a)
    pt = np.sqrt(px * px + py * py)
    if kind == "E":
        return e
    if kind == "PX":
        return px
    if kind == "PY":
        return py
    if kind == "PZ":
        return pz
    if kind == "PT":
        return pt
    if kind == "PABS":
        return np.sqrt(px * px + py * py + pz * pz)
    if kind == "PHI":
        return np.arctan2(py, px)
    if kind == "THETA":
        return np.arctan2(pt, pz)
    if kind in ("Y", "ABSY"):
        y = 0.5 * np.log((e + pz) / (e - pz))
        return np.abs(y) if kind == "ABSY" else y
    if kind in ("ETA", "ABSETA"):
        eta = _eta(px, py, pz)
        return np.abs(eta) if kind == "ABSETA" else eta
    e2, qx, qy, qz = _vec(p, b)
    if kind in ("DPHI", "DR"):
        d = np.abs(np.arctan2(py, px) - np.arctan2(qy, qx))
        dphi = np.where(d > np.pi, 2.0 * np.pi - d, d)
        if kind == "DPHI":
            return dphi
        deta = _eta(px, py, pz) - _eta(qx, qy, qz)
        return np.sqrt(deta * deta + dphi * dphi)
    if kind == "DETA":
        return np.abs(_eta(px, py, pz) - _eta(qx, qy, qz))
    if kind == "MASS":
        m2 = (e + e2) ** 2 - (px + qx) ** 2 - (py + qy) ** 2 - (pz + qz) ** 2
        return np.sqrt(np.maximum(m2, 0.0))
    if kind == "SQRT_SHAT":
        ea, ax, ay, az = _vec(p, 0)
        eb, bx, by, bz = _vec(p, 1)
        m2 = (ea + eb) ** 2 - (ax + bx) ** 2 - (ay + by) ** 2 - (az + bz) ** 2
        return np.sqrt(np.maximum(m2, 0.0))
    if kind in ("ET_TOT", "HT"):
        out = np.zeros(p.shape[1])
        for i in range(2, 2 + n_out):
            e, px, py, pz = _vec(p, i)
            pt2 = px * px + py * py
            pabs2 = pt2 + pz * pz
            if kind == "ET_TOT":
                out = out + e * np.sqrt(pt2) / np.sqrt(pabs2)                       # Eq. 79
            else:
                out = out + np.sqrt(np.maximum(e * e - pabs2, 0.0) + pt2)           # Eq. 80
        return out
    raise ValueError(kind)


def cut(w, obs, lo=-np.inf, hi=np.inf):
    """Weights with the events outside lo <= obs <= hi set to 0 (a NaN observable fails the cut)."""
    keep = (obs >= lo) & (obs <= hi)
    return np.where(keep, w, 0.0)


def histogram(obs, w, lo, hi, n_bins):
    """(sum w, sum w^2) per slot: slot 0 underflow, 1..n_bins the bins of width (hi-lo)/n_bins, n_bins+1 overflow;
    NaN observables are not filled."""
    sw, sw2 = np.zeros(n_bins + 2), np.zeros(n_bins + 2)
    t = (obs - lo) * (n_bins / (hi - lo))
    ok = ~np.isnan(t)
    k = np.where(t < 0.0, 0, np.where(t >= n_bins, n_bins + 1, np.floor(np.where(ok, t, 0.0)).astype(np.int64) + 1))
    np.add.at(sw, k[ok], w[ok])
    np.add.at(sw2, k[ok], (w * w)[ok])
    return sw, sw2
