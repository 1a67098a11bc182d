"""oracle.invariant_maps -- TEST INFRASTRUCTURE: the analytic 1-D mappings for invariants of PAPER.md:150-192
(Eq. 15-20), literally, in numpy fp64: Breit-Wigner (Eq. 16-17), power law (Eq. 18), its logarithmic limit nu = 1
(Eq. 19) and flat (Eq. 20), each as x = G(r) with density g(x) = |dG^-1/dx| (Eq. 15), and the inverse r = G^-1(x)
obtained by solving the printed G for r.  m2 may be negative (the auxiliary mass -a of PAPER.md:185).
"""
from __future__ import annotations

import numpy as np

KINDS = ("FLAT", "POWER", "BW")


def forward(kind, r, x_min, x_max, m2=0.0, par=0.0):
    """par = nu for POWER (nu = 1 selects Eq. 19), = m * Gamma for BW.  Returns (x, g(x))."""
    r = np.asarray(r, dtype=np.float64)
    if kind == "FLAT":                                                   # Eq. 20
        return x_min + (x_max - x_min) * r, np.full_like(r, 1.0) / (x_max - x_min)
    if kind == "BW":                                                     # Eq. 16-17
        mg = par
        u1, u2 = np.arctan((x_min - m2) / mg), np.arctan((x_max - m2) / mg)
        x = mg * np.tan(u1 + (u2 - u1) * r) + m2
        return x, mg / ((u2 - u1) * ((x - m2) ** 2 + mg * mg))
    nu = par
    a, b = x_min - m2, x_max - m2
    if nu == 1.0:                                                        # Eq. 19
        x = np.exp(r * np.log(b) + (1.0 - r) * np.log(a)) + m2
        return x, 1.0 / ((x - m2) * (np.log(b) - np.log(a)))
    p = 1.0 - nu                                                         # Eq. 18
    x = (r * b ** p + (1.0 - r) * a ** p) ** (1.0 / p) + m2
    return x, p / ((b ** p - a ** p) * (x - m2) ** nu)


def inverse(kind, x, x_min, x_max, m2=0.0, par=0.0):
    """Returns (r, g(x))."""
    x = np.asarray(x, dtype=np.float64)
    if kind == "FLAT":
        return (x - x_min) / (x_max - x_min), np.full_like(x, 1.0) / (x_max - x_min)
    if kind == "BW":
        mg = par
        u1, u2 = np.arctan((x_min - m2) / mg), np.arctan((x_max - m2) / mg)
        return (np.arctan((x - m2) / mg) - u1) / (u2 - u1), mg / ((u2 - u1) * ((x - m2) ** 2 + mg * mg))
    nu = par
    a, b = x_min - m2, x_max - m2
    if nu == 1.0:
        return (np.log(x - m2) - np.log(a)) / (np.log(b) - np.log(a)), 1.0 / ((x - m2) * (np.log(b) - np.log(a)))
    p = 1.0 - nu
    return ((x - m2) ** p - a ** p) / (b ** p - a ** p), p / ((b ** p - a ** p) * (x - m2) ** nu)
