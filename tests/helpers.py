"""Test helpers: the oracle-side chain for a workload, and Workload -> PathSpec translation.

The oracle chain calls ONLY ``oracle`` (CPU, fp64 C) and ``ms_inputs``; the CUDA path is never consulted for an
expected value.
"""
from __future__ import annotations

import numpy as np

import ms_inputs


from oracle.chain import oracle_chain, oracle_uniforms  # noqa: F401  (re-exported for the tests)


def path_spec(wl: ms_inputs.Workload, edges=None):
    from paper_2602_06895_b200.pipeline import PathSpec
    return PathSpec(n=wl.n, sqrt_s=wl.sqrt_s, mapping=wl.mapping, edges=wl.grid() if edges is None else edges,
                    pdf=wl.pdf, tau_min=wl.tau_min, masses=tuple(wl.masses), massive_mode=wl.massive_mode, toy=wl.toy, toy_reg=ms_inputs.TOY_REG,
                    unweight=wl.unweight, inverse=wl.inverse, prerun=ms_inputs.PRERUN,
                    seed_events=ms_inputs.SEED_EVENTS, seed_unweight=ms_inputs.SEED_UNWEIGHT)


def toy_condition(p, n, e_scale, reg=ms_inputs.TOY_REG):
    """kappa_f of DESIGN.md reading T: |df|/f <= eta * kappa_f for a momentum perturbation eta * e_scale."""
    k = np.zeros(p.shape[1])
    for i in range(n - 1):
        a, b = p[4 * (i + 2):4 * (i + 2) + 4], p[4 * (i + 3):4 * (i + 3) + 4]
        na, nb = a[1:] / a[0], b[1:] / b[0]
        sij = a[0] * b[0] * np.sum((na - nb) ** 2, axis=0)
        k += 2 * (a[0] + b[0]) * e_scale / (sij + reg)
    return k


EPS = 2.220446049250313e-16


# Events allowed to need the kappa_f term of the toy-weight bound: none in a batch below
# 50 000 events, one per 50 000 beyond (measured on B200, round 2: 1 of 131 405 cfg-2 events at 1.03e-12, 0 of 131 405
# cfg-5 events, 0 of every smaller batch).
TOY_FALLBACK_BASE, TOY_FALLBACK_PER = 0, 50000


def assert_toy_weights(w, w_ref, p_ref, n, e_scale, eta, label, tol=1e-12, max_fallback=None):
    """End-to-end parity of the integrand-weighted weights: each
    side evaluates f on its OWN momenta, so |dw|/w <= 1e-12 is expected for every event but only
    1e-12 + 4 max(eta, eps) kappa_f is guaranteed (f is ill-conditioned in the momenta; eta = max |dp| / E_scale of this
    batch).  Every event is held to the guaranteed bound; the events that NEED its kappa_f term are counted, printed
    and limited to `max_fallback` (default: one per TOY_FALLBACK_PER events of the batch)."""
    rel = np.abs(w - w_ref) / np.abs(w_ref)
    kappa = toy_condition(p_ref, n, e_scale)
    bound = tol + 4.0 * max(eta, EPS) * kappa
    n_fallback = int(np.sum(rel > tol))
    worst = float(np.max(rel)) if rel.size else 0.0
    k_worst = int(np.argmax(rel)) if rel.size else 0
    if max_fallback is None:
        max_fallback = TOY_FALLBACK_BASE + rel.size // TOY_FALLBACK_PER
    print("[toy parity] %s: %d events, max rel dw = %.3e (event %d: kappa_f = %.3g, bound %.3e), eta = %.2e, n_fallback "
          "(rel > %.0e) = %d (allowed %d), max kappa_f = %.3g"
          % (label, rel.size, worst, k_worst, float(kappa[k_worst]) if kappa.size else 0.0,
             float(bound[k_worst]) if kappa.size else 0.0, eta, tol, n_fallback, max_fallback,
             float(np.max(kappa)) if kappa.size else 0.0))
    assert np.all(rel <= bound), "weight beyond 1e-12 + 4 eta kappa_f: max excess ratio %.3g" % float(np.max(rel / bound))
    assert n_fallback <= max_fallback, "%d events need the kappa_f term (allowed %d), max rel %.3e" % (n_fallback, max_fallback, worst)
    return {"n_fallback": n_fallback, "max_rel": worst}


def inverse_weight_bound(p, n, masses=None, c=2.0, tol=1e-12):
    """Per-event bound on the relative difference between two fp64 evaluations of the INVERSE map's weight on identical
    momenta (reading F-8).  Both sides rebuild M_i = sqrt(Q_i^2) from the momenta -- |dM/M| <= eps gamma_i^2,
    gamma_i = Q_i^0 / M_i -- and form 1 - u_i^2 and 1 - y_i by subtraction (Eq. 64, 67 literally), so a step contributes
    eps (2k+3) (gamma_i^2 a_i + gamma_{i-1}^2 a_{i-1} + 2) / (1 - u_i^2), with a_i = M_i / K_i for the massive map
    (u_i = K_i / K_{i-1}, K = M - sum of masses: one more cancellation) and 1 otherwise; the massive map's rho ratio adds
    eps gamma_{i-1} p^0_{i-1} / q_{i-1} (rest-frame momentum recovered from boosted components).
    bound = tol + c eps * sum over steps."""
    out = np.stack([p[4 * (j + 2):4 * (j + 2) + 4] for j in range(n)])          # [n][4][N]
    Q = np.cumsum(out[::-1], axis=0)[::-1]                                       # Q[i] = sum_{j>=i} p_j (0-based)
    M = np.sqrt(np.maximum(Q[:, 0] ** 2 - Q[:, 1] ** 2 - Q[:, 2] ** 2 - Q[:, 3] ** 2, 0.0))
    N = p.shape[1]
    gam2 = np.full((n, N), 1.0)
    amp = np.ones((n, N))
    K = M.copy()
    if masses is not None:
        msuf = np.cumsum(np.asarray(masses, dtype=float)[::-1])[::-1]
        K = M - msuf[:, None]
        K[n - 1] = 0.0
    with np.errstate(divide="ignore", invalid="ignore"):
        gam2[:n - 1] = (Q[:n - 1, 0] / M[:n - 1]) ** 2
        if masses is not None:
            amp[:n - 1] = M[:n - 1] / K[:n - 1]
        kappa = np.full(N, 2.0 * n)
        for i in range(1, n - 1):                                                # 0-based: u = K[i] / K[i-1], k = n - 1 - i
            k = n - 1 - i
            u = K[i] / K[i - 1]
            kappa += (2 * k + 3) * (gam2[i] * amp[i] + gam2[i - 1] * amp[i - 1] + 2.0) / (1.0 - u * u)
        if masses is not None:
            for i in range(1, n):                                                # decay Q[i-1] -> p[i-1] + Q[i]
                m1 = masses[i - 1]
                m2 = M[i] if i < n - 1 else masses[n - 1]
                lam = (M[i - 1] ** 2 - (m1 + m2) ** 2) * (M[i - 1] ** 2 - (m1 - m2) ** 2)
                q = np.sqrt(np.maximum(lam, 0.0)) / (2.0 * M[i - 1])
                kappa += np.sqrt(gam2[i - 1]) * out[i - 1, 0] / q
    kappa = np.where(np.isfinite(kappa), kappa, np.inf)
    return tol + c * EPS * kappa
