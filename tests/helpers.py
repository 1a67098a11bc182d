"""Test helpers: the oracle-side chain for a workload, and Workload -> PathSpec translation.

The oracle chain calls ONLY ``oracle`` (CPU, fp64 C) and ``ms_inputs``; the CUDA path is never consulted for an
expected value.
"""
from __future__ import annotations

import numpy as np

import ms_inputs


def oracle_uniforms(orc, d, seed, stream, events):
    """Uniform rows [d, len(events)] for arbitrary global event indices (counter-based => one by one is exact)."""
    events = np.asarray(events, dtype=np.int64)
    if len(events) and np.all(np.diff(events) == 1):
        return orc.fill_uniforms(len(events), d, seed, stream, int(events[0]))
    out = np.empty((d, len(events)))
    for k, e in enumerate(events):
        out[:, k] = orc.fill_uniforms(1, d, seed, stream, int(e))[:, 0]
    return out


def oracle_chain(orc, wl: ms_inputs.Workload, events, edges=None):
    """Everything ms_generate computes for `events`, stage by stage with the oracle."""
    n = wl.n
    r = oracle_uniforms(orc, wl.d, ms_inputs.SEED_EVENTS, ms_inputs.STREAM_EVENTS, events)
    edges = wl.grid() if edges is None else edges
    if edges is not None:
        x, jac = orc.vegas_forward(edges, r)
    else:
        x, jac = r, np.ones(r.shape[1])
    off = 0
    out = {"r": r, "x": x, "jac": jac}
    if wl.pdf:
        x1x2, sqrt_shat, jx = orc.pdf_x_sample(wl.sqrt_s ** 2, wl.tau_min, np.ascontiguousarray(x[0:2]))
        off = 2
        energy = sqrt_shat
        out.update(x1x2=x1x2, sqrt_shat=sqrt_shat, jx=jx)
    else:
        energy = wl.sqrt_s
        jx = 1.0
    xs = np.ascontiguousarray(x[off:off + 3 * n - 4])
    fn = orc.fastrambo if wl.mapping == "fastrambo" else orc.rambo_massless
    p, w = fn(n, xs, energy)
    out["p_massless"], out["w_ps"] = p, w
    if wl.masses:
        p, w, nfail = orc.massive_rescale(n, wl.sqrt_s, wl.masses, p, w)
        out["nfail"] = nfail
    if wl.pdf:
        p = orc.pdf_boost(n, wl.sqrt_s ** 2, x1x2, p)
    wtot = w * jac * jx
    out["w_nof"] = wtot
    if wl.toy:
        f = orc.toy_integrand(n, p, ms_inputs.TOY_REG)
        out["f"] = f
        wtot = wtot * f
    out["p"], out["w"] = p, wtot
    return out


def path_spec(wl: ms_inputs.Workload, edges=None):
    from paper_2602_06895_b200.pipeline import PathSpec
    return PathSpec(n=wl.n, sqrt_s=wl.sqrt_s, mapping=wl.mapping, edges=wl.grid() if edges is None else edges,
                    pdf=wl.pdf, tau_min=wl.tau_min, masses=tuple(wl.masses), toy=wl.toy, toy_reg=ms_inputs.TOY_REG,
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
