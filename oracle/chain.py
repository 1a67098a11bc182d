"""oracle.chain -- TEST INFRASTRUCTURE: the oracle-side call sequence of one pass of the hot path for a workload
(stage by stage, in the paper's order), used by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs.  Calls only ``oracle`` and the shared seeded-input module ``ms_inputs``.
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
    if wl.masses and wl.massive_mode == "reweight":
        p, w, nbad = orc.rambo_massive_reweight(n, xs, wl.sqrt_s, wl.masses, exact=(wl.mapping == "rambo"))
        out["nfail"] = nbad
    else:
        fn = orc.fastrambo if wl.mapping == "fastrambo" else orc.rambo_massless
        p, w = fn(n, xs, energy)
    out["p_massless"], out["w_ps"] = p, w
    if wl.masses and wl.massive_mode == "rescale":
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
