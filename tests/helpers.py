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
