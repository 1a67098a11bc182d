"""oracle.vegas_adapt -- TEST INFRASTRUCTURE: refinement step of the classic VEGAS grid adaptation, plain Python.

PAPER.md:603 ("the classic VEGAS algorithm"), :746 ("grids ... optimized during an initial adaptation phase and ...
then frozen"); the paper prints no equations.  Reading V-4: G. P. Lepage's algorithm (J. Comput. Phys. 27
(1978) 192; refs PAPER.md:859, :886-887), one dimension at a time, in its published order:

  1. d_j = sum of (f J)^2 over the events whose uniform fell into bin j        (the accumulation pass)
  2. smooth:    d_j <- (d_{j-1} + 6 d_j + d_{j+1}) / 8,  ends (7 d_0 + d_1)/8, (d_{nb-2} + 7 d_{nb-1})/8; normalise to sum 1
  3. compress:  d_j <- ((1 - d_j) / ln(1 / d_j))^alpha                          (damping; d_j = 0 stays 0)
  4. re-split:  new edges such that every new bin holds the same share sum(d)/nb, by linear interpolation inside the
                old bins.
A dimension whose histogram is identically zero is left unchanged.  Pure-Python loops: the tables are tiny (d x n_bins).
"""
from __future__ import annotations

import math

import numpy as np


def smooth(d):
    nb = len(d)
    if nb == 1:
        return [float(d[0])]
    out = [0.0] * nb
    out[0] = (7.0 * d[0] + d[1]) / 8.0
    for j in range(1, nb - 1):
        out[j] = (d[j - 1] + 6.0 * d[j] + d[j + 1]) / 8.0
    out[nb - 1] = (d[nb - 2] + 7.0 * d[nb - 1]) / 8.0
    return out


def compress(d, alpha):
    out = []
    for v in d:
        if v <= 0.0:
            out.append(0.0)
        elif v >= 1.0:                      # a single occupied bin: (1-d)/ln(1/d) -> 1 as d -> 1
            out.append(1.0)
        else:
            out.append(((1.0 - v) / math.log(1.0 / v)) ** alpha)
    return out


def resplit(edges, d):
    """New edges with equal shares of sum(d) per bin (Lepage's rebinning walk)."""
    nb = len(d)
    share = sum(d) / nb
    new = [0.0] * (nb + 1)
    new[nb] = 1.0
    j, acc = -1, 0.0
    for i in range(1, nb):
        while acc < share:
            j += 1
            acc += d[j]
        acc -= share
        new[i] = edges[j + 1] - (acc / d[j]) * (edges[j + 1] - edges[j])
    return new


def refine(edges, hist, alpha=0.5):
    """edges [d][nb+1], hist [d][nb] -> refined edges [d][nb+1]."""
    edges = np.asarray(edges, dtype=np.float64)
    hist = np.asarray(hist, dtype=np.float64)
    out = edges.copy()
    for dim in range(edges.shape[0]):
        d = [float(v) for v in hist[dim]]
        total = sum(d)
        if not total > 0.0:
            continue
        d = smooth(d)
        total = sum(d)
        d = [v / total for v in d]
        d = compress(d, alpha)
        out[dim] = resplit([float(v) for v in edges[dim]], d)
    return out
