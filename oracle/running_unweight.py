"""oracle.running_unweight -- TEST INFRASTRUCTURE: unweighting against a running maximum weight with an overweight
allowance, plain numpy / Python.

PAPER.md:693: "We estimate the maximum event weight on the fly, allowing for a user-defined amount of overweight events
relative to the total cross section.  The maximum weight therefore increases during the generation process, hence the
events in the intermediate files are only partially unweighted.  Once the estimated number of unweighted events reaches
the target event count, a final unweighting with respect to the final maximum weight is performed."  (:755, :772: the
allowance used is 0.1 %.)  The paper gives no formulas; reading U-2:

  * statistics: a histogram of all weights seen so far over FIXED logarithmic bins -- bin index = bits 62..48 of the
    IEEE-754 pattern (11 exponent bits + 4 mantissa bits: 16 bins per octave); only counts are kept, so the statistic
    is exact and independent of the order in which events arrive;
  * w_max(f): with lo_k the lower edge of bin k, C_k = number of events in bins >= k, the overweight excess above the
    threshold lo_k is bounded by X_k = sum_{j>=k} count_j (lo_{j+1} - lo_k) and the total by T = sum_j count_j lo_j;
    w_max = the smallest lo_k with X_k <= f T, which guarantees  sum_{w > w_max} (w - w_max) <= f sum w;
    the running maximum never decreases: w_max <- max(previous w_max, this value);
  * every batch is unweighted against the w_max known after that batch (accept u w_max < w, keep w and that w_max);
  * final pass over the kept events against the final w_f: an event kept with probability min(1, w / w_old) must survive
    with probability min(1, w / w_f) / min(1, w / w_old) = min(1, max(w, w_old) / w_f), so it is the same hit-or-miss test
    applied to w_eff = max(w, w_old) with a fresh uniform (stream 2, counter = position in the kept list); the
    output weight max(1, w_eff / w_f) = max(1, w / w_f).
"""
from __future__ import annotations

import numpy as np

N_BINS = 1 << 15


def bin_index(w):
    """Bin of each weight (int64), -1 for weights that are not positive finite numbers."""
    w = np.ascontiguousarray(w, dtype=np.float64)
    bits = w.view(np.uint64)
    k = ((bits >> np.uint64(48)) & np.uint64(0x7FFF)).astype(np.int64)
    ok = (w > 0.0) & np.isfinite(w)
    return np.where(ok, k, -1)


def bin_lower_edge(k):
    return np.array([int(k) << 48], dtype=np.uint64).view(np.float64)[0]


def histogram(w, counts=None):
    if counts is None:
        counts = np.zeros(N_BINS, dtype=np.int64)
    k = bin_index(w)
    np.add.at(counts, k[k >= 0], 1)
    return counts


def wmax_from_histogram(counts, fraction):
    """Smallest bin edge lo_k with X_k <= fraction * T (see the module docstring); 0.0 for an empty histogram, +inf if
    no finite edge qualifies (weights in the very last finite bin)."""
    top = 0x7FF0                                   # first bin of the exponent 0x7FF (inf / nan): never counted
    lo = np.array([k << 48 for k in range(top + 1)], dtype=np.uint64).view(np.float64)   # lo[top] = +inf
    T = 0.0
    for k in range(top):
        c = int(counts[k])
        if c:
            T += float(c) * float(lo[k])
    if not T > 0.0:
        return 0.0
    allowed = fraction * T
    X, C, best = 0.0, 0, float("inf")
    for k in range(top - 1, -1, -1):               # threshold lo_k, walking down: X_k = X_{k+1} + C_k (lo_{k+1} - lo_k)
        C += int(counts[k])
        if C:
            X = X + float(C) * (float(lo[k + 1]) - float(lo[k]))
        if X <= allowed:
            best = float(lo[k])
        else:
            break
    return best


def running_unweight(batches, fraction, seed, orc):
    """batches: list of (global_event_offset, weights).  Returns (kept global indices, their weights, their w_old, w_max
    after each batch, final indices into the kept list, final output weights)."""
    counts = np.zeros(N_BINS, dtype=np.int64)
    w_max = 0.0
    kept_idx, kept_w, kept_old, trace = [], [], [], []
    for offset, w in batches:
        w = np.ascontiguousarray(w, dtype=np.float64)
        histogram(w, counts)
        w_max = max(w_max, wmax_from_histogram(counts, fraction))
        trace.append(w_max)
        idx, _, n_acc = orc.unweight(w, w_max, seed, 1, offset, len(w))
        kept_idx.append(idx + offset)
        kept_w.append(w[idx])
        kept_old.append(np.full(len(idx), w_max))
    kept_idx, kept_w, kept_old = np.concatenate(kept_idx), np.concatenate(kept_w), np.concatenate(kept_old)
    w_eff = np.ascontiguousarray(np.maximum(kept_w, kept_old))
    fin_idx, fin_wout, _ = orc.unweight(w_eff, w_max, seed, 2, 0, len(w_eff))
    return kept_idx, kept_w, kept_old, trace, fin_idx, fin_wout
