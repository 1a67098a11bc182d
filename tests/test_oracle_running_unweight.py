"""Pins for the oracle's running-maximum unweighting with an overweight allowance (reading U-2;
SURVEY.md section 8(f) NEXT-3).

  * the histogram: brute force on the bit patterns; bins are contiguous, 16 per octave; non-positive / non-finite weights
    are not counted; counts are exact and order independent;
  * w_max(f) from the counts: the DEFINING property, checked exactly by sorting the weights -- the overweight excess
    sum_{w > w_max} (w - w_max) is <= f * sum w, while one bin lower it would not be guaranteed; f = 0 gives the first
    edge above every weight; monotone in f;
  * the two-stage procedure is unbiased: the expected number of finally accepted events equals sum min(w, w_f) / w_f
    and the expected sum of output weights equals sum w / w_f, compared with the single-pass values within binomial
    errors; every finally accepted event was kept in the first stage; output weights are max(1, w / w_f);
  * the running maximum never decreases.
"""
import math

import numpy as np

from oracle import running_unweight as ru


def lognormal(seed, n, sigma=2.0):
    rs = np.random.Generator(np.random.Philox(key=seed))
    return np.exp(sigma * rs.standard_normal(n))


def test_histogram_bins():
    w = np.array([1.0, 1.0624, 1.0625, 1.99999, 2.0, 3.0, 1e-300, 5e-324, 0.0, -1.0, np.inf, np.nan, 1.79e308])
    k = ru.bin_index(w)
    assert list(k[8:12]) == [-1, -1, -1, -1]
    assert k[0] == k[1] == 0x3FF0 and k[2] == 0x3FF1 and k[3] == 0x3FFF and k[4] == 0x4000 and k[5] == 0x4008
    assert k[7] == 0 and k[12] == 0x7FEF
    for kk in (0x3FF0, 0x3FF1, 0x4008):
        lo, hi = ru.bin_lower_edge(kk), ru.bin_lower_edge(kk + 1)
        assert lo < hi and hi / lo <= 1.0625 + 1e-15          # 16 bins per octave
        assert ru.bin_index(np.array([lo, np.nextafter(hi, 0)])).tolist() == [kk, kk]
    c = ru.histogram(w)
    assert c.sum() == 9 and c[0x3FF0] == 2
    w2 = lognormal(3, 50000)
    a = ru.histogram(w2)
    b = ru.histogram(w2[::-1].copy())
    b2 = ru.histogram(w2[:100], ru.histogram(w2[100:]))
    assert np.array_equal(a, b) and np.array_equal(a, b2)


def exact_excess(w, thr):
    return float(np.sum(np.maximum(np.sort(w) - thr, 0.0)))


def test_wmax_defining_property():
    for seed, sigma in ((1, 1.0), (2, 2.0), (3, 3.0)):
        w = lognormal(seed, 200000, sigma)
        c = ru.histogram(w)
        prev = float("inf")
        for f in (0.0, 1e-4, 1e-3, 1e-2, 0.1):
            wm = ru.wmax_from_histogram(c, f)
            assert exact_excess(w, wm) <= f * float(np.sum(w)) * (1 + 1e-12)
            assert wm <= prev                                    # larger allowance, lower maximum
            prev = wm
            if f == 0.0:
                assert wm > w.max() and wm / w.max() <= 1.0625 + 1e-12
            else:
                # not over-conservative: two bins lower the exact excess already exceeds the allowance
                k = int(ru.bin_index(np.array([wm]))[0])
                assert exact_excess(w, ru.bin_lower_edge(k - 2)) > 0.5 * f * float(np.sum(w))
    assert ru.wmax_from_histogram(np.zeros(ru.N_BINS, dtype=np.int64), 1e-3) == 0.0


def test_two_stage_unweighting_is_unbiased(orc):
    n_batches, n = 12, 1 << 15
    batches = [(b * n, lognormal(100 + b, n, 2.0)) for b in range(n_batches)]
    kept_idx, kept_w, kept_old, trace, fin_idx, fin_wout = ru.running_unweight(batches, 1e-3, 3, orc)
    assert all(b >= a for a, b in zip(trace, trace[1:])) and trace[-1] > trace[0]
    w_f = trace[-1]
    w_all = np.concatenate([w for _, w in batches])
    assert np.all(np.diff(kept_idx) > 0) and np.all(np.diff(fin_idx) > 0)
    # first stage kept everything the final maximum would always accept
    assert set(np.nonzero(w_all >= w_f)[0]).issubset(set(kept_idx.tolist()))
    final_w = kept_w[fin_idx]
    assert np.array_equal(fin_wout, np.maximum(1.0, final_w / w_f))
    # expectations of a single-pass unweighting at w_f
    p = np.minimum(1.0, w_all / w_f)
    exp_n, var_n = p.sum(), (p * (1 - p)).sum()
    assert abs(len(fin_idx) - exp_n) < 5 * math.sqrt(var_n)
    exp_sum = (w_all / w_f).sum()
    var_sum = (np.maximum(1.0, w_all / w_f) ** 2 * p * (1 - p)).sum()
    assert abs(fin_wout.sum() - exp_sum) < 5 * math.sqrt(var_sum) + 1e-9
    # the overweight part of the final sample is within the allowance
    assert (fin_wout - 1.0).sum() <= 1e-3 * exp_sum * 1.5 + 5 * math.sqrt(var_sum)
