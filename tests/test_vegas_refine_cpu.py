"""ms_vegas_refine is host-only code of the library, so its parity with the oracle's refinement (oracle.vegas_adapt,
reading V-4) is checked here without a GPU: same smoothing, damping and re-split, edge by edge."""
import numpy as np
import pytest

import ms_inputs
from oracle import vegas_adapt


@pytest.fixture(scope="module")
def ms():
    import paper_2602_06895_b200 as m
    m.lib()
    return m


@pytest.mark.parametrize("d,nb,alpha", [(1, 2, 0.5), (3, 7, 1.5), (8, 128, 0.5), (20, 128, 1.0), (2, 1024, 0.5), (4, 1, 0.5)])
def test_refine_matches_the_oracle(ms, d, nb, alpha):
    rs = np.random.Generator(np.random.Philox(key=1000 + nb))
    edges = ms_inputs.seeded_grid(d, nb) if nb > 1 else ms_inputs.uniform_grid(d, 1)
    hist = rs.random((d, nb)) ** 4 * 1e-12          # wide dynamic range, tiny scale (weights squared)
    hist[0, : nb // 3] = 0.0                        # empty bins
    got = ms.ms_vegas_refine(hist, edges, alpha)
    ref = vegas_adapt.refine(edges, hist, alpha)
    # the equal-share walk carries a running sum over n_bins steps: rounding-level agreement, ~n_bins * eps
    assert np.max(np.abs(got - ref)) <= 1e-12
    assert ms.ms_check_grid(got) == 0


def test_refine_fixed_points_and_errors(ms):
    d, nb = 3, 32
    edges = ms_inputs.seeded_grid(d, nb)
    assert np.array_equal(ms.ms_vegas_refine(np.zeros((d, nb)), edges), edges)           # nothing learnt
    flat = ms.ms_vegas_refine(np.full((d, nb), 3.0), edges, 0.5)
    assert np.max(np.abs(flat - edges)) <= 1e-15                                          # equal shares already
    bad = edges.copy()
    bad[1, 5] = bad[1, 4]
    with pytest.raises(ms.MadSpaceError) as e:
        ms.ms_vegas_refine(np.ones((d, nb)), bad)
    assert e.value.code == ms.MS_EGRID
    neg = np.ones((d, nb))
    neg[0, 0] = -1.0
    with pytest.raises(ms.MadSpaceError) as e:
        ms.ms_vegas_refine(neg, edges)
    assert e.value.code == ms.MS_EINVAL
    with pytest.raises(ms.MadSpaceError):
        ms.ms_vegas_refine(np.ones((d, nb - 1)), edges)


def test_wmax_from_histogram_matches_the_oracle(ms):
    """ms_wmax_from_histogram is host-only code: identical doubles to the oracle's walk over the same counts."""
    from oracle import running_unweight as ru
    rs = np.random.Generator(np.random.Philox(key=31))
    for sigma in (0.5, 2.0, 4.0):
        w = np.exp(sigma * rs.standard_normal(100000))
        counts = ru.histogram(w)
        for f in (0.0, 1e-4, 1e-3, 1e-2, 0.3, 1.0, 5.0):
            assert ms.ms_wmax_from_histogram(counts, f) == ru.wmax_from_histogram(counts, f)
    empty = np.zeros(ru.N_BINS, dtype=np.int64)
    assert ms.ms_wmax_from_histogram(empty, 1e-3) == 0.0
    top = empty.copy()
    top[0x7FEF] = 1
    assert ms.ms_wmax_from_histogram(top, 1e-3) == float("inf") == ru.wmax_from_histogram(top, 1e-3)
    with pytest.raises(ms.MadSpaceError):
        ms.ms_wmax_from_histogram(empty, -1.0)
    with pytest.raises(ms.MadSpaceError):
        ms.ms_wmax_from_histogram(empty[:100], 1e-3)
