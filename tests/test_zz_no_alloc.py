"""ms_unweight_static (include/madspace_b200.h): the unweighting entry point that allocates nothing -- its scratch is a static
device array inside the library -- against the existing ms_unweight with caller-supplied scratch.  Same kernels, so the
bar is the one of the other unweighting tests: decisions, order, output weights, gathered rows and the count bit-exact.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

DEV = "cuda:0"
SEED_UNWEIGHT = 4242


@pytest.fixture(scope="module")
def ms():
    assert torch.cuda.is_available(), "GPU tests selected on a box without CUDA"
    import paper_2602_06895_b200 as m
    m.lib()
    return m


def _inputs(N, n_rows, key, frac):
    rs = np.random.Generator(np.random.Philox(key=key))
    ld = N + (N & 1)
    w = rs.random(ld) ** 3
    rows = rs.standard_normal((n_rows, ld))
    wmax = float(np.mean(w[:N]) / frac)
    return (torch.from_numpy(w).to(DEV), torch.from_numpy(np.array([wmax])).to(DEV),
            torch.from_numpy(np.ascontiguousarray(rows)).to(DEV), ld)


def _outputs(cap, n_rows):
    return (torch.full((cap,), -1, dtype=torch.int64, device=DEV), torch.zeros(cap, dtype=torch.float64, device=DEV),
            torch.zeros((n_rows, cap), dtype=torch.float64, device=DEV), torch.full((1,), -7, dtype=torch.int64, device=DEV))


def _both_paths(ms, N, n_rows, key, frac, offset):
    """One call of the existing path, one of the static-scratch path, same inputs; returns the accepted count."""
    d_w, d_wmax, d_rows, ld = _inputs(N, n_rows, key, frac)
    cap = N
    r = ms.rng(SEED_UNWEIGHT, 1, offset)
    idx_a, wout_a, rows_a, nacc_a = _outputs(cap, n_rows)
    sb = ms.ms_unweight_scratch_bytes(N)
    scratch = torch.full((sb,), 0xAB, dtype=torch.uint8, device=DEV)
    ms.ms_unweight(N, d_w, d_wmax, r, n_rows, d_rows, cap, idx_a, wout_a, rows_a, nacc_a, scratch, sb, ld)
    idx_b, wout_b, rows_b, nacc_b = _outputs(cap, n_rows)
    ms.ms_unweight_static(N, d_w, d_wmax, r, n_rows, d_rows, cap, idx_b, wout_b, rows_b, nacc_b, ld)
    torch.cuda.synchronize()
    n_a, n_b = int(nacc_a.item()), int(nacc_b.item())
    assert n_a == n_b and 0 < n_a < N
    assert torch.equal(idx_a, idx_b) and torch.equal(wout_a, wout_b) and torch.equal(rows_a, rows_b)
    assert bool((idx_b[n_b:] == -1).all())                               # nothing written past the end
    return n_b


def test_static_scratch_matches_existing_path_on_calls_in_a_row(ms):
    # a large call, then a smaller one with other weights and another acceptance rate (the array still holds the first call's
    # ballots, counts and block totals), then a large one again: every call must stand on its own
    n1 = _both_paths(ms, 3 * (1 << 20) + 5, 4, key=11, frac=0.3, offset=0)
    n2 = _both_paths(ms, 70001, 4, key=12, frac=0.01, offset=1 << 33)
    n3 = _both_paths(ms, (1 << 21) + 513, 24, key=13, frac=1e-3, offset=12345)
    assert n1 > n3 > n2


def test_static_scratch_same_call_twice(ms):
    # the same inputs twice in a row through the static path: identical outputs
    N, n_rows = (1 << 20) + 77, 8
    d_w, d_wmax, d_rows, ld = _inputs(N, n_rows, key=21, frac=0.05)
    outs = []
    for _ in range(2):
        idx, wout, rows, nacc = _outputs(N, n_rows)
        ms.ms_unweight_static(N, d_w, d_wmax, ms.rng(SEED_UNWEIGHT, 1, 0), n_rows, d_rows, N, idx, wout, rows, nacc, ld)
        outs.append((idx, wout, rows, nacc))
    torch.cuda.synchronize()
    for a, b in zip(outs[0], outs[1]):
        assert torch.equal(a, b)
    assert int(outs[0][3].item()) > 0


def test_static_scratch_limits(ms):
    one = torch.zeros(2, dtype=torch.float64, device=DEV)
    nacc = torch.full((1,), -7, dtype=torch.int64, device=DEV)
    # beyond the array's capacity: a clear error, nothing enqueued
    with pytest.raises(ms.MadSpaceError, match="MS_ELIMIT"):
        ms.ms_unweight_static(ms.MS_UNWEIGHT_STATIC_MAX_EVENTS + 1, one, one, ms.rng(1, 1, 0), 0, None, 0, None, None, None, nacc,
                              ms.MS_UNWEIGHT_STATIC_MAX_EVENTS + 2)
    torch.cuda.synchronize()
    assert int(nacc.item()) == -7
    with pytest.raises(ms.MadSpaceError, match="MS_EINVAL"):
        ms.ms_unweight_static(-1, one, one, ms.rng(1, 1, 0), 0, None, 0, None, None, None, nacc, 2)
    # N = 0 (the set-up call before a stream capture): count 0, no output touched
    ms.ms_unweight_static(0, None, one, ms.rng(1, 1, 0), 0, None, 0, None, None, None, nacc, 0)
    torch.cuda.synchronize()
    assert int(nacc.item()) == 0


def test_static_scratch_at_the_maximum_size(ms):
    N = ms.MS_UNWEIGHT_STATIC_MAX_EVENTS
    _both_paths(ms, N, 2, key=31, frac=1e-4, offset=7)
