"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (HotPath.step on N = 2^24 ...
2^26 events): sampled outputs the oracle computes one by one, plus properties that hold at any size, evaluated over
EVERY event on the device.

Sampled indices: the first and the last 256-event tile, the 32 events around every quarter of the batch, and 4096
seeded random indices.  Properties over all events: weights finite and positive, no failure flag, four-momentum
conservation, on-shell masses, (cfg 5) the round trip back to the Philox uniforms with the condition-aware tolerance of
DESIGN.md reading F-7, (cfg 2, 5) the unweighted list bit-exact against the oracle fed the same 2^24 weights.
"""
import numpy as np
import pytest
import torch

import ms_inputs
from helpers import assert_toy_weights, inverse_weight_bound, oracle_chain, path_spec

pytestmark = pytest.mark.gpu

DEV = "cuda:0"
TOL_P = 1e-12
TOL_W = 1e-12


@pytest.fixture(scope="module")
def ms():
    assert torch.cuda.is_available(), "GPU tests selected on a box without CUDA"
    import paper_2602_06895_b200 as m
    m.lib()
    return m


def sample_indices(N, seed):
    rs = np.random.Generator(np.random.Philox(key=seed))
    parts = [np.arange(0, 256), np.arange(N - 256, N), rs.integers(0, N, 4096)]
    for q in (1, 2, 3):
        parts.append(np.arange(q * N // 4 - 16, q * N // 4 + 16))
    return np.unique(np.concatenate(parts)).astype(np.int64)


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg4", "cfg4rw", "cfg5"])
def test_full_size_step(ms, orc, name):
    from paper_2602_06895_b200.pipeline import HotPath
    wl = ms_inputs.WORKLOADS[name]
    N, n = wl.N, wl.n
    # bench.py's configuration, except that the round trip (cfg 5) runs as the two calls ms_fastrambo_inverse + ms_vegas_map, whose
    # x-space output and phase-space weight are checked below; the fused call is then compared with them bit for bit
    hp = HotPath(path_spec(wl), N, DEV, cap=max(1 << 16, N // 256), fuse_inverse=False)
    hp.step(0)
    torch.cuda.synchronize()
    assert int(hp.fail.item()) == 0

    # ---- sampled outputs against the oracle, event by event
    idx = sample_indices(N, 11)
    t_idx = torch.from_numpy(idx).to(DEV)
    p = hp.p[:, t_idx].cpu().numpy()
    w = hp.w[t_idx].cpu().numpy()
    ref = oracle_chain(orc, wl, idx)
    eta = float(np.max(np.abs(p - ref["p"])) / wl.sqrt_s)
    assert eta <= TOL_P, "max |dp|/E_scale = %.3e" % eta
    rel = np.abs(w - ref["w"]) / ref["w"]
    if wl.toy:
        assert_toy_weights(w, ref["w"], ref["p"], n, wl.sqrt_s, eta, "%s full size, %d sampled events" % (name, idx.size))
    else:
        assert np.max(rel) <= TOL_W, "max rel dw = %.3e" % np.max(rel)

    # ---- cfg 1 (k = 1, c = 2 makes FastRambo exact): EVERY weight of the 2^16
    # events equals Phi_3(1000 GeV) = 125.982556379686 GeV^2, and the step replayed from a CUDA graph (how a sub-wave
    # batch is run without launch latency) reproduces the buffers bit for bit
    if name == "cfg1":
        assert float((hp.w[:N] / 125.982556379686 - 1.0).abs().max()) < 1e-13
        p0, w0 = hp.p.clone(), hp.w.clone()
        g = hp.capture(0)
        hp.p.fill_(-7.0)
        hp.w.fill_(-7.0)
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(hp.p, p0) and torch.equal(hp.w, w0)

    # ---- properties over ALL events, on the device
    assert bool(torch.isfinite(hp.w[:N]).all()) and bool((hp.w[:N] > 0).all())
    assert hp.ld == N
    P = hp.p.view(n + 2, 4, N)
    total = P[2:].sum(dim=0) - P[0] - P[1]                               # sum p_f - p_a - p_b
    scale = (P[0, 0] + P[1, 0])                                          # sqrt(s) partonic, or E_a + E_b in the lab
    assert float((total.abs().amax(dim=0) / scale).max()) <= 1e-13
    m2 = P[2:, 0] ** 2 - (P[2:, 1:] ** 2).sum(dim=1)                     # [n, N]
    masses = torch.tensor(list(wl.masses) if wl.masses else [0.0] * n, dtype=torch.float64, device=DEV)
    # relative to (E_a + E_b)^2 = s in the partonic frame, gamma^2 s-hat in the lab (the recoil p_n = Q_n carries the
    # rounding of the whole chain, and the boost multiplies absolute errors by gamma <= ~34: SURVEY.md section 8c D/X pins)
    assert float(((m2 - masses[:, None] ** 2).abs() / scale ** 2).max()) <= 1e-13
    del total, m2

    # ---- unweighting at full size: the oracle unweights the GPU's 2^24 weights
    if wl.unweight:
        w_all = hp.w[:N].cpu().numpy()
        wmax_o = orc.wmax(np.ascontiguousarray(w_all[:ms_inputs.PRERUN]))
        assert hp.wmax.item() == wmax_o
        idx_o, wout_o, nacc_o = orc.unweight(np.ascontiguousarray(w_all), wmax_o, ms_inputs.SEED_UNWEIGHT, 1, 0, N)
        nacc = int(hp.n_acc.item())
        assert nacc == nacc_o and 0 < nacc <= hp.cap
        assert np.array_equal(hp.idx[:nacc].cpu().numpy(), idx_o)
        assert np.array_equal(hp.w_out[:nacc].cpu().numpy(), wout_o)
        assert torch.equal(hp.rows_out[:, :nacc], hp.p[:, torch.from_numpy(idx_o).to(DEV)])
        del w_all

    # ---- cfg 5: r -> V -> F -> F^-1 -> V^-1 -> r' over every value of every event (reading F-7)
    if wl.inverse:
        d = 3 * n - 4
        nb = wl.grid_bins
        r = torch.empty((d, hp.ld), dtype=torch.float64, device=DEV)
        ms.ms_fill_uniforms(N, d, ms.rng(ms_inputs.SEED_EVENTS, 0, 0), r, hp.ld)
        x = torch.empty_like(r)
        ms.ms_vegas_map(N, d, nb, hp.d_edges, 0, r, ms.rng(0), x, None, hp.ld)      # forward map (bit-exact vs oracle)
        phi_rows = torch.tensor([n - 1 + 2 * a for a in range(n - 1)], device=DEV)

        def wrapped(dev):                                                 # phi is periodic: 0 and 1 are the same point
            dev[phi_rows] = torch.minimum(dev[phi_rows], 1.0 - dev[phi_rows])
            return dev

        # condition of an event: u_min over the chain of invariant masses (last pair dominates, reading F-7)
        Q = P[2:].flip(0).cumsum(dim=0).flip(0)                          # suffix sums Q_i, i = 1..n
        M = (Q[:, 0] ** 2 - (Q[:, 1:] ** 2).sum(dim=1)).clamp_min(0).sqrt()
        u_min = (M[1:n] / M[0:n - 1]).amin(dim=0)                        # u_2 .. u_n-1 and M_n-1/M_n-2
        tol_x = 1e-10 * torch.clamp(1e-3 / u_min, min=1.0) ** 2
        del Q, M
        # (a) phase-space inverse: x' against x
        dx = wrapped((hp.x_inv[:, :N] - x[:, :N]).abs())
        worst_x = dx.amax(dim=0)
        n_bad_x = int((worst_x > tol_x).sum())
        n_over_x = int((worst_x > 1e-10).sum())
        med_x = float(dx.median())
        # (b) through the grid: dr = dx / (n_bins * bin width); seeded bins are as narrow as ~1e-6
        j = torch.clamp((r[:, :N] * nb).long(), max=nb - 1)
        edges = hp.d_edges[:d]
        width = torch.gather(edges, 1, j + 1) - torch.gather(edges, 1, j)
        dr = wrapped((hp.r_inv[:, :N] - r[:, :N]).abs())
        n_bad_r = int(((dr > (tol_x[None, :] + 4e-16) / (nb * width) * 1.01 + 1e-15).any(dim=0)).sum())
        n_over_r = int((dr.amax(dim=0) > 1e-10).sum())
        med_r = float(dr.median())
        print("round trip over %d events x %d dims: x-space median %.2e, >1e-10: %d events, beyond F-7 tolerance: %d; "
              "r-space median %.2e, >1e-10: %d events, beyond tolerance: %d"
              % (N, d, med_x, n_over_x, n_bad_x, med_r, n_over_r, n_bad_r))
        assert n_bad_x == 0 and n_bad_r == 0
        assert n_over_x <= 64 and n_over_r <= 1024, "expected O(10) / O(100) per 2^24 (reading F-7)"
        assert med_x <= 1e-15 and med_r <= 1e-14
        # the inverse returns the forward phase-space weight
        w_ps = hp.w_inv[t_idx].cpu().numpy()
        rel_ps = np.abs(w_ps - ref["w_ps"]) / ref["w_ps"]
        bound = inverse_weight_bound(ref["p"], n)                        # reading F-8
        print("inverse weight vs forward weight: max rel = %.3e, max rel/bound = %.3g, beyond 1e-12: %d of %d"
              % (rel_ps.max(), (rel_ps / bound).max(), int((rel_ps > 1e-12).sum()), rel_ps.size))
        assert np.all(rel_ps <= bound) and np.median(rel_ps) <= 1e-13
        # the fused inverse (bench.py's default): the same uniforms bit for bit over all 20 x 2^24 values, and the phase-space
        # weight times the grid's Jacobian
        assert hp.can_fuse_inverse
        r_two = hp.r_inv.clone()
        w_two = hp.w_inv.clone()
        hp.r_inv.zero_()
        hp.invert_fused()
        torch.cuda.synchronize()
        assert torch.equal(hp.r_inv[:, :N], r_two[:, :N])
        jac = (nb * width).prod(dim=0)                                    # of the generating bins = the bins found (r' ~ r)
        ok = dr.amax(dim=0) < 0.25 / nb                                   # events whose r' stayed in r's bins
        rel_j = ((hp.w_inv[:N] - w_two[:N] * jac).abs() / (w_two[:N] * jac))[ok]
        assert int(ok.sum()) > 0.999 * N and float(rel_j.max()) <= 1e-12
        del r_two, w_two
