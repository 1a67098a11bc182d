"""HotPath -- device buffers plus the call sequence of one pass of the hot path (what bench.py times and the
tests check).  Marshalling and buffer ownership only: every arithmetic step is a call into the C ABI.

One step = ms_generate (Philox -> VEGAS -> [x1,x2] -> Rambo/FastRambo -> [rescale] -> [boost] -> [toy] -> weight)
           [unweighting: ms_generate_unweight instead -- the hit-or-miss decision against w_max of the pre-run (computed
            once per grid) is taken in the generation kernel -- then ms_unweight_compact (stable compaction)]
           [-> ms_fastrambo_inverse -> ms_vegas_map(inverse)]            (round trip, cfg 5)
"""
from __future__ import annotations

import contextlib
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np
import torch

from . import (ms_elementwise_max, ms_weight_histogram, ms_wmax_from_histogram, MS_HIST_BINS,
               ms_vegas_accumulate, ms_vegas_refine, gen_config, ms_check_grid, ms_fastrambo_inverse, ms_generate, ms_reduce_max, ms_unweight,
               ms_unweight_scratch_bytes, ms_vegas_map, rng, MadSpaceError, MS_EGRID, ms_generate_unweight,
               ms_unweight_compact, ms_accept_bits_words)


@contextlib.contextmanager
def _on(stream):
    """Make `stream` (a torch.cuda.Stream, a raw cudaStream_t handle, or None = keep the current one) torch's current
    stream, so that the library calls (which then take the current stream) and the few torch bookkeeping ops between
    them (zeroing a scalar, allocations) are ordered on ONE stream."""
    if stream is None:
        yield
        return
    s = stream if isinstance(stream, torch.cuda.Stream) else torch.cuda.ExternalStream(int(stream))
    with torch.cuda.stream(s):
        yield


@dataclass
class PathSpec:
    """What one step computes (mirrors ms_gen_config plus the unweighting / round-trip stages)."""
    n: int
    sqrt_s: float
    mapping: str = "fastrambo"            # "fastrambo" | "rambo"
    edges: Optional[np.ndarray] = None    # host VEGAS table [d][n_bins+1] or None
    pdf: bool = False
    tau_min: float = 0.0
    masses: Sequence[float] = ()
    massive_mode: str = "rescale"       # "rescale" (strategy i, Newton) | "reweight" (strategy ii, Eq. 68-69)
    toy: bool = False
    toy_reg: float = 100.0
    unweight: bool = False
    inverse: bool = False
    prerun: int = 1 << 16                 # w_max = max weight of events 0..prerun-1 (reading U)
    seed_events: int = 1
    seed_unweight: int = 3
    rel_tol: float = 1e-14
    max_iter: int = 10

    @property
    def d_used(self) -> int:
        return 3 * self.n - 4 + (2 if self.pdf else 0)

    @property
    def rows_p(self) -> int:
        return 4 * (self.n + 2)


class HotPath:
    def __init__(self, spec: PathSpec, N: int, device="cuda:0", cap: Optional[int] = None, gather_rows: bool = True,
                 fuse_decision: bool = True):
        if not torch.cuda.is_available():
            raise RuntimeError("HotPath needs a CUDA device: there is no CPU fallback")
        self.spec, self.N, self.device = spec, int(N), torch.device(device)
        self.ld = (self.N + 1) // 2 * 2                      # even row stride keeps every row 16-byte aligned
        f64 = dict(dtype=torch.float64, device=self.device)
        self.p = torch.empty((spec.rows_p, self.ld), **f64)
        self.w = torch.empty(self.ld, **f64)
        self.x1x2 = torch.empty((2, self.ld), **f64) if spec.pdf else None
        self.fail = torch.zeros(1, dtype=torch.int32, device=self.device)
        self.d_edges = None
        self.grid_dims = self.grid_bins = 0
        self.tail_unit_jacobian = False
        if spec.edges is not None:
            self.set_grid(spec.edges)
        self.cfg = gen_config(spec.n, spec.mapping, spec.sqrt_s, self.grid_dims, self.grid_bins, spec.pdf, spec.tau_min,
                              tuple(spec.masses), spec.rel_tol, spec.max_iter, spec.toy, spec.toy_reg,
                              tail_unit_jacobian=self.tail_unit_jacobian, massive_mode=spec.massive_mode)
        if spec.unweight:
            self.cap = int(cap) if cap is not None else max(1024, self.N // 64)
            self.wmax = torch.zeros(1, **f64)
            self.idx = torch.empty(self.cap, dtype=torch.int64, device=self.device)
            self.w_out = torch.empty(self.cap, **f64)
            self.gather_rows = gather_rows
            self.rows_out = torch.empty((spec.rows_p, self.cap), **f64) if gather_rows else None
            self.n_acc = torch.zeros(1, dtype=torch.int64, device=self.device)
            self.scratch_bytes = ms_unweight_scratch_bytes(self.N)
            self.scratch = torch.empty(self.scratch_bytes, dtype=torch.uint8, device=self.device)
            self._pre = None                                   # buffers of the replayed pre-run, allocated on first use
            self.fail_pre = torch.zeros(1, dtype=torch.int32, device=self.device)
            self._wmax_cached = False                          # w_max is a function of (spec, grid): computed once
            # fuse_decision: generate() also takes the accept/reject decisions (one bit per event) and unweight() only
            # compacts; False keeps the two-call form ms_generate + ms_unweight (same results, bit for bit)
            self.fuse_decision = bool(fuse_decision)
            self.accept_bits = torch.empty(max(ms_accept_bits_words(self.N), 4), dtype=torch.int32, device=self.device)
            self._bits_offset = None                           # event offset the bits in accept_bits belong to
        if spec.inverse:
            self.d_inv = 3 * spec.n - 4
            self.x_inv = torch.empty((self.d_inv, self.ld), **f64)
            self.w_inv = torch.empty(self.ld, **f64)
            self.r_inv = torch.empty((self.d_inv, self.ld), **f64) if self.d_edges is not None else None

    def set_grid(self, h_edges: np.ndarray) -> None:
        h_edges = np.ascontiguousarray(h_edges, dtype=np.float64)
        if ms_check_grid(h_edges) != 0:
            raise MadSpaceError("ms_check_grid", MS_EGRID)
        self.grid_dims, self.grid_bins = h_edges.shape[0], h_edges.shape[1] - 1
        self._wmax_cached = False                              # a new grid changes every weight, hence w_max
        self._bits_offset = None
        # unused trailing dimensions whose bins all have n_bins * width == 1.0 exactly contribute a Jacobian of exactly 1
        tail = h_edges[self.spec.d_used:]
        self.tail_unit_jacobian = bool(tail.shape[0] > 0 and np.all(self.grid_bins * np.diff(tail, axis=1) == 1.0))
        if hasattr(self, "cfg"):
            self.cfg.tail_unit_jacobian = int(self.tail_unit_jacobian)
        t = torch.from_numpy(h_edges)
        if self.d_edges is None:
            self.d_edges = torch.empty(h_edges.shape, dtype=torch.float64, device=self.device)
        self.d_edges.copy_(t, non_blocking=True)

    # ---- stages -------------------------------------------------------------------------------
    def generate(self, event_offset: int = 0, stream=None) -> None:
        s = self.spec
        if s.unweight and self.fuse_decision:
            self.ensure_wmax(stream)
            with _on(stream):
                ms_generate_unweight(self.cfg, self.N, rng(s.seed_events, 0, event_offset), self.d_edges, self.p, self.w,
                                     self.x1x2, self.ld, self.fail, self.wmax, rng(s.seed_unweight, 1, event_offset),
                                     self.accept_bits, None)
            self._bits_offset = event_offset
            return
        with _on(stream):
            ms_generate(self.cfg, self.N, rng(s.seed_events, 0, event_offset), self.d_edges, self.p, self.w,
                        self.x1x2, self.ld, self.fail, None)
        if s.unweight:
            self._bits_offset = None

    def adapt_grid(self, event_offset: int = 0, alpha: float = 0.5, stream=None) -> np.ndarray:
        """One VEGAS adaptation step from the weights of the last generate(event_offset): accumulate w^2 per bin on the
        device, refine on the host (tiny tables), install the new grid.  Returns the new host edges."""
        if self.d_edges is None:
            raise RuntimeError("adapt_grid needs a grid")
        with _on(stream):
            hist = torch.zeros((self.grid_dims, self.grid_bins), dtype=torch.float64, device=self.device)
            ms_vegas_accumulate(self.N, self.grid_dims, self.grid_bins, self.w, rng(self.spec.seed_events, 0, event_offset),
                                hist, None)
            new_edges = ms_vegas_refine(hist.cpu().numpy(), self.d_edges.cpu().numpy(), alpha)
            self.set_grid(new_edges)
        return new_edges

    def invalidate_wmax(self) -> None:
        """Forget the cached w_max (set_grid does it; call it after changing anything else the weights depend on)."""
        self._wmax_cached = False

    def ensure_wmax(self, stream=None) -> None:
        """w_max = the maximum weight of the pre-run, the GLOBAL events 0..prerun-1 of the event stream (reading R-4;
        BASELINE.json cfg 2: "w_max = max weight of a 2^16-event pre-run"), whatever range a batch or a rank owns.  It is
        a pure function of (spec, grid), so it is computed ONCE per grid -- a deterministic replay of those events into a
        13 MB side buffer, no communication between ranks -- and kept on the device until
        set_grid() / invalidate_wmax(); fail_pre counts the pre-run's failed events."""
        if self._wmax_cached:
            return
        s = self.spec
        with _on(stream):
            if self._pre is None:
                ld = (s.prerun + 1) // 2 * 2
                f64 = dict(dtype=torch.float64, device=self.device)
                self._pre = (torch.empty((s.rows_p, ld), **f64), torch.empty(ld, **f64),
                             torch.empty((2, ld), **f64) if s.pdf else None, ld)
            p_pre, w_pre, x_pre, ld = self._pre
            self.wmax.zero_()
            self.fail_pre.zero_()
            ms_generate(self.cfg, s.prerun, rng(s.seed_events, 0, 0), self.d_edges, p_pre, w_pre, x_pre, ld,
                        self.fail_pre, None)
            ms_reduce_max(s.prerun, w_pre, self.wmax, None)
        self._wmax_cached = True

    def unweight(self, event_offset: int = 0, stream=None) -> None:
        s = self.spec
        self.ensure_wmax(stream)
        rows_n, rows = (s.rows_p, self.p) if self.gather_rows else (0, None)
        with _on(stream):
            if self.fuse_decision and self._bits_offset == event_offset:
                # the generation kernel has decided already: count + scatter only
                ms_unweight_compact(self.N, self.w, self.wmax, self.accept_bits, rows_n, rows, self.cap, self.idx,
                                    self.w_out, self.rows_out, self.n_acc, self.scratch, self.scratch_bytes, self.ld, None)
                return
            ms_unweight(self.N, self.w, self.wmax, rng(s.seed_unweight, 1, event_offset), s.rows_p if self.gather_rows else 0,
                        self.p if self.gather_rows else None, self.cap, self.idx, self.w_out, self.rows_out, self.n_acc,
                        self.scratch, self.scratch_bytes, self.ld, None)

    def invert_phase_space(self, stream=None) -> None:
        with _on(stream):
            ms_fastrambo_inverse(self.N, self.spec.n, self.p, self.x_inv, self.w_inv, self.ld, None)

    def invert_grid(self, stream=None) -> None:
        if self.d_edges is not None:
            # only the dimensions the phase-space map consumed are inverted
            with _on(stream):
                ms_vegas_map(self.N, self.d_inv, self.grid_bins, self.d_edges, 1, self.x_inv, rng(0), self.r_inv, None,
                             self.ld, None)

    def invert(self, stream=None) -> None:
        self.invert_phase_space(stream)
        self.invert_grid(stream)

    def step(self, event_offset: int = 0, stream=None) -> None:
        if self.spec.unweight:
            self.ensure_wmax(stream)
        self.generate(event_offset, stream)
        if self.spec.unweight:
            self.unweight(event_offset, stream)
        if self.spec.inverse:
            self.invert(stream)

    def stages(self):
        """(name, callable(event_offset)) of one step, in order: what bench.py brackets with CUDA events."""
        out = [("generate", lambda off: self.generate(off))]
        if self.spec.unweight:
            out.append(("unweight", lambda off: self.unweight(off)))
        if self.spec.inverse:
            out.append(("fastrambo_inverse", lambda off: self.invert_phase_space()))
            if self.d_edges is not None:
                out.append(("vegas_inverse", lambda off: self.invert_grid()))
        return out

    def capture(self, event_offset: int = 0) -> "torch.cuda.CUDAGraph":
        """One step recorded as a CUDA graph (the library calls neither allocate nor synchronise, so a step is
        capturable as it stands): replay() re-runs it with one launch call, which is what makes sub-wave batches
        (cfg 1: 2^16 events, 4 kernels of ~5-20 us each) launch-latency-free.  The event offset is baked into the graph:
        capture one graph per offset in flight, or use step() for varying offsets."""
        side = torch.cuda.Stream(device=self.device)
        side.wait_stream(torch.cuda.current_stream(self.device))
        with torch.cuda.stream(side):
            self.step(event_offset)                         # warm-up: sets the kernels' shared-memory attributes
        torch.cuda.current_stream(self.device).wait_stream(side)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            self.step(event_offset)
        return g

    def launches(self, event_offset: int = 0) -> int:
        """Kernels of this library enqueued by one step in steady state (w_max cached; memsets/copies not counted)."""
        k = 1
        if self.spec.unweight:
            k += 2                                  # count (or decide) / scatter
        if self.spec.inverse:
            k += 2 if self.d_edges is not None else 1
        return k

    @property
    def launches_per_step(self) -> int:
        return self.launches(0)


class RunningUnweighter:
    """Unweighting against a running maximum weight with an overweight allowance (reading U-2),
    batch by batch on the device: exact weight histogram -> w_max on the host (32768 counts) -> partial unweighting of
    the batch (ms_unweight) -> kept (global index, weight, w_max at the time); finalize() re-unweights the kept events
    against the final maximum.  Marshalling and buffer ownership only: every arithmetic step is a library call."""

    def __init__(self, fraction: float, seed: int, device="cuda:0", n_rows: int = 0):
        self.fraction, self.seed, self.device = float(fraction), int(seed), torch.device(device)
        self.counts = torch.zeros(MS_HIST_BINS, dtype=torch.int64, device=self.device)
        self.w_max = 0.0
        self.trace = []
        self.kept_idx, self.kept_w, self.kept_old, self.kept_rows = [], [], [], []
        self.n_rows = n_rows

    def add_batch(self, w: torch.Tensor, N: int, event_offset: int, rows: Optional[torch.Tensor] = None, ld: int = 0,
                  stream=None) -> int:
        with _on(stream):
            return self._add_batch(w, N, event_offset, rows, ld)

    def _add_batch(self, w, N, event_offset, rows, ld) -> int:
        stream = None                                        # torch's current stream (set by add_batch)
        ms_weight_histogram(N, w, self.counts, stream)
        self.w_max = max(self.w_max, ms_wmax_from_histogram(self.counts.cpu().numpy(), self.fraction))
        self.trace.append(self.w_max)
        f64 = dict(dtype=torch.float64, device=self.device)
        d_wmax = torch.tensor([self.w_max], **f64)
        cap = N
        idx = torch.empty(cap, dtype=torch.int64, device=self.device)
        w_out = torch.empty(cap, **f64)
        n_acc = torch.zeros(1, dtype=torch.int64, device=self.device)
        sb = ms_unweight_scratch_bytes(N)
        scratch = torch.empty(sb, dtype=torch.uint8, device=self.device)
        use_rows = rows is not None and self.n_rows > 0
        rows_out = torch.empty((self.n_rows, cap), **f64) if use_rows else None
        ms_unweight(N, w, d_wmax, rng(self.seed, 1, event_offset), self.n_rows if use_rows else 0, rows if use_rows else None,
                    cap, idx, w_out, rows_out, n_acc, scratch, sb, ld if use_rows else N, stream)
        k = int(n_acc.item())
        self.kept_idx.append(idx[:k] + event_offset)
        self.kept_w.append(w[idx[:k]])                       # gather of the kept weights (indexing, no arithmetic)
        self.kept_old.append(torch.full((k,), self.w_max, **f64))
        if use_rows:
            self.kept_rows.append(rows_out[:, :k])
        return k

    def finalize(self, stream=None):
        """Returns (global indices, output weights, rows or None) of the finally unweighted events."""
        with _on(stream):
            return self._finalize()

    def _finalize(self):
        stream = None                                        # torch's current stream (set by finalize)
        f64 = dict(dtype=torch.float64, device=self.device)
        idx_all = torch.cat(self.kept_idx) if self.kept_idx else torch.empty(0, dtype=torch.int64, device=self.device)
        K = idx_all.numel()
        if K == 0:
            return idx_all, torch.empty(0, **f64), None
        pad = K + (K & 1)
        w_all, old_all = torch.zeros(pad, **f64), torch.zeros(pad, **f64)
        w_all[:K] = torch.cat(self.kept_w)
        old_all[:K] = torch.cat(self.kept_old)
        w_eff = torch.empty(pad, **f64)
        ms_elementwise_max(K, w_all, old_all, w_eff, stream)
        d_wmax = torch.tensor([self.w_max], **f64)
        fin = torch.empty(K, dtype=torch.int64, device=self.device)
        w_out = torch.empty(K, **f64)
        n_acc = torch.zeros(1, dtype=torch.int64, device=self.device)
        sb = ms_unweight_scratch_bytes(K)
        scratch = torch.empty(sb, dtype=torch.uint8, device=self.device)
        ms_unweight(K, w_eff, d_wmax, rng(self.seed, 2, 0), 0, None, K, fin, w_out, None, n_acc, scratch, sb, pad, stream)
        k = int(n_acc.item())
        rows = torch.cat(self.kept_rows, dim=1)[:, fin[:k]] if self.kept_rows else None
        return idx_all[fin[:k]], w_out[:k], rows
