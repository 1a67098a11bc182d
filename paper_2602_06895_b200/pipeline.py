"""HotPath -- device buffers plus the call sequence of one pass of the hot path (what bench.py times and the
tests check).  Marshalling and buffer ownership only: every arithmetic step is a call into the C ABI.

One step = ms_generate (Philox -> VEGAS -> [x1,x2] -> Rambo/FastRambo -> [rescale] -> [boost] -> [toy] -> weight)
           [unweighting: ms_generate_unweight instead -- the hit-or-miss decision against w_max of the pre-run (computed
            once per grid) is taken in the generation kernel -- then ms_unweight_compact (stable compaction)]
           [-> ms_fastrambo_inverse_vegas, or ms_fastrambo_inverse -> ms_vegas_map(inverse)]   (round trip, cfg 5)
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
               ms_unweight_compact, ms_accept_bits_words, ms_gather, ms_fastrambo_inverse_vegas)


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
                 fuse_decision: bool = True, fuse_inverse: bool = True):
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
        # fuse_inverse: the round trip goes momenta -> uniforms in one kernel where ms_fastrambo_inverse_vegas applies
        # (can_fuse_inverse); False keeps ms_fastrambo_inverse + ms_vegas_map (same r_inv, bit for bit)
        self.fuse_inverse = bool(fuse_inverse)
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

    @property
    def can_fuse_inverse(self) -> bool:
        """ms_fastrambo_inverse_vegas serves the round trip: a 64- or 128-bin grid of exactly 3n-4 dimensions on the
        massless FastRambo chain."""
        s = self.spec
        return (self.d_edges is not None and self.grid_dims == 3 * s.n - 4 and self.grid_bins in (64, 128)
                and s.mapping == "fastrambo" and not s.masses and not s.pdf)

    def invert_fused(self, stream=None) -> None:
        """Momenta -> uniforms in one kernel (r_inv, w_inv = weight with the grid's Jacobian); x_inv is not written."""
        with _on(stream):
            ms_fastrambo_inverse_vegas(self.N, self.spec.n, self.p, self.d_edges, self.grid_dims, self.grid_bins, self.r_inv,
                                       self.w_inv, self.ld, None)

    def invert(self, stream=None) -> None:
        if self.fuse_inverse and self.can_fuse_inverse:
            self.invert_fused(stream)
            return
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
            if self.fuse_inverse and self.can_fuse_inverse:
                out.append(("inverse_fused", lambda off: self.invert_fused()))
            else:
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
            k += 1 if (self.fuse_inverse and self.can_fuse_inverse) or self.d_edges is None else 2
        return k

    @property
    def launches_per_step(self) -> int:
        return self.launches(0)


class RunningUnweighter:
    """Unweighting against a running maximum weight with an overweight allowance (reading U-2),
    batch by batch on the device: exact weight histogram -> w_max on the host (32768 counts) -> partial unweighting of
    the batch (ms_unweight) -> kept (global index, weight, w_max at the time, rows); finalize() re-unweights the kept
    events against the final maximum.  Every buffer is allocated once; every step that touches data is a library call
    (ms_weight_histogram, ms_unweight, ms_gather, ms_elementwise_max) or a plain copy / fill; the host reads one count
    per batch and the 256 KB histogram through pinned memory."""

    def __init__(self, fraction: float, seed: int, device="cuda:0", n_rows: int = 0, batch_cap: int = 1 << 20,
                 kept_cap: int = 1 << 20):
        self.fraction, self.seed, self.device = float(fraction), int(seed), torch.device(device)
        self.n_rows = int(n_rows)
        f64 = dict(dtype=torch.float64, device=self.device)
        i64 = dict(dtype=torch.int64, device=self.device)
        self.counts = torch.zeros(MS_HIST_BINS, **i64)
        self.h_counts = torch.zeros(MS_HIST_BINS, dtype=torch.int64).pin_memory()
        self.d_wmax = torch.zeros(2, **f64)
        self.h_wmax = torch.zeros(2, dtype=torch.float64).pin_memory()
        self.n_acc = torch.zeros(2, **i64)
        self.h_nacc = torch.zeros(2, dtype=torch.int64).pin_memory()
        self.w_max = 0.0
        self.trace = []
        self.fill = 0                                        # kept events so far
        self._alloc_batch(int(batch_cap))
        self._alloc_kept(int(kept_cap))

    # ---- buffers ---------------------------------------------------------------------------------
    def _alloc_batch(self, cap: int) -> None:
        cap = (cap + 1) // 2 * 2
        f64 = dict(dtype=torch.float64, device=self.device)
        self.batch_cap = cap
        self.b_idx = torch.empty(cap, dtype=torch.int64, device=self.device)
        self.b_wout = torch.empty(cap, **f64)
        self.b_rows = torch.empty((self.n_rows, cap), **f64) if self.n_rows > 0 else None
        self.scratch_bytes = ms_unweight_scratch_bytes(cap)
        self.scratch = torch.empty(self.scratch_bytes, dtype=torch.uint8, device=self.device)

    def _alloc_kept(self, cap: int) -> None:
        cap = (cap + 1) // 2 * 2
        f64 = dict(dtype=torch.float64, device=self.device)
        i64 = dict(dtype=torch.int64, device=self.device)
        old = (self.kept_idx, self.kept_w, self.kept_old, self.kept_rows) if self.fill > 0 else None
        self.kept_cap = cap
        self.kept_idx = torch.empty(cap, **i64)
        self.kept_w = torch.empty(cap, **f64)
        self.kept_old = torch.empty(cap, **f64)
        self.kept_rows = torch.empty((self.n_rows, cap), **f64) if self.n_rows > 0 else None
        self.w_eff = torch.empty(cap, **f64)
        self.fin = torch.empty(cap, **i64)
        self.f_wout = torch.empty(cap, **f64)
        self.f_idx = torch.empty(cap, **i64)
        self.f_rows = torch.empty((self.n_rows, cap), **f64) if self.n_rows > 0 else None
        self.f_scratch_bytes = ms_unweight_scratch_bytes(cap)
        self.f_scratch = torch.empty(self.f_scratch_bytes, dtype=torch.uint8, device=self.device)
        if old is not None:                                  # growth: plain copies of what was kept
            k = self.fill
            self.kept_idx[:k].copy_(old[0][:k])
            self.kept_w[:k].copy_(old[1][:k])
            self.kept_old[:k].copy_(old[2][:k])
            if self.n_rows > 0:
                self.kept_rows[:, :k].copy_(old[3][:, :k])

    def _read_count(self) -> int:
        self.h_nacc.copy_(self.n_acc, non_blocking=True)
        torch.cuda.current_stream(self.device).synchronize()
        return int(self.h_nacc[0])

    def _set_wmax(self, value: float) -> None:
        self.h_wmax[0] = value
        self.d_wmax.copy_(self.h_wmax, non_blocking=True)

    # ---- batches ----------------------------------------------------------------------------------
    def add_batch(self, w: torch.Tensor, N: int, event_offset: int, rows: Optional[torch.Tensor] = None, ld: int = 0,
                  stream=None) -> int:
        with _on(stream):
            return self._add_batch(w, N, event_offset, rows, ld)

    def _add_batch(self, w, N, event_offset, rows, ld) -> int:
        stream = None                                        # torch's current stream (set by add_batch)
        if N > self.batch_cap:
            self._alloc_batch(N)
        # (1) the exact histogram of all weights so far -> the running maximum (host walk over 32768 counts)
        ms_weight_histogram(N, w, self.counts, stream)
        self.h_counts.copy_(self.counts, non_blocking=True)
        torch.cuda.current_stream(self.device).synchronize()
        self.w_max = max(self.w_max, ms_wmax_from_histogram(self.h_counts.numpy(), self.fraction))
        self.trace.append(self.w_max)
        self._set_wmax(self.w_max)
        # (2) partial unweighting of the batch against it
        use_rows = rows is not None and self.n_rows > 0
        ms_unweight(N, w, self.d_wmax, rng(self.seed, 1, event_offset), self.n_rows if use_rows else 0,
                    rows if use_rows else None, self.batch_cap, self.b_idx, self.b_wout, self.b_rows if use_rows else None,
                    self.n_acc, self.scratch, self.scratch_bytes, ld if use_rows else N, stream)
        k = self._read_count()
        if k == 0:
            return 0
        if self.fill + k > self.kept_cap:
            self._alloc_kept(max(2 * self.kept_cap, self.fill + k))
        # (3) append: kept weight = w[idx], global index = idx + offset (one ms_gather), w_max at the time, rows
        f = self.fill
        ms_gather(k, self.b_idx, 1, w, 0, self.kept_w[f:], self.kept_cap - f, event_offset, self.kept_idx[f:], stream)
        self.kept_old[f:f + k].fill_(self.w_max)
        if use_rows:
            self.kept_rows[:, f:f + k].copy_(self.b_rows[:, :k])
        self.fill = f + k
        return k

    def finalize(self, stream=None):
        """Returns (global indices, output weights, rows or None) of the finally unweighted events (views of buffers this
        object owns: copy them before the next finalize())."""
        with _on(stream):
            return self._finalize()

    def _finalize(self):
        stream = None                                        # torch's current stream (set by finalize)
        K = self.fill
        if K == 0:
            return self.f_idx[:0], self.f_wout[:0], None
        # an event kept with probability min(1, w/w_old) survives with min(1, max(w, w_old)/w_f): the same hit-or-miss
        # test on max(w, w_old) with a fresh uniform stream (stream 2, counter = position in the kept list)
        ms_elementwise_max(K, self.kept_w, self.kept_old, self.w_eff, stream)
        self._set_wmax(self.w_max)
        ms_unweight(K, self.w_eff, self.d_wmax, rng(self.seed, 2, 0), 0, None, self.kept_cap, self.fin, self.f_wout, None,
                    self.n_acc, self.f_scratch, self.f_scratch_bytes, self.kept_cap, stream)
        k = self._read_count()
        if k == 0:
            return self.f_idx[:0], self.f_wout[:0], None
        # global indices (int64 copied as 8-byte words) and rows of the survivors
        ms_gather(k, self.fin, 1, self.kept_idx.view(torch.float64), 0, self.f_idx.view(torch.float64), self.kept_cap, 0, None,
                  stream)
        rows = None
        if self.n_rows > 0:
            ms_gather(k, self.fin, self.n_rows, self.kept_rows, self.kept_cap, self.f_rows, self.kept_cap, 0, None, stream)
            rows = self.f_rows[:, :k]
        return self.f_idx[:k], self.f_wout[:k], rows
