"""ms_inputs -- seeded synthetic inputs and workload descriptions shared by the oracle tests,
the CUDA tests and bench.py.

This module holds NONE of the method's arithmetic (no Philox, no maps, no weights): only
the five BASELINE.json workload descriptions and the frozen VEGAS grid tables that both
sides take as *inputs*.  The event uniforms themselves are not generated here: they come
from the counter-based generator that the oracle and the CUDA library each implement
on their own (reading R-2/R-3).

Grid recipe: a *uniform* grid has edges j/n_bins exactly; a
*seeded* grid takes, per dimension, n_bins-1 interior edges = sorted doubles drawn from
numpy's own Philox bit generator (``np.random.Generator(np.random.Philox(key=seed))``),
standing in for the adapted-then-frozen VEGAS grid of PAPER.md:603, :746.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SEED_EVENTS = 1   # reading R-4: phase-space uniforms (Philox stream 0)
SEED_GRID = 2     # VEGAS edge tables (numpy Philox, host side)
SEED_UNWEIGHT = 3  # unweighting uniform (Philox stream 1)
STREAM_EVENTS = 0
STREAM_UNWEIGHT = 1
TOY_REG = 100.0   # (10 GeV)^2 regulator of the toy integrand, BASELINE.json configs[1]
PRERUN = 1 << 16  # w_max = max weight of events 0 .. 2^16-1 of the same stream


def uniform_grid(d: int, n_bins: int) -> np.ndarray:
    e = np.arange(n_bins + 1, dtype=np.float64) / float(n_bins)
    return np.ascontiguousarray(np.tile(e, (d, 1)))


def seeded_grid(d: int, n_bins: int, seed: int = SEED_GRID) -> np.ndarray:
    rng = np.random.Generator(np.random.Philox(key=seed))
    edges = np.empty((d, n_bins + 1), dtype=np.float64)
    for dim in range(d):
        while True:
            inner = np.sort(rng.random(n_bins - 1))
            row = np.concatenate(([0.0], inner, [1.0]))
            if np.all(np.diff(row) > 0.0):
                break
        edges[dim] = row
    return edges


@dataclass(frozen=True)
class Workload:
    name: str
    n: int                     # outgoing particles
    N: int                     # events at full size (BASELINE.json)
    sqrt_s: float              # partonic sqrt(s) (fixed) or hadronic sqrt(s_had) when pdf=True
    grid_dims: int             # VEGAS dimensions (0 = no grid)
    grid_bins: int
    grid_kind: str             # "uniform" | "seeded" | "none"
    mapping: str               # "fastrambo" | "rambo"
    pdf: bool = False
    tau_min: float = 0.0
    masses: tuple = ()
    massive_mode: str = "rescale"   # "rescale": strategy (i), Newton; "reweight": strategy (ii), Eq. 68-69
    toy: bool = False
    unweight: bool = False
    inverse: bool = False
    note: str = ""

    @property
    def d_ps(self) -> int:
        """uniforms consumed by the phase-space map (3n-4; +2 with the x sampling)."""
        return 3 * self.n - 4 + (2 if self.pdf else 0)

    @property
    def d(self) -> int:
        """uniforms drawn per event = grid dimensions if a grid is used, else d_ps."""
        return self.grid_dims if self.grid_dims > 0 else self.d_ps

    def grid(self):
        if self.grid_kind == "uniform":
            return uniform_grid(self.grid_dims, self.grid_bins)
        if self.grid_kind == "seeded":
            return seeded_grid(self.grid_dims, self.grid_bins)
        return None

    @property
    def out_rows(self) -> int:
        return 4 * (self.n + 2) + 1

    @property
    def out_bytes_per_event(self) -> int:
        return 8 * self.out_rows


WORKLOADS = {
    "cfg1": Workload("cfg1", n=3, N=1 << 16, sqrt_s=1000.0, grid_dims=5, grid_bins=64, grid_kind="uniform",
                     mapping="fastrambo", note="massless 2->3 FastRambo, uniform 64x5 grid"),
    "cfg2": Workload("cfg2", n=4, N=1 << 24, sqrt_s=1000.0, grid_dims=8, grid_bins=128, grid_kind="seeded",
                     mapping="fastrambo", toy=True, unweight=True,
                     note="massless 2->4 FastRambo, seeded 128x8 grid, toy integrand, unweighting"),
    "cfg3": Workload("cfg3", n=5, N=1 << 26, sqrt_s=13600.0, grid_dims=15, grid_bins=64, grid_kind="uniform",
                     mapping="rambo", pdf=True, tau_min=(200.0 / 13600.0) ** 2,
                     note="pp 13.6 TeV: tau,y sampling + exact Rambo 2->5 + lab boost, uniform 64x15 grid"),
    "cfg4": Workload("cfg4", n=4, N=1 << 25, sqrt_s=2000.0, grid_dims=0, grid_bins=0, grid_kind="none",
                     mapping="fastrambo", masses=(173.0, 173.0, 0.0, 0.0),
                     note="massive 2->4 (173,173,0,0): FastRambo + Newton rescale"),
    # not a BASELINE.json config: cfg4's process with the paper's own massive strategy
    "cfg4rw": Workload("cfg4rw", n=4, N=1 << 25, sqrt_s=2000.0, grid_dims=0, grid_bins=0, grid_kind="none",
                       mapping="fastrambo", masses=(173.0, 173.0, 0.0, 0.0), massive_mode="reweight",
                       note="massive 2->4 (173,173,0,0): FastRambo with mass reweighting (Eq. 68-69)"),
    "cfg5": Workload("cfg5", n=8, N=1 << 24, sqrt_s=3000.0, grid_dims=20, grid_bins=128, grid_kind="seeded",
                     mapping="fastrambo", toy=True, unweight=True, inverse=True,
                     note="massless 2->8 FastRambo, seeded 128x20 grid, toy integrand, unweighting, round trip"),
}
