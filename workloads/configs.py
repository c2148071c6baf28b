"""Workload recipes C1..C6 (BASELINE.json configs; PAPER.md:305 for the box).

Every generator is deterministic given its arguments (numpy ``default_rng(seed)``) and returns a
``Workload`` with host numpy arrays.  Nothing here computes any step of the SDM method.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import math

import numpy as np

KERNEL_GOLOVIN = 0
KERNEL_GRAVITATIONAL = 1

# mean volume of the exponential spectrum, vbar = (30.531 um)^3 * 4*pi/3
V_MEAN_BOX = (30.531e-6) ** 3 * 4.0 * math.pi / 3.0
# BASELINE.json config 5: exponential init with mean radius 15 um
V_MEAN_C5 = (15e-6) ** 3 * 4.0 * math.pi / 3.0


@dataclass
class Workload:
    name: str
    xi: np.ndarray          # int64 [n]   multiplicities
    v: np.ndarray           # float64 [n] volumes, m^3
    cell_id: np.ndarray     # int32 [n]
    n_cell: int
    dt: float
    dV: float
    kernel: int             # KERNEL_GOLOVIN / KERNEL_GRAVITATIONAL
    kparam: float           # Golovin: b [1/s]; gravitational: E
    steps: int
    seed: int = 0           # Philox seed of the simulation (BASELINE.json: seed 0)
    notes: dict = field(default_factory=dict)

    @property
    def n_sd(self) -> int:
        return int(self.xi.shape[0])


def _box_state(n_sd: int):
    """PAPER.md:305 + SURVEY.md A25: equal multiplicities, quantile-spaced exponential volumes."""
    total = (2 ** 23) * 10 ** 6            # N0 * V particles
    if total % n_sd != 0:
        raise ValueError("n_sd must divide N0*V = 2^23 * 10^6")
    xi = np.full(n_sd, total // n_sd, dtype=np.int64)
    i = np.arange(n_sd, dtype=np.float64)
    if n_sd > 1:
        q = 1e-5 + i * ((1.0 - 2e-5) / (n_sd - 1))
    else:
        q = np.array([0.5])
    v = -V_MEAN_BOX * np.log1p(-q)
    cell = np.zeros(n_sd, dtype=np.int32)
    return xi, v.astype(np.float64), cell


def golovin_box(n_sd: int = 2 ** 13, steps: int = 3600) -> Workload:
    """C1 / C2: Golovin additive-kernel box, 1 cell, dV=1e6 m^3, b=1500 1/s, dt=1 s."""
    xi, v, cell = _box_state(n_sd)
    return Workload(f"golovin_box_n{n_sd}", xi, v, cell, 1, 1.0, 1e6, KERNEL_GOLOVIN, 1500.0, steps)


def gravitational_box(n_sd: int = 2 ** 20, steps: int = 100) -> Workload:
    """C3: same initial state, gravitational kernel with E=1."""
    xi, v, cell = _box_state(n_sd)
    return Workload(f"gravitational_box_n{n_sd}", xi, v, cell, 1, 1.0, 1e6, KERNEL_GRAVITATIONAL, 1.0, steps)


def grid_poisson(nx: int = 128, ny: int = 128, mean_per_cell: float = 64.0, shuffled: bool = True,
                 steps: int = 600, seed: int = 0) -> Workload:
    """C4: nx*ny cells, per-cell count ~ Poisson(mean), lognormal radii (median 10 um, sigma_g 1.4),
    xi ~ uniform integer in [1e5, 1e7], Golovin b=1500, dV=1e3, dt=1.

    ``shuffled=True`` scatters the droplets of a cell through storage (as after advection);
    ``shuffled=False`` keeps storage cell-contiguous."""
    rng = np.random.default_rng(seed)
    n_cell = nx * ny
    counts = rng.poisson(mean_per_cell, n_cell)
    n = int(counts.sum())
    cell = np.repeat(np.arange(n_cell, dtype=np.int32), counts)
    r = 10e-6 * np.exp(math.log(1.4) * rng.standard_normal(n))
    v = (4.0 * math.pi / 3.0) * r ** 3
    xi = rng.integers(10 ** 5, 10 ** 7, size=n, endpoint=True, dtype=np.int64)
    if shuffled:
        perm = rng.permutation(n)
        cell, v, xi = cell[perm], v[perm], xi[perm]
    return Workload(f"grid{nx}x{ny}_poisson{int(mean_per_cell)}_{'shuffled' if shuffled else 'contig'}",
                    xi, np.ascontiguousarray(v), np.ascontiguousarray(cell), n_cell,
                    1.0, 1e3, KERNEL_GOLOVIN, 1500.0, steps,
                    notes={"count_min": int(counts.min()), "count_max": int(counts.max())})


def grid_uniform(nx: int = 512, ny: int = 512, per_cell: int = 256, steps: int = 100, seed: int = 0,
                 kernel: int = KERNEL_GRAVITATIONAL, shuffled: bool = False) -> Workload:
    """C5: nx*ny cells x per_cell droplets, cell-contiguous storage, exponential volumes with mean
    radius 15 um, xi = 1e6 for every droplet, gravitational kernel E=1, dV=1e3, dt=1."""
    rng = np.random.default_rng(seed)
    n_cell = nx * ny
    n = n_cell * per_cell
    v = rng.standard_exponential(n) * V_MEAN_C5
    # guard the (measure-zero) draw of exactly 0: volumes must be > 0
    np.maximum(v, V_MEAN_C5 * 1e-12, out=v)
    xi = np.full(n, 10 ** 6, dtype=np.int64)
    cell = np.repeat(np.arange(n_cell, dtype=np.int32), per_cell)
    kparam = 1.0 if kernel == KERNEL_GRAVITATIONAL else 1500.0
    if shuffled:                      # storage order after displacement: droplets of a cell scattered
        perm = rng.permutation(n)
        cell, v, xi = np.ascontiguousarray(cell[perm]), np.ascontiguousarray(v[perm]), np.ascontiguousarray(xi[perm])
    return Workload(f"grid{nx}x{ny}x{per_cell}{'_shuffled' if shuffled else ''}", xi, v, cell, n_cell, 1.0, 1e3, kernel,
                    kparam, steps)


def grid_small_multiplicity(nx: int = 64, ny: int = 64, per_cell: int = 32, steps: int = 50,
                            seed: int = 0, shuffled: bool = False) -> Workload:
    """C6 (added for coverage of the update and compaction rows): xi in {1,2,3},
    v = 1, Golovin with b*dt/dV = 0.01 so that p = 0.01*2*xi_max*(n_s-1|1) is about 0.6..1.9:
    exercises gamma > 1, the cap, the equal-multiplicity split, xi -> 0 and real compaction."""
    rng = np.random.default_rng(seed)
    n_cell = nx * ny
    n = n_cell * per_cell
    xi = rng.integers(1, 3, size=n, endpoint=True, dtype=np.int64)
    v = np.ones(n, dtype=np.float64)
    cell = np.repeat(np.arange(n_cell, dtype=np.int32), per_cell)
    if shuffled:
        perm = rng.permutation(n)
        cell, xi = cell[perm], xi[perm]
    return Workload(f"small_xi_grid{nx}x{ny}x{per_cell}_{'shuffled' if shuffled else 'contig'}",
                    xi, v, np.ascontiguousarray(cell), n_cell, 1.0, 1.0, KERNEL_GOLOVIN, 0.01, steps)


def spectrum_bins(n_bins: int = 100, r_min: float = 1e-6, r_max: float = 5e-3):
    """Fig. 6's grid ("ca. 100 bins"; the range is not given): n_bins bins equally spaced in ln r.
    Returns (v_edges[n_bins+1], dlnr[n_bins], r_mid[n_bins]); plain input data for both implementations."""
    ln_edges = np.linspace(math.log(r_min), math.log(r_max), n_bins + 1)
    r_edges = np.exp(ln_edges)
    v_edges = (4.0 * math.pi / 3.0) * r_edges ** 3
    dlnr = np.diff(ln_edges)
    r_mid = np.exp(0.5 * (ln_edges[1:] + ln_edges[:-1]))
    return np.ascontiguousarray(v_edges), np.ascontiguousarray(dlnr), r_mid


def make(name: str, **kw) -> Workload:
    """Named access used by bench.py and the tests: C1..C6."""
    table = {
        "C1": lambda: golovin_box(2 ** 13, **kw),
        "C2a": lambda: golovin_box(2 ** 17, **kw),
        "C2b": lambda: golovin_box(2 ** 20, **kw),
        "C3": lambda: gravitational_box(2 ** 20, **kw),
        "C4": lambda: grid_poisson(**kw),
        "C5": lambda: grid_uniform(**kw),
        "C6": lambda: grid_small_multiplicity(**kw),
    }
    return table[name]()
