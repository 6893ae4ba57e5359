"""Seeded synthetic inputs for the SDM coalescence step (BASELINE.json configs[0..4]).

This module serves BOTH the oracle-side tests and the CUDA-side tests/bench, and therefore holds
none of the method's arithmetic: it only draws initial super-droplet attributes
(multiplicity xi int64, volume v fp64 [m^3], cell_id int32) with numpy's own generator, following
the recipe in DESIGN.md ("Input recipe", readings R23..R32 of SURVEY.md section 8(c)).  It imports
neither `oracle` nor `paper_2103_17238_b200`.

No public dataset is involved: the paper's workloads are parameterised set-ups (PAPER.md:48-53,
74-75, 112-118) and these inputs take their shapes and distributions.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

GOLOVIN = 0
GEOMETRIC = 1

PHILOX_SEED = 42  # R31 (configs[0] says 42; used everywhere)

# scale = 1.19e5 um^3 = 4/3 pi (30.531 um)^3 ; norm_factor 8.39e12 = 2^23 m^-3 * 1e6 m^3
V0 = 4.0 / 3.0 * math.pi * (30.531e-6) ** 3
N0_PER_M3 = 2.0 ** 23


@dataclasses.dataclass
class Workload:
    name: str
    xi: np.ndarray          # int64[n_sd]
    v: np.ndarray           # float64[n_sd]
    cell_id: np.ndarray     # int32[n_sd]
    n_cell: int
    dt: float
    dV: float
    kernel_kind: int
    b: float                # Golovin coefficient [1/s] (0 for geometric)
    E: float                # geometric collision efficiency (0 for Golovin)
    n_steps: int
    compact_every: int      # 0 = never
    seed: int = PHILOX_SEED

    @property
    def n_sd(self) -> int:
        return int(self.xi.shape[0])

    def copy(self) -> "Workload":
        return dataclasses.replace(self, xi=self.xi.copy(), v=self.v.copy(), cell_id=self.cell_id.copy())


def _rng(config_index: int) -> np.random.Generator:
    return np.random.default_rng(1000 + config_index)  # R31: generator seed = 1000 + config index


def _volume_of_radius(r: np.ndarray) -> np.ndarray:
    return (4.0 / 3.0 * math.pi) * r ** 3


def _bimodal_lognormal_radius(rng, n, med_a, sg_a, med_b, sg_b) -> np.ndarray:
    """R25: each SD picks the small or the large mode with probability 1/2."""
    pick = rng.random(n) < 0.5
    za = rng.standard_normal(n)
    ra = med_a * np.exp(math.log(sg_a) * za)
    rb = med_b * np.exp(math.log(sg_b) * za)
    return np.where(pick, ra, rb)


def _interleave(rng, xi, v, cell_id):
    perm = rng.permutation(xi.shape[0])
    return xi[perm].copy(), v[perm].copy(), cell_id[perm].copy()


def cfg0(n_sd: int = 2 ** 13, n_steps: int = 3600) -> Workload:
    """configs[0]: box, 1 cell, Golovin, deterministic equal-multiplicity sampling (R28)."""
    i = np.arange(n_sd, dtype=np.float64)
    v = -V0 * np.log(1.0 - (i + 0.5) / n_sd)
    total = int(N0_PER_M3 * 1e6)
    xi = np.full(n_sd, total // n_sd, dtype=np.int64)
    cell = np.zeros(n_sd, dtype=np.int32)
    return Workload("cfg0", xi, v, cell, 1, 1.0, 1e6, GOLOVIN, 1500.0, 0.0, n_steps, 0)


def cfg1(n_sd: int = 2 ** 20, n_steps: int = 1000) -> Workload:
    """configs[1]: box, 1 cell, geometric kernel, random multiplicities with mean 2^23*dV/n_sd (R27)."""
    rng = _rng(1)
    mbar = N0_PER_M3 * 1e6 / n_sd
    xi = (1 + np.floor(2.0 * mbar * rng.random(n_sd))).astype(np.int64)
    v = rng.exponential(V0, n_sd)
    v = np.maximum(v, 1e-30)
    cell = np.zeros(n_sd, dtype=np.int32)
    return Workload("cfg1", xi, v, cell, 1, 1.0, 1e6, GEOMETRIC, 0.0, 1.0, n_steps, 0)


def cfg2(n_cell: int = 128 * 128, per_cell: int = 32, n_steps: int = 500, interleave: bool = False) -> Workload:
    """configs[2]: 2D kinematic grid, 32 SDs/cell, bimodal lognormal radii, Golovin (R23, R25, R26)."""
    rng = _rng(2)
    n = n_cell * per_cell
    r = _bimodal_lognormal_radius(rng, n, 0.04e-6, 1.4, 10e-6, 1.3)
    v = _volume_of_radius(r)
    xi = np.maximum(1, np.rint(1e8 * np.exp(0.5 * rng.standard_normal(n)))).astype(np.int64)
    cell = np.repeat(np.arange(n_cell, dtype=np.int32), per_cell)
    if interleave:
        xi, v, cell = _interleave(rng, xi, v, cell)
    return Workload("cfg2", xi, v, cell, n_cell, 1.0, 400.0, GOLOVIN, 1500.0, 0.0, n_steps, 0)


def cfg3(n_cell: int = 256 * 256, per_cell: int = 128, n_steps: int = 200, interleave: bool = False,
         zero_fraction: float = 0.0) -> Workload:
    """configs[3]: 2D grid, 128 SDs/cell, bimodal lognormal, geometric kernel, compaction every step
    (R24).  zero_fraction=0.02 gives the parity-only variant "3z" (R32)."""
    rng = _rng(3)
    n = n_cell * per_cell
    r = _bimodal_lognormal_radius(rng, n, 0.03e-6, 1.6, 12e-6, 1.25)
    v = _volume_of_radius(r)
    xi = rng.integers(10 ** 6, 10 ** 9, size=n, endpoint=True, dtype=np.int64)
    cell = np.repeat(np.arange(n_cell, dtype=np.int32), per_cell)
    if zero_fraction > 0.0:
        xi[rng.random(n) < zero_fraction] = 0
    if interleave:
        xi, v, cell = _interleave(rng, xi, v, cell)
    name = "cfg3z" if zero_fraction > 0.0 else "cfg3"
    return Workload(name, xi, v, cell, n_cell, 1.0, 400.0, GEOMETRIC, 0.0, 1.0, n_steps, 1)


def cfg4(n_cell: int = 2 ** 16, n_steps: int = 200, interleave: bool = False, stress: bool = False,
         max_per_cell: int = 200) -> Workload:
    """configs[4]: irregular occupancy, n_c ~ U{0..200} (both ends inclusive), exponential volumes,
    xi ~ U{1..1e9}, 2 % of each cell's SDs share one multiplicity (R29), Golovin, dt = 0.5 s.
    stress=True gives the parity-only variant "4s": dV = 1 m^3, compaction every 10 steps (R32)."""
    rng = _rng(4)
    counts = rng.integers(0, max_per_cell, size=n_cell, endpoint=True)
    n = int(counts.sum())
    cell = np.repeat(np.arange(n_cell, dtype=np.int32), counts)
    v = np.maximum(rng.exponential(V0, n), 1e-30)
    xi = rng.integers(1, 10 ** 9, size=n, endpoint=True, dtype=np.int64)
    starts = np.concatenate(([0], np.cumsum(counts)))
    shared = rng.integers(1, 10 ** 9, size=n_cell, endpoint=True, dtype=np.int64)
    for c in np.nonzero(counts >= 2)[0]:
        k = max(2, int(round(0.02 * counts[c])))
        sel = starts[c] + rng.choice(counts[c], size=k, replace=False)
        xi[sel] = shared[c]
    if interleave:
        xi, v, cell = _interleave(rng, xi, v, cell)
    dV = 1.0 if stress else 400.0
    return Workload("cfg4s" if stress else "cfg4", xi, v, cell, n_cell, 0.5, dV, GOLOVIN, 1500.0, 0.0,
                    n_steps, 10 if stress else 0)


FULL = {"cfg0": cfg0, "cfg1": cfg1, "cfg2": cfg2, "cfg3": cfg3, "cfg4": cfg4}


def small(name: str, interleave: bool = False) -> Workload:
    """Scaled-down versions of the five configs (same distributions and structure) that the serial
    oracle finishes in seconds yet that span several sort tiles and a ragged tail."""
    if name == "cfg0":
        return cfg0(n_steps=40)
    if name == "cfg1":
        return cfg1(n_sd=40_000 + 123, n_steps=6)
    if name == "cfg2":
        return cfg2(n_cell=37 * 29, per_cell=32, n_steps=6, interleave=interleave)
    if name == "cfg3":
        return cfg3(n_cell=19 * 17, per_cell=128, n_steps=6, interleave=interleave)
    if name == "cfg3z":
        return cfg3(n_cell=19 * 17, per_cell=128, n_steps=6, interleave=interleave, zero_fraction=0.02)
    if name == "cfg4":
        return cfg4(n_cell=401, n_steps=6, interleave=interleave)
    if name == "cfg4s":
        return cfg4(n_cell=401, n_steps=30, interleave=interleave, stress=True)
    raise KeyError(name)


@dataclasses.dataclass
class Shard:
    """One rank's part of a cell-major workload: whole cells [cell_lo, cell_hi), array entries
    [index_base, index_base + work.n_sd).  `work.cell_id` is rebased to start at 0."""
    work: Workload
    rank: int
    world: int
    cell_lo: int
    cell_hi: int
    index_base: int


def shard(w: Workload, rank: int, world: int) -> Shard:
    """Splits a multi-cell, cell-major workload into `world` contiguous cell ranges (cells are
    independent within a step, so ranks exchange nothing).  Pure index bookkeeping: no method arithmetic."""
    if not (0 <= rank < world):
        raise ValueError("rank outside [0, world)")
    if w.n_cell < world:
        raise ValueError("fewer cells than ranks: single-cell boxes do not shard (replicas only)")
    if np.any(np.diff(w.cell_id) < 0):
        raise ValueError("shard() needs cell-major order (non-decreasing cell_id)")
    cell_lo = (w.n_cell * rank) // world
    cell_hi = (w.n_cell * (rank + 1)) // world
    lo = int(np.searchsorted(w.cell_id, cell_lo, side="left"))
    hi = int(np.searchsorted(w.cell_id, cell_hi, side="left"))
    work = dataclasses.replace(w, xi=w.xi[lo:hi].copy(), v=w.v[lo:hi].copy(),
                               cell_id=(w.cell_id[lo:hi] - cell_lo).astype(np.int32), n_cell=cell_hi - cell_lo)
    return Shard(work, rank, world, cell_lo, cell_hi, lo)


def rebase(n_sd_per_rank) -> list:
    """index_base of every rank after a compaction: rank r's first entry is preceded by the survivors of the ranks
    before it (exclusive scan of the per-rank counts -- what an 8-byte all_gather gives every rank).  Pure index
    bookkeeping, R34."""
    bases, acc = [], 0
    for n in n_sd_per_rank:
        if n < 0:
            raise ValueError("negative count")
        bases.append(acc)
        acc += int(n)
    return bases


# ------------------------------------------------------------------------------------------------
# Inputs of the displacement step ("a prescribed single-eddy non-divergent
# flow ... updraft in the left-hand part of the domain, downdraft in the right-hand part").  Input generation only:
# the method's arithmetic (the Euler step, the wrap, the cell index) lives in oracle/ and in csrc/, not here.
def grid_shape(n_cell: int):
    """(nx, nz) of a square 2-D grid with n_cell cells (configs[2]: 128 x 128, configs[3]: 256 x 256)."""
    nx = int(round(math.sqrt(n_cell)))
    if nx * nx != n_cell:
        raise ValueError("not a square grid")
    return nx, nx


def positions_in_cells(cell_id: np.ndarray, nx: int, nz: int, seed: int = 7):
    """Uniformly random positions (grid units) inside the cell every super-droplet is listed in."""
    rng = np.random.default_rng(seed)
    n = cell_id.shape[0]
    x = (cell_id % nx).astype(np.float64) + rng.random(n)
    z = (cell_id // nx).astype(np.float64) + rng.random(n)
    return np.minimum(x, np.nextafter(float(nx), 0.0)), np.minimum(z, np.nextafter(float(nz), 0.0))


def single_eddy(nx: int, nz: int, courant_max: float = 0.5, dt: float = 1.0):
    """Per-cell velocities (grid units per second) of the single-eddy non-divergent flow of the paper's Fig. 2
    set-up: stream function psi = -A sin(pi z / nz) cos(2 pi x / nx), u = -dpsi/dz, w = dpsi/dx at the cell centres,
    scaled so that the largest Courant number |u| dt, |w| dt is `courant_max`.  Updraft on the left, downdraft on
    the right.  Returns (u_cell, w_cell), each float64[nx * nz], row-major like cell_id."""
    xc = (np.arange(nx) + 0.5) / nx
    zc = (np.arange(nz) + 0.5) / nz
    X, Z = np.meshgrid(xc, zc)                      # shape (nz, nx): row = z index
    u = (math.pi / nz) * np.cos(math.pi * Z) * np.cos(2 * math.pi * X) * nz
    w = (2 * math.pi / nx) * np.sin(math.pi * Z) * np.sin(2 * math.pi * X) * nx
    scale = courant_max / (dt * max(np.abs(u).max(), np.abs(w).max()))
    return (u * scale).ravel().copy(), (w * scale).ravel().copy()
