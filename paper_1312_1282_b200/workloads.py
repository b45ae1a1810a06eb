"""Seeded synthetic workloads for the He-4 VMC hot path (inputs only).

This module is the ONE place both the CUDA path and the CPU oracle take their
inputs from.  It holds no arithmetic of the method (no u(r), no potential, no
Metropolis step, no Philox): only the numbers that describe a workload -- atom
count, box edge, Jastrow parameter b, walker count, step, seed, the potential's
published constants -- and a seeded generator of liquid-like configurations
used to feed identical coordinates to both sides.

Shapes follow the paper's benchmark workloads (liquid He-4 at
rho = 21.86 nm^-3 in a cubic periodic box, cutoff L/2; l.484: N = 64 ... 1952;
l.527: up to ~10^4 atoms) as fixed by BASELINE.json `configs`.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Tuple

import numpy as np

# --- physical constants handed to both sides as plain numbers -----------------
# HFD-B(HE) "Aziz II" (Ref.[20] l.562).  PAPER.md only names the
# potential; these are the published constants (reading R3), order:
# eps/k [K], r_m [A], A, alpha, beta, c6, c8, c10, D.
AZIZ_HFDB_HE: Tuple[float, ...] = (
    10.948, 2.963, 1.8443101e5, 10.43329537, -2.27965105,
    1.36745214, 0.42123807, 0.17473318, 1.4826,
)
HBAR2_OVER_2M: float = 6.0596     # K*A^2 (BASELINE.json; reading R4)
RHO_EQ: float = 0.02186           # A^-3  ("21.86 nm^-3")
SEED: int = 20131212              # any fixed u64; recorded in DESIGN.md
JITTER: float = 0.05              # A, initial-lattice jitter (BASELINE.json configs)

MODE_FP64 = 0    # fp64 coordinates and arithmetic
MODE_FP32C = 1   # fp32 coordinates + pair arithmetic, fp64 sums


def box_edge(n_atoms: int, rho: float) -> float:
    """Cubic box edge L [A] holding n_atoms at number density rho [A^-3]."""
    return float((n_atoms / rho) ** (1.0 / 3.0))


@dataclass(frozen=True)
class Group:
    """One parameter point: walkers sharing (L, b, step)."""
    rho: float
    b: float
    walkers: int
    step: float      # half-width of the uniform-cube proposal [A], frozen double


@dataclass(frozen=True)
class Workload:
    name: str
    n_atoms: int
    groups: Tuple[Group, ...]
    sweeps: int
    mode: int
    seed: int = SEED
    aziz: Tuple[float, ...] = AZIZ_HFDB_HE
    hbar2_over_2m: float = HBAR2_OVER_2M
    note: str = ""

    @property
    def n_walkers(self) -> int:
        return sum(g.walkers for g in self.groups)

    @property
    def box_L(self) -> List[float]:
        return [box_edge(self.n_atoms, g.rho) for g in self.groups]

    @property
    def jastrow_b(self) -> List[float]:
        return [g.b for g in self.groups]

    @property
    def steps(self) -> List[float]:
        return [g.step for g in self.groups]

    @property
    def walkers_per_group(self) -> List[int]:
        return [g.walkers for g in self.groups]

    def truncated(self, walkers_per_group: int, sweeps: int | None = None) -> "Workload":
        """Same workload with fewer walkers per group (walker w's trajectory does
        not depend on the walker count: counter-based randomness)."""
        gs = tuple(Group(g.rho, g.b, min(g.walkers, walkers_per_group), g.step) for g in self.groups)
        return Workload(self.name + "-trunc", self.n_atoms, gs,
                        self.sweeps if sweeps is None else sweeps, self.mode,
                        self.seed, self.aziz, self.hbar2_over_2m, self.note)


# Steps "tuned to ~50 % acceptance" (BASELINE.json): frozen doubles.  The values
# were found once by bisection on short runs and are part of the workload, so
# both sides receive the same bits.  (rho, b) -> step [A]; see DESIGN.md.
_STEP_TABLE = {
    (0.02186, 2.89): 1.0,
    (0.0196, 2.7): 1.24, (0.0196, 2.8): 1.15, (0.0196, 2.9): 1.07, (0.0196, 3.0): 0.99,
    (0.0219, 2.7): 1.14, (0.0219, 2.8): 1.06, (0.0219, 2.9): 0.98, (0.0219, 3.0): 0.91,
    (0.0240, 2.7): 1.06, (0.0240, 2.8): 0.98, (0.0240, 2.9): 0.91, (0.0240, 3.0): 0.84,
    (0.0262, 2.7): 0.98, (0.0262, 2.8): 0.91, (0.0262, 2.9): 0.84, (0.0262, 3.0): 0.78,
}


def _g(rho: float, b: float, walkers: int) -> Group:
    return Group(rho, b, walkers, _STEP_TABLE[(rho, b)])


def config(index: int) -> Workload:
    """BASELINE.json `configs[index-1]` (1-based, as SURVEY.md numbers them)."""
    if index == 1:
        return Workload("c1-N64", 64, (_g(RHO_EQ, 2.89, 64),), 200, MODE_FP64,
                        note="fp64 throughout; energy every sweep")
    if index == 2:
        return Workload("c2-N256", 256, (_g(RHO_EQ, 2.89, 1024),), 500, MODE_FP64,
                        note="fp64; both kinetic estimators every sweep")
    if index == 3:
        return Workload("c3-N1952", 1952, (_g(RHO_EQ, 2.89, 2048),), 1000, MODE_FP32C,
                        note="paper-scale liquid; fp32 coords, fp64 sums (+ an fp64 run)")
    if index == 4:
        return Workload("c4-N10000", 10000, (_g(RHO_EQ, 2.89, 296),), 100, MODE_FP32C,
                        note="shared-memory capacity stress: 120 KB of fp32 coords per walker")
    if index == 5:
        gs = tuple(_g(rho, b, 1024) for rho in (0.0196, 0.0219, 0.0240, 0.0262)
                   for b in (2.7, 2.8, 2.9, 3.0))
        return Workload("c5-N512-scan", 512, gs, 300, MODE_FP64,
                        note="16 parameter points x 1024 walkers in one launch")
    raise ValueError("config index must be 1..5")


def with_mode(w: Workload, mode: int) -> Workload:
    return Workload(w.name + ("-fp64" if mode == MODE_FP64 else "-fp32c"), w.n_atoms, w.groups,
                    w.sweeps, mode, w.seed, w.aziz, w.hbar2_over_2m, w.note)


def liquid_configuration(n_atoms: int, box_L: float, seed: int, d_min: float = 2.3,
                         fp32_grid: bool = False) -> np.ndarray:
    """Seeded liquid-like configuration: random sequential insertion of points in
    the periodic cube [0,L)^3 keeping every minimum-image pair distance >= d_min
    (a hard-core gas at He-4 liquid density: packing fraction ~0.14, far below
    jamming).  Returns float64 [3][N] (SoA).  With fp32_grid every coordinate is
    x = (k / 2^23) * L with integer k: the grid an fp32 state of the FP32C mode
    holds exactly (it stores 1 + x/L in [1,2)), so both
    sides see the same configuration.  No wavefunction or potential is involved.
    """
    from scipy.spatial import cKDTree  # input structure only

    rng = np.random.default_rng(seed)
    pts = np.empty((0, 3))
    while len(pts) < n_atoms:
        need = n_atoms - len(pts)
        cand = rng.uniform(0.0, box_L, size=(2 * need + 16, 3))
        if fp32_grid:
            cand = np.floor(cand / box_L * 8388608.0) / 8388608.0 * box_L
        cand = cand[(cand >= 0.0).all(1) & (cand < box_L * (1 - 1e-7)).all(1)]
        # drop candidates too close to accepted points
        if len(pts):
            tree = cKDTree(pts, boxsize=box_L)
            d, _ = tree.query(cand, k=1)
            cand = cand[d >= d_min]
        # drop candidates too close to an earlier candidate (greedy, ordered)
        if len(cand) > 1:
            tree = cKDTree(cand, boxsize=box_L)
            pairs = tree.query_pairs(d_min, output_type="ndarray")
            drop = np.zeros(len(cand), bool)
            for i, j in pairs[np.lexsort((pairs[:, 0], pairs[:, 1]))] if len(pairs) else []:
                if not drop[i]:
                    drop[j] = True
            cand = cand[~drop]
        pts = np.vstack([pts, cand[:need]])
    return np.ascontiguousarray(pts.T)


def walker_shard(n_walkers: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous walker range [begin, end) owned by `rank` of `world` processes
    (walkers are independent Markov chains; the walker
    id is part of the Philox counter so sharding does not change any trajectory)."""
    base, rem = divmod(n_walkers, world)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def shard_groups(w: Workload, begin: int, end: int) -> Tuple[List[int], int]:
    """Walkers-per-group of the global walker range [begin, end) of `w` (walkers are numbered group by
    group) and the global id of its first walker.  Groups outside the range get 0 walkers."""
    lo, out = 0, []
    for n in w.walkers_per_group:
        out.append(max(0, min(end, lo + n) - max(begin, lo)))
        lo += n
    return out, begin
