"""Seeded synthetic inputs shared by the oracle tests, the GPU tests and bench.py.

Holds NONE of the method's arithmetic: only the five workload descriptions of
BASELINE.json ``configs`` (sizes in SURVEY.md 8.0) and the seeded generators for the
coefficient table and the initial positions.  The recipe:

* coefficient table ``P[Ng][Ng][Ng][M]``, orbital index innermost: config 1 ~U(-1,1) fp64,
  configs 2-5 ~N(0,1) fp32, numpy ``default_rng(1000 + cfg)``;
* initial positions ``[W][N][3]`` ~U[0,L)^3 fp64, numpy ``default_rng(2000 + cfg)``; a crowd
  of W walkers is the first W walkers of the largest crowd of that config;
* Philox key = seed 1, global walker id = walker index.

These stand in for the paper's NiO supercell workloads,
whose orbital files are not available: same shapes (N, M = N/2, table size, walker counts),
random contents.
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import numpy as np


@dataclass(frozen=True)
class Workload:
    cfg: int            # 1..5, BASELINE.json configs[cfg-1]
    name: str
    n_elec: int         # N
    grid: int           # Ng per axis
    box: float          # L
    coef_dtype: str     # "f64" | "f32"
    coef_dist: str      # "uniform" | "normal"
    n_walkers: int      # W (largest crowd for cfg 5)
    tau: float
    delay_rank: int
    sweeps: int
    j2_a: float = 0.5
    j2_b: float = 1.0
    seed: int = 1

    @property
    def n(self) -> int:
        return self.n_elec // 2

    @property
    def n_orb(self) -> int:
        return self.n_elec // 2

    @property
    def table_bytes(self) -> int:
        return self.grid ** 3 * self.n_orb * (8 if self.coef_dtype == "f64" else 4)

    def with_(self, **kw) -> "Workload":
        return replace(self, **kw)


# tau for configs 3-5 and the J2 parameters for 2-5 are not stated in BASELINE.json:
# readings A17 (tau = 0.01, a = 0.5, b = 1).
WORKLOADS = {
    1: Workload(1, "cfg1_tiny_vmc", 8, 16, 5.0, "f64", "uniform", 4, 0.02, 1, 10),
    2: Workload(2, "cfg2_64e", 64, 32, 10.0, "f32", "normal", 256, 0.01, 1, 100),
    3: Workload(3, "cfg3_192e", 192, 48, 14.0, "f32", "normal", 1024, 0.01, 32, 50),
    4: Workload(4, "cfg4_384e", 384, 60, 18.0, "f32", "normal", 2048, 0.01, 32, 20),
    5: Workload(5, "cfg5_768e", 768, 80, 23.0, "f32", "normal", 4096, 0.01, 32, 10),
}
CFG5_CROWD_SIZES = (64, 128, 256, 512, 1024, 2048, 4096)
CFG5_DELAY_RANKS = (1, 16, 32, 64)


def make_coefs(wl: Workload, grid: int | None = None, n_orb: int | None = None) -> np.ndarray:
    """Coefficient table [Ng][Ng][Ng][M] (C order, orbital innermost)."""
    g = wl.grid if grid is None else grid
    m = wl.n_orb if n_orb is None else n_orb
    rng = np.random.default_rng(1000 + wl.cfg)
    shape = (g, g, g, m)
    if wl.coef_dist == "uniform":
        t = rng.uniform(-1.0, 1.0, size=shape)
    else:
        t = rng.standard_normal(size=shape, dtype=np.float32 if wl.coef_dtype == "f32" else np.float64)
    return np.ascontiguousarray(t, dtype=np.float32 if wl.coef_dtype == "f32" else np.float64)


def make_positions(wl: Workload, n_walkers: int | None = None) -> np.ndarray:
    """Initial positions [W][N][3] ~ U[0,L)^3; smaller crowds are prefixes of the largest."""
    rng = np.random.default_rng(2000 + wl.cfg)
    full = rng.uniform(0.0, wl.box, size=(wl.n_walkers, wl.n_elec, 3))
    w = wl.n_walkers if n_walkers is None else n_walkers
    if w > wl.n_walkers:
        extra = np.random.default_rng(3000 + wl.cfg).uniform(0.0, wl.box, size=(w - wl.n_walkers, wl.n_elec, 3))
        full = np.concatenate([full, extra], axis=0)
    return np.ascontiguousarray(full[:w])


def small_workload(n_elec=8, grid=8, box=4.0, coef_dtype="f64", coef_dist="uniform", n_walkers=3,
                   tau=0.02, delay_rank=1, sweeps=2, cfg=0, **kw) -> Workload:
    """Free-form small case for tests (same generators, cfg index 0 unless given)."""
    return Workload(cfg, f"small_{n_elec}e", n_elec, grid, box, coef_dtype, coef_dist, n_walkers, tau,
                    delay_rank, sweeps, **kw)
