"""Seeded synthetic workloads C1..C5 (BASELINE.json `configs`) and the beta ladders of reading R8.

This module holds NO arithmetic of the method: it only names shapes and builds the `betas` arrays that the
harness passes, unchanged, to both the CUDA library and the CPU oracle.  It is the only
module the tests' two sides share, and it belongs to neither: it sits at the repo root, outside the product package and
outside oracle/.  No public dataset is involved: the paper's workloads are random +-J samples
generated in-program; couplings and spins are drawn from `SEED` by each side's own Philox.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

SEED = 200304621


def betas_linear(b_min: float, b_max: float, T: int) -> np.ndarray:
    """beta_t = b_min + (b_max - b_min) * t / (T - 1), evaluated in double in exactly this order (R8)."""
    if T == 1:
        return np.array([b_min], dtype=np.float64)
    return np.array([b_min + (b_max - b_min) * t / (T - 1) for t in range(T)], dtype=np.float64)


def betas_geometric(b_min: float, b_max: float, T: int) -> np.ndarray:
    """beta_t = b_min * pow(b_max / b_min, t / (T - 1)) in double (R8)."""
    if T == 1:
        return np.array([b_min], dtype=np.float64)
    return np.array([b_min * pow(b_max / b_min, t / (T - 1)) for t in range(T)], dtype=np.float64)


def gaussian_couplings_fixed(seed: int, S: int, d: int, N: int, fbits: int = 16, sample_offset: int = 0) -> np.ndarray:
    """Standard-normal couplings rounded to fixed point, int32 [S][d][N], J = Jq * 2^-fbits.  An INPUT of a
    run (a disorder sample), drawn per global sample index with numpy's PCG64 so that shards agree; no arithmetic of the
    method lives here."""
    out = np.empty((S, d, N), dtype=np.int32)
    for s in range(S):
        rng = np.random.default_rng([seed, sample_offset + s, 7])
        out[s] = np.rint(rng.standard_normal((d, N)) * (1 << fbits)).astype(np.int32)
    return out


@dataclass(frozen=True)
class Workload:
    name: str
    d: int
    L: int
    S: int
    T: int
    ladder: str          # "linear" | "geometric"
    b_min: float
    b_max: float
    n_mcs: int
    houdayer: bool
    measure_every: int   # 0 = never

    @property
    def N(self) -> int:
        return self.L ** self.d

    def betas(self) -> np.ndarray:
        f = betas_linear if self.ladder == "linear" else betas_geometric
        return f(self.b_min, self.b_max, self.T)

    def flips_per_sweep(self, S: int | None = None) -> int:
        return (self.S if S is None else S) * 2 * self.T * self.N


# BASELINE.json configs[0..4]; MCS order per PAPER.md:142-147: sweep, (Houdayer), exchange.
C1 = Workload("C1", 2, 8, 4, 8, "linear", 0.2, 2.0, 1000, False, 0)
C2 = Workload("C2", 2, 32, 1024, 32, "geometric", 0.2, 3.0, 10000, True, 0)
C3 = Workload("C3", 3, 8, 2048, 24, "geometric", 0.4, 1.1, 10000, False, 10)
C4 = Workload("C4", 3, 16, 512, 32, "geometric", 0.4, 1.1, 10000, False, 0)
C5 = Workload("C5", 2, 128, 128, 48, "geometric", 0.2, 3.5, 10000, True, 0)
CONFIGS = {w.name: w for w in (C1, C2, C3, C4, C5)}
