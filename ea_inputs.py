"""Seeded synthetic inputs shared by the CUDA path's tests/bench and the CPU oracle.

This module holds NONE of the method's arithmetic (no thresholds, no Philox,
no energies): only the workload shapes of BASELINE.json's five configs, the
temperature ladder handed to both sides as plain doubles, and numpy-seeded
+-1 arrays used to exercise ea_set_couplings / ea_set_spins.

The paper uses no dataset: disorder is random by construction
("bimodal with a mean value of zero"), so seeded iid +-1 couplings
with p = 1/2 *are* the paper's workload.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class Config:
    name: str
    L: int
    R: int            # disorder realizations (bits)
    n_temps: int
    T_min: float
    T_max: float
    swap_interval: int
    sweeps: int
    seed: int

    @property
    def N(self) -> int:
        return self.L ** 3

    @property
    def W(self) -> int:
        return (self.R + 31) // 32

    @property
    def attempts_per_sweep(self) -> int:
        return self.N * self.n_temps * self.R


# BASELINE.json "configs".
CONFIGS = {
    1: Config("cfg1_L4", 4, 1, 16, 0.5, 2.0, 1, 1000, 1),
    2: Config("cfg2_L8", 8, 32, 16, 0.5, 2.0, 1, 10_000, 2),
    3: Config("cfg3_L12", 12, 64, 20, 0.6, 2.0, 2, 10_000, 3),
    4: Config("cfg4_L16", 16, 2048, 24, 0.7, 2.0, 1, 100_000, 4),
    5: Config("cfg5_L32", 32, 256, 32, 0.9, 2.0, 1, 10_000, 5),
}


def temperature_ladder(n_temps: int, T_min: float, T_max: float) -> np.ndarray:
    """Geometric ladder, index 0 = coldest, end points exact (R15)."""
    if n_temps == 1:
        return np.array([T_min], dtype=np.float64)
    k = np.arange(n_temps, dtype=np.float64)
    T = T_min * (T_max / T_min) ** (k / (n_temps - 1))
    T[0] = T_min
    T[-1] = T_max
    return T


def betas_for(cfg: Config) -> np.ndarray:
    """beta_k = 1 / T_k as float64; the SAME array object content goes to both paths."""
    return np.ascontiguousarray(1.0 / temperature_ladder(cfg.n_temps, cfg.T_min, cfg.T_max))


def random_pm1(shape, seed: int) -> np.ndarray:
    """iid +-1 int8 with p = 1/2 (numpy PCG64, seeded)."""
    rng = np.random.default_rng(seed)
    return (2 * rng.integers(0, 2, size=shape, dtype=np.int8) - 1).astype(np.int8)


def random_couplings(R: int, N: int, seed: int) -> np.ndarray:
    """J[r][d][site] for ea_set_couplings."""
    return random_pm1((R, 3, N), seed)


def random_spins(R: int, n_temps: int, N: int, seed: int) -> np.ndarray:
    """s[r][slot][site] for ea_set_spins."""
    return random_pm1((R, n_temps, N), seed)
