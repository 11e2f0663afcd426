"""Seeded synthetic workloads: BASELINE.json's five configs and the temperature ladders.

This module serves both the CUDA path's tests/bench and the oracle's; it holds none
of the method's arithmetic (no Hamiltonian, no RNG, no thresholds) -- only the
parameters of each workload and the two ladder shapes of SURVEY.md section 8(d):
linear  T_t = Tmin + (Tmax - Tmin) t / (R - 1)   and
geometric T_t = Tmin (Tmax / Tmin)^(t / (R - 1)), computed once in binary64 and handed
identically to both sides.  The paper measures on its own generated disorder
(PAPER.md:68), not on a public dataset; every input here is regenerated from a seed.
"""
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

BIMODAL, GAUSSIAN = 0, 1


def linear_ladder(t_min: float, t_max: float, n: int) -> np.ndarray:
    t = np.arange(n, dtype=np.float64)
    return t_min + (t_max - t_min) * t / float(n - 1)


def geometric_ladder(t_min: float, t_max: float, n: int) -> np.ndarray:
    t = np.arange(n, dtype=np.float64)
    return t_min * np.power(t_max / t_min, t / float(n - 1))


@dataclass(frozen=True)
class Workload:
    name: str
    L: int
    R: int
    J: float
    h: float
    field_kind: int
    ladder: str            # "linear" | "geometric"
    t_min: float
    t_max: float
    sweeps: int
    exchange_every: int
    seeds: tuple           # one seed per disorder realisation (D = len(seeds))
    adapt_trials: int = 0
    adapt_trial_sweeps: int = 0

    @property
    def D(self) -> int:
        return len(self.seeds)

    @property
    def N(self) -> int:
        return self.L ** 3

    def temperatures(self) -> np.ndarray:
        f = linear_ladder if self.ladder == "linear" else geometric_ladder
        return f(self.t_min, self.t_max, self.R)

    def attempts_per_sweep(self) -> int:
        return self.N * self.R * self.D


# BASELINE.json "configs", in order.
CONFIGS = {
    "cfg1": Workload("cfg1", L=8, R=16, J=1.0, h=1.0, field_kind=BIMODAL, ladder="linear",
                     t_min=1.0, t_max=5.0, sweeps=1000, exchange_every=10, seeds=(1,)),
    "cfg2": Workload("cfg2", L=16, R=32, J=1.0, h=1.0, field_kind=GAUSSIAN, ladder="geometric",
                     t_min=1.0, t_max=6.0, sweeps=10000, exchange_every=10, seeds=(2,)),
    "cfg3": Workload("cfg3", L=32, R=64, J=1.0, h=2.0, field_kind=BIMODAL, ladder="linear",
                     t_min=0.8, t_max=6.0, sweeps=10000, exchange_every=5, seeds=(3,),
                     adapt_trials=3, adapt_trial_sweeps=2000),
    "cfg4": Workload("cfg4", L=64, R=128, J=1.0, h=2.0, field_kind=GAUSSIAN, ladder="geometric",
                     t_min=0.8, t_max=6.0, sweeps=10000, exchange_every=10, seeds=(4,)),
    "cfg5": Workload("cfg5", L=32, R=32, J=1.0, h=1.5, field_kind=GAUSSIAN, ladder="geometric",
                     t_min=1.0, t_max=6.0, sweeps=10000, exchange_every=10,
                     seeds=tuple(1000 + d for d in range(32))),
}


def random_spins(L: int, seed: int) -> np.ndarray:
    """A +-1 int8 configuration for set_spins tests (numpy PCG64, not the method's RNG)."""
    rng = np.random.default_rng(seed)
    return (2 * rng.integers(0, 2, size=L ** 3, dtype=np.int8) - 1).astype(np.int8)
