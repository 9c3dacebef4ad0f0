"""Seeded synthetic workloads: the five BASELINE.json configs and the temperature ladder.

This module is the only thing the CPU oracle's tests and the CUDA path's tests share.  It
holds NO arithmetic of the method (no RNG, no thresholds, no update rule): a config is a
tuple of plain parameters, and the ladder is computed here ONCE and handed as the same
doubles to both sides (R15), so `pow` is never evaluated on two sides.

The paper's workloads use no dataset: couplings are i.i.d. +-1, the field is a
constant and the ladder is geometric (Table I caption).
"""
from dataclasses import dataclass, replace
from typing import Tuple

PMJ, GAUSS = 0, 1


@dataclass(frozen=True)
class Workload:
    name: str
    L: int
    n_samples: int
    kind: int
    seed: int
    h: float
    n_replicas: int
    n_temps: int
    T_lo: float
    T_hi: float
    n_sweeps: int
    pt_every: int
    meas_every: int

    @property
    def N(self) -> int:
        return self.L ** 3

    @property
    def n_words(self) -> int:
        return (self.n_samples + 31) // 32

    def temps(self) -> Tuple[float, ...]:
        return ladder(self.T_lo, self.T_hi, self.n_temps)

    def flip_attempts(self, n_sweeps: int = None) -> int:
        """Active-lane spin-flip attempts: N * samples * R * N_T * sweeps."""
        k = self.n_sweeps if n_sweeps is None else n_sweeps
        return self.N * self.n_samples * self.n_replicas * self.n_temps * k

    def scaled(self, **kw) -> "Workload":
        return replace(self, **kw)


def ladder(T_lo: float, T_hi: float, n: int) -> Tuple[float, ...]:
    """Geometric ladder T_t = T_lo * (T_hi/T_lo)^(t/(n-1)), slot 0 coldest."""
    if n == 1:
        return (float(T_lo),)
    out = [float(T_lo) * (float(T_hi) / float(T_lo)) ** (t / (n - 1)) for t in range(n)]
    out[0], out[-1] = float(T_lo), float(T_hi)
    return tuple(out)


# BASELINE.json "configs", in order.  meas_every where the config is silent: DESIGN.md R16.
CONFIGS = (
    Workload("C1", 4, 1, PMJ, 1, 0.3, 4, 8, 0.5, 2.0, 1000, 1, 10),
    Workload("C2", 8, 2048, PMJ, 2, 0.2, 4, 20, 0.5, 2.0, 1 << 14, 1, 16),
    Workload("C3", 12, 4096, PMJ, 3, 0.1, 4, 24, 0.4, 1.8, 1 << 15, 1, 16),
    Workload("C4", 16, 512, GAUSS, 4, 0.3, 4, 32, 0.2, 1.5, 1 << 13, 1, 16),
    Workload("C5", 32, 8192, PMJ, 5, 0.2, 4, 32, 0.4, 2.0, 1024, 4, 0),
)
BY_NAME = {w.name: w for w in CONFIGS}
