"""The five BASELINE.json configs as plain data (SURVEY.md §8 size table and §8(d) settings)."""
from __future__ import annotations

from dataclasses import dataclass


@dataclass(frozen=True)
class Config:
    name: str
    n: int               # grid points per axis (cubic)
    spacing: float       # A
    solvent: str         # key for workloads.solvent_by_name / workloads.load_chi
    closure: str         # "KH" | "PSE" | "HNC"
    pse_order: int
    mdiis_nvec: int      # M
    mdiis_b: float = 0.5
    mdiis_restart: float = 10.0
    temperature: float = 298.0
    kappa: float = 1.0           # A^-1, Eq. 29-30
    r_min: float = 1e-3          # A, SURVEY.md §8(c) Q11
    rcut: float = 0.0            # <= 0: all pairs; > 0 SURVEY.md §8(c) Q12
    tol: float = 1e-6

    @property
    def n_points(self) -> int:
        return self.n ** 3


CONFIGS = {
    "C1": Config("C1", 32, 0.5, "water", "KH", 1, 5),
    "C2": Config("C2", 64, 0.5, "water", "KH", 1, 5),
    "C3": Config("C3", 128, 0.5, "water_nacl_0.1M", "PSE", 2, 8),
    "C4": Config("C4", 256, 0.375, "water_nacl_0.1M", "KH", 1, 10, rcut=16.0),
    "C5": Config("C5", 512, 0.5, "water_nacl_0.15M", "KH", 1, 5, rcut=16.0),
}


def get_config(name: str) -> Config:
    return CONFIGS[name]
