"""Seeded synthetic inputs for the 3D-RISM hot path (BASELINE.json `configs`).

This package serves BOTH the CPU oracle (through the tests) and the CUDA path (tests, bench.py,
smoke()).  It holds only *input data*: solute atom lists, solvent site parameters, grid / solver
settings of the five configs, and loaders for the stored solvent-susceptibility tables under
`workloads/chi/` (written by `oracle/make_chi_tables.py`).  None of the method's arithmetic lives
here, and it imports neither `oracle` nor `paper_2403_01039_b200`.

The paper's own workload (RBD-ACE2, 12 877 atoms) is not available; these inputs take
its shape (atom count, net charge, 4 solvent site types, 256^3-512^3 grids) and stand in for it.
"""
from .solvents import Solvent, water, water_nacl, solvent_by_name
from .solutes import Solute, make_solute
from .configs import Config, CONFIGS, get_config
from .chi_io import load_chi, load_solvent_thermo, chi_path

__all__ = [
    "Solvent", "water", "water_nacl", "solvent_by_name",
    "Solute", "make_solute",
    "Config", "CONFIGS", "get_config",
    "load_chi", "load_solvent_thermo", "chi_path",
]
