"""Writes workloads/chi/<solvent>.npz: the solvent susceptibility chi_{g'g}(k) of the
three solvents the BASELINE.json configs use, from the 1D XRISM solve of oracle/rism1d.py, together with the bulk
isothermal compressibility chi_T (A^3 mol/kcal; enters Eq. 19) and the bulk pressure P of Eq. 20 (kcal/(mol A^3);
enters Eq. 21) of the same solve.

TEST INFRASTRUCTURE.  Calls only `oracle/`; the tables are INPUT DATA of the 3D path, read unchanged by
both the 3D oracle and the CUDA library.

    python -m oracle.make_chi_tables            # all three, ~5 minutes on 8 cores

Settings: XRISM, KH closure, T = 298 K, 16384 radial points at 0.025 A, kappa = 1,
charges ramped 0 -> 1 in seven steps, MDIIS with 10 vectors, b = 0.3, no restart, tolerance 1e-10.
The table keeps k_m = (m + 1) dk_1D up to 16 A^-1 (the 3D grids reach 14.5 A^-1).
"""
from __future__ import annotations

import os
import sys

import numpy as np

from oracle.rism1d import Xrism1d
from workloads import solvent_by_name
from workloads.chi_io import chi_path

RAMP = (0.0, 0.25, 0.5, 0.75, 0.85, 0.95, 1.0)
K_MAX = 16.0


def make(name: str, n_points: int = 16384, dr: float = 0.025, verbose: bool = True):
    sv = solvent_by_name(name)
    x = Xrism1d(sv, temperature=298.0, closure="KH", n_points=n_points, dr=dr, kappa=1.0)
    iters = x.solve_with_charge_ramp(ramp=RAMP, tol=1e-10, nvec=10, b=0.3, restart=0.0, max_iter=3000)
    chi = x.chi_types()
    n_k = int(np.ceil(K_MAX / x.grid.dk)) + 4
    if verbose:
        print(f"{name}: {iters} iterations, n_k = {n_k}, dk = {x.grid.dk:.6f}", flush=True)
    # bulk thermodynamics of the same converged solve: chi_T for Eq. 19, P of Eq. 20 for Eq. 21
    return dict(k0=x.grid.dk, dk=x.grid.dk, chi=np.ascontiguousarray(chi[:n_k]),
                names=np.array(sv.type_names), n_points=n_points, dr=dr, iterations=iters,
                chi_t=x.compressibility(), pressure=x.pressure())


def main(names):
    os.makedirs(os.path.dirname(chi_path("x")), exist_ok=True)
    for name in names:
        np.savez_compressed(chi_path(name), **make(name))


if __name__ == "__main__":
    main(sys.argv[1:] or ["water", "water_nacl_0.1M", "water_nacl_0.15M"])
