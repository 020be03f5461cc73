"""Load a stored solvent-susceptibility table chi_{gamma' gamma}(k).

The tables under `workloads/chi/` are INPUT DATA of the 3D path: they are
written once by `oracle/make_chi_tables.py` (the 1D XRISM solvent solve, oracle-only) and read
unchanged by both the 3D oracle and the CUDA library.  Format: .npz with
  k0, dk   : abscissae k_m = k0 + m*dk  (A^-1)
  chi      : float64 [n_k][n_v][n_v], chi[m][gamma'][gamma]  (gamma' = summed index of Eq. 13)
  names    : site type names
  chi_t    : isothermal compressibility of the bulk solvent, A^3 mol / kcal   (enters Eq. 19)
  pressure : bulk pressure of Eq. 20, kcal / (mol A^3)                        (enters Eq. 21)
"""
from __future__ import annotations

import os

import numpy as np

_DIR = os.path.join(os.path.dirname(os.path.abspath(__file__)), "chi")


def chi_path(solvent_name: str) -> str:
    return os.path.join(_DIR, f"{solvent_name}.npz")


def load_chi(solvent_name: str):
    """-> (k0, dk, chi[n_k][n_v][n_v]) ; raises FileNotFoundError with the regeneration command."""
    p = chi_path(solvent_name)
    if not os.path.exists(p):
        raise FileNotFoundError(
            f"{p} missing: run `python -m oracle.make_chi_tables` (1D solvent solve, CPU oracle)")
    z = np.load(p)
    return float(z["k0"]), float(z["dk"]), np.ascontiguousarray(z["chi"], dtype=np.float64)


def load_solvent_thermo(solvent_name: str):
    """-> (chi_t, pressure) of the bulk solvent, stored beside its chi table by the same 1D solve."""
    z = np.load(chi_path(solvent_name))
    if "chi_t" not in z.files:
        raise KeyError(f"{chi_path(solvent_name)} has no chi_t / pressure: rerun `python -m oracle.make_chi_tables`")
    return float(z["chi_t"]), float(z["pressure"])
