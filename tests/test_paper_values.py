"""-m "not gpu": statements the paper prints (tests/golden/paper_2403_01039_values.json, each cited) checked against
the oracle and the library's host logic, where they can be checked without the paper's protein data."""
import ctypes as C
import json
import math
import os

import numpy as np
import pytest

from oracle import rism3d as o3
from tests._util import synthetic_chi
from workloads import load_chi, make_solute, water

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_2403_01039_values.json")))


def _solve(n=16, spacing=0.6, tol=1e-9, cfg="C1", **kw):
    sv = water()
    k0, dk, chi = load_chi("water") if n * spacing >= 16 else synthetic_chi(2, sv.rho)
    sol = make_solute(cfg)
    orc = o3.Rism3dOracle(n, spacing, 2, **kw)
    orc.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    orc.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps)
    n_it, rms = orc.iterate(3000, tol)
    assert rms < tol
    return orc, n_it


def test_residual_decays_log_linearly():
    """'The logarithms of the RMS residual decrease almost linearly with increasing number of iterations'
    (324 steps to 1e-6, 552 to 1e-9 for the complex: 76 steps per decade).  Same behaviour of the oracle on C2."""
    g = GOLD["iterations_complex"]
    per_decade_paper = (g["to_1e-9"] - g["to_1e-6"]) / 3.0
    assert 50 < per_decade_paper < 100
    orc, n_it = _solve(n=32, spacing=0.5, tol=1e-9, cfg="C2", mdiis_nvec=10)
    h = np.log10(np.array(orc.rms_history))
    i6 = int(np.argmax(h < -6.0))
    tail = np.arange(i6 // 2, len(h))
    slope, icpt = np.polyfit(tail, h[tail], 1)
    resid = h[tail] - (slope * tail + icpt)
    assert slope < 0.0 and np.std(resid) < 0.35           # within a third of a decade of a straight line
    assert (n_it - i6) > 0.2 * i6                          # going from 1e-6 to 1e-9 costs a comparable share, as in the paper


def test_threshold_1e6_fixes_the_free_energy_to_the_papers_accuracy():
    g = GOLD["sfe_threshold_sensitivity"]
    assert abs(g["abs_kcal_mol"] / g["of_kcal_mol"] - g["relative"]) < 2e-7
    sv = water()
    k0, dk, chi = load_chi("water")
    sol = make_solute("C2")
    mus = []
    for tol in (GOLD["convergence_threshold"]["value"], 1e-9):
        orc = o3.Rism3dOracle(32, 0.5, 2, mdiis_nvec=10)
        orc.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
        orc.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps)
        orc.iterate(3000, tol)
        mus.append(orc.free_energy()[0])
    assert abs(mus[0] - mus[1]) < 2.0 * g["relative"] * abs(mus[1]) + 1e-6


def test_modified_anderson_parameters_of_the_paper():
    g = GOLD["modified_anderson"]
    assert (g["histories"], g["s1"], g["s2"], g["picard_steps_first"]) == (2, 0.2, 0.0, 2)
    its = {}
    # 'in the range 0.2 <= s1 + s2 <= 0.7 ... does not change significantly' is the paper's experience with proteins in
    # NaCl solution; on this small, strongly charged case (Na+ on a 16 A box) the usable window is narrower: s1 = 0.45
    # needs 4x the iterations of s1 = 0.2 and s1 = 0.7 diverges (recorded in DESIGN.md Q17) -- only the lower part
    # of the range is asserted
    for s1 in (g["s1"], 0.3):
        _, its[s1] = _solve(n=32, spacing=0.5, tol=1e-8, accelerator="ANDERSON", mdiis_b=0.6, anderson_s=(s1, g["s2"]))
    assert max(its.values()) < 3.0 * min(its.values())
    _, it_mdiis10 = _solve(n=32, spacing=0.5, tol=1e-8, mdiis_nvec=10)
    assert its[0.2] < 2.5 * it_mdiis10                     # 'comparable to ... MDIIS with 10 subspaces'
    _, it_plain = _solve(n=32, spacing=0.5, tol=1e-8, accelerator="ANDERSON", mdiis_b=0.6, anderson_s=(0.0, 0.0))
    assert it_plain > 2 * its[0.2]                         # the tuning parameter is what 'adapts the Anderson method'


def test_mdiis_memory_at_256_cubed_water():
    """256^3, water (2 site types), MDIIS 10, double precision needs 9 GB in the paper's code; the
    library's workspace for the same problem must not exceed that (it keeps 2M + 3 field-sets + phi, phi~)."""
    from paper_2403_01039_b200 import build as _build
    _build.build(force=False)
    import paper_2403_01039_b200 as lib
    g = GOLD["mdiis_memory_256_water"]
    p = lib.Rism3dParams()
    p.nx = p.ny = p.nz = g["grid"]
    p.spacing, p.n_sites, p.closure, p.pse_order, p.temperature = 0.5, 2, 1, 1, 298.0
    p.mdiis_nvec, p.mdiis_b, p.mdiis_restart, p.kappa, p.r_min = g["subspace"], 0.5, 10.0, 1.0, 1e-3
    nbytes = lib.load_library().rism3d_workspace_bytes(C.byref(p))
    field = g["grid"] ** 3 * 2 * 8
    assert 23 * field < nbytes < g["gigabytes"] * 1e9
    p.accelerator = 1                                      # modified Anderson: 'GPUs in 2010 had a maximum of only 4 GB'
    assert lib.load_library().rism3d_workspace_bytes(C.byref(p)) < 4e9
