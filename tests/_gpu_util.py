"""Helpers shared by the -m gpu parity tests: build an oracle and a CUDA solver from the same inputs."""
import numpy as np

from oracle import rism3d as o3
from workloads import get_config, load_chi, make_solute, solvent_by_name


def make_pair(cfg_name=None, *, n=None, spacing=None, solvent="water", closure="KH", pse_order=1, M=5, b=0.5,
              restart=10.0, chi=None, solute=None, rcut=0.0, origin=None, n_override=None, accelerator="MDIIS",
              anderson_s=(0.2, 0.0), kappa=1.0, **extra):
    """-> (oracle, cuda solver, solute, rcut) with identical settings.  cfg_name picks a BASELINE config;
    n_override shrinks its grid (same spacing) so the oracle stays fast."""
    import paper_2403_01039_b200 as lib
    if cfg_name is not None:
        cfg = get_config(cfg_name)
        n = n_override or cfg.n
        spacing, solvent, closure, pse_order = cfg.spacing, cfg.solvent, cfg.closure, cfg.pse_order
        M, b, restart, rcut = cfg.mdiis_nvec, cfg.mdiis_b, cfg.mdiis_restart, cfg.rcut
        solute = make_solute(cfg_name)
    sv = solvent_by_name(solvent) if isinstance(solvent, str) else solvent
    k0, dk, table = load_chi(sv.name) if chi is None else chi
    orc = o3.Rism3dOracle(n, spacing, sv.n_v, closure=closure, pse_order=pse_order, mdiis_nvec=M, mdiis_b=b,
                          mdiis_restart=restart, origin=origin, accelerator=accelerator, anderson_s=anderson_s,
                          kappa=kappa, **extra)
    orc.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, table)
    gpu = lib.Solver(n, spacing, sv.n_v, closure=closure, pse_order=pse_order, mdiis_nvec=M, mdiis_b=b,
                     mdiis_restart=restart, origin=origin, accelerator=accelerator, anderson_s=anderson_s,
                     kappa=kappa, **extra)
    gpu.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, table)
    if solute is not None:
        orc.set_solute(solute.xyz, solute.q, solute.sigma, solute.eps, rcut=rcut)
        gpu.set_solute(solute.xyz, solute.q, solute.sigma, solute.eps, rcut=rcut)
    return orc, gpu, solute, rcut


def oracle_spectrum_in_gpu_layout(f, spacing):
    """Oracle forward transform of a real field [n_v][n][n][n] in the library's k-space layout
    [jx][jy][p][site] (p <-> j_z = 2p), without the dV factor and with the origin at grid index 0."""
    F = o3.shifted_dft_forward(f, spacing, (0.0, 0.0, 0.0)) / spacing ** 3
    return np.ascontiguousarray(np.moveaxis(F[:, :, :, 0::2], 0, -1))
