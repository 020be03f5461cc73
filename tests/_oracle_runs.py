"""Full-size oracle runs for tests/test_gpu_fullsize.py, executed in background processes.

The numpy oracle needs minutes at 128^3 x 4 sites x 50 iterations and at 256^3 x 4 sites x 12 iterations.  So that
the `-m gpu` suite stays within its time limit, tests/conftest.py starts one process per case when the session
begins (only when a CUDA device is present and a test that needs them was selected); the other GPU tests run in the
meantime and the full-size tests join the processes and compare the CUDA path with what they wrote.  Nothing here
touches the CUDA path: a worker imports only `oracle` and `workloads`.

Cases (grid, solvent, closure, MDIIS settings and cutoff exactly as the BASELINE.json config; the solute is a subset
of the config's atoms because the oracle's O(N N_a) setup costs seconds per atom at these grids, and the loop kernels
do not depend on the atom count):
  C3full  C3: 128^3 at 0.5 A, water + 0.1 M NaCl, PSE-2, MDIIS 8, all pairs; the 100 innermost atoms; 50 iterations,
          state also saved after 25.  This case is far from convergence after 50 iterations (rms 2e-3, g up to 650,
          |tau| up to 340) and its MDIIS path amplifies rounding: the worker therefore also runs a TWIN oracle whose
          initial guess is perturbed by one unit in the last place (t * (1 + 2^-52)) and reports how far the twin
          has moved from the oracle after 50 iterations (measured: 1e-8 in g) -- the distance two correct fp64
          implementations of the same arithmetic can be apart at that point.
  C4grid  C4: 256^3 at 0.375 A, water + 0.1 M NaCl, KH, MDIIS 10, rcut 16 A; the first 24 atoms of the chain;
          12 iterations (the history of 10 fills and wraps twice)
  C5grid  C5: 512^3 at 0.5 A, water + 0.15 M NaCl, KH, MDIIS 5, rcut 16 A; the first 3 atoms of the first chain;
          2 iterations (a 512^3 x 4-site oracle iteration takes more than two minutes): the 512-point instantiations
          of every loop kernel, whole grid
"""
from __future__ import annotations

import json
import os
import sys
import time
import traceback

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CASES = {
    "C3full": dict(config="C3", atoms=("innermost", 100), iterations=50, checkpoint=25, twin=True, host_gb=5.0),
    "C4grid": dict(config="C4", atoms=("first", 24), iterations=12, host_gb=22.0),
    "C5grid": dict(config="C5", atoms=("first", 3), iterations=2, host_gb=90.0, disk_gb=16.0, save_phi=False),
}


def case_inputs(name: str):
    """-> (cfg, solvent, sub-solute, (k0, dk, chi), iterations): the inputs both sides of the comparison use."""
    from workloads import Solute, get_config, load_chi, make_solute, solvent_by_name
    case = CASES[name]
    cfg = get_config(case["config"])
    sv = solvent_by_name(cfg.solvent)
    full = make_solute(case["config"])
    how, na = case["atoms"]
    keep = np.argsort(np.linalg.norm(full.xyz, axis=1), kind="stable")[:na] if how == "innermost" else np.arange(na)
    sub = Solute(f"{full.name}_{how}{na}", full.xyz[keep], full.q[keep], full.sigma[keep], full.eps[keep])
    return cfg, sv, sub, load_chi(sv.name), case["iterations"]


def solver_kwargs(cfg) -> dict:
    return dict(closure=cfg.closure, pse_order=cfg.pse_order, mdiis_nvec=cfg.mdiis_nvec, mdiis_b=cfg.mdiis_b,
                mdiis_restart=cfg.mdiis_restart, temperature=cfg.temperature, kappa=cfg.kappa, r_min=cfg.r_min)


def run_case(name: str, outdir: str) -> None:
    """Worker: run the oracle on one case and write G, TAU, W, PHI (.npy) + done.json into outdir."""
    status = {"case": name, "ok": False}
    try:
        if ROOT not in sys.path:
            sys.path.insert(0, ROOT)
        from oracle import rism3d as o3
        cfg, sv, sub, (k0, dk, chi), iters = case_inputs(name)
        t0 = time.perf_counter()
        orc = o3.Rism3dOracle(cfg.n, cfg.spacing, sv.n_v, **solver_kwargs(cfg))
        orc.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
        orc.set_solute(sub.xyz, sub.q, sub.sigma, sub.eps, rcut=cfg.rcut)
        t1 = time.perf_counter()
        np.save(os.path.join(outdir, "W.npy"), orc.get_field("W"))
        if CASES[name].get("save_phi", True):
            np.save(os.path.join(outdir, "PHI.npy"), orc.phi)
        ckpt = CASES[name].get("checkpoint", 0)
        if ckpt:
            orc.iterate(ckpt, 0.0)
            np.save(os.path.join(outdir, "G_ckpt.npy"), orc.get_field("G"))
            np.save(os.path.join(outdir, "TAU_ckpt.npy"), orc.get_field("TAU"))
        orc.iterate(iters - ckpt, 0.0)
        t2 = time.perf_counter()
        g_ref, tau_ref = orc.get_field("G"), orc.get_field("TAU")
        np.save(os.path.join(outdir, "G.npy"), g_ref)
        np.save(os.path.join(outdir, "TAU.npy"), tau_ref)
        if CASES[name].get("twin"):
            # same oracle, initial guess moved by one unit in the last place: its distance from the oracle after the
            # same number of iterations is the rounding sensitivity of the case itself
            twin = o3.Rism3dOracle(cfg.n, cfg.spacing, sv.n_v, **solver_kwargs(cfg))
            twin.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
            twin.set_solute(sub.xyz, sub.q, sub.sigma, sub.eps, rcut=cfg.rcut)
            twin.t = twin.t * (1.0 + 2.0 ** -52)
            twin.iterate(iters, 0.0)
            status.update(twin_dg=float(np.max(np.abs(twin.get_field("G") - g_ref))),
                          twin_dtau=float(np.max(np.abs(twin.get_field("TAU") - tau_ref))))
            del twin
        status.update(ok=True, checkpoint=ckpt, rms_history=[float(r) for r in orc.rms_history], setup_s=t1 - t0, loop_s=t2 - t1,
                      dmu=float(orc.free_energy()[0]))
    except BaseException:                                   # report, never hang the joining test
        status["error"] = traceback.format_exc()
    with open(os.path.join(outdir, "done.json.tmp"), "w") as f:
        json.dump(status, f)
    os.replace(os.path.join(outdir, "done.json.tmp"), os.path.join(outdir, "done.json"))


def host_memory_gb() -> float:
    try:
        import psutil
        return psutil.virtual_memory().available / 1e9
    except Exception:
        return 0.0


if __name__ == "__main__":
    run_case(sys.argv[1], sys.argv[2])
