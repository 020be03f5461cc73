"""-m gpu: the CUDA path at BASELINE.json's full C4 size (256^3 x 4 sites, KH, MDIIS 10, rcut 16 A), in the launch
configuration bench.py times.  The oracle cannot run the 256^3 loop in seconds, so this compares what it can compute
point by point (potential, long-range function, closure at sampled grid points -- all atoms, its own cutoff rule)
and checks properties that hold at any size (fixed point reached, run-to-run bit reproducibility of the reductions,
spectrum of sampled k points from the defining sum)."""
import numpy as np
import pytest

from oracle import rism3d as o3
from workloads import get_config, load_chi, make_solute, solvent_by_name

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def c4():
    import paper_2403_01039_b200 as lib
    cfg = get_config("C4")
    sv = solvent_by_name(cfg.solvent)
    sol = make_solute("C4")
    k0, dk, chi = load_chi(sv.name)
    s = lib.Solver(cfg.n, cfg.spacing, sv.n_v, closure=cfg.closure, pse_order=cfg.pse_order, mdiis_nvec=cfg.mdiis_nvec,
                   mdiis_b=cfg.mdiis_b, mdiis_restart=cfg.mdiis_restart)
    s.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    s.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps, rcut=cfg.rcut)
    yield cfg, sv, sol, s
    s.close()


def _sample_points(cfg, sol, rng, n_rand=300, n_near=300):
    """grid indices: uniform ones plus ones close to atoms (where the potential is steep)"""
    n = cfg.n
    idx = rng.integers(0, n, size=(n_rand, 3))
    atoms = sol.xyz[rng.integers(0, sol.n_atoms, size=n_near)]
    near = np.rint((atoms + rng.uniform(-3.0, 3.0, size=(n_near, 3))) / cfg.spacing).astype(int) + n // 2
    return np.clip(np.vstack([idx, near]), 0, n - 1)


def test_c4_setup_fields_at_sampled_points(c4):
    cfg, sv, sol, s = c4
    rng = np.random.default_rng(44)
    idx = _sample_points(cfg, sol, rng)
    pts = (idx - cfg.n // 2) * cfg.spacing
    beta = 1.0 / (o3.K_BOLTZMANN * cfg.temperature)
    w_o = o3.w_short_at(pts, sol.xyz, sol.q, sol.sigma, sol.eps, sv.q, sv.sigma, sv.eps, beta, cfg.r_min, cfg.kappa,
                        cfg.rcut)
    phi_o = o3.phi_at(pts, sol.xyz, sol.q, beta, cfg.kappa)
    phi = s.get_field("PHI", 0)[idx[:, 0], idx[:, 1], idx[:, 2]]
    assert np.max(np.abs(phi - phi_o)) < 1e-11 * np.max(np.abs(phi_o))
    for g in range(sv.n_v):
        w = s.get_field("W", g)[idx[:, 0], idx[:, 1], idx[:, 2]]
        finite = np.abs(w_o[g]) < 600.0
        assert finite.sum() > 300
        assert np.max(np.abs(w - w_o[g])[finite]) < 1e-9 * np.maximum(1.0, np.abs(w_o[g][finite])).max()
        assert np.all(w[~finite] < -600.0)


def test_c4_loop_properties_and_reproducibility(c4):
    cfg, sv, sol, s = c4
    n_done, rms = s.iterate(25, 0.0)
    assert n_done == 25 and np.isfinite(rms)
    hist1 = s.rms_history().copy()
    tau1 = s.get_field("TAU", 1)
    # closure identity at sampled points: G = closure(W + TAU) with the oracle's closure
    rng = np.random.default_rng(45)
    idx = _sample_points(cfg, sol, rng, 200, 200)
    for g in (0, 3):
        w = s.get_field("W", g)[idx[:, 0], idx[:, 1], idx[:, 2]]
        t = s.get_field("TAU", g)[idx[:, 0], idx[:, 1], idx[:, 2]]
        gg = s.get_field("G", g)[idx[:, 0], idx[:, 1], idx[:, 2]]
        expect = o3.closure_g(w + t, cfg.closure, cfg.pse_order)
        assert np.max(np.abs(gg - expect)) < 1e-12 * max(1.0, expect.max())
    # same solve again: every reduction runs in a fixed order, so the history is bit-identical
    s.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps, rcut=cfg.rcut)
    s.iterate(25, 0.0)
    assert np.array_equal(s.rms_history(), hist1)
    assert np.array_equal(s.get_field("TAU", 1), tau1)
    # 25 iterations in one call == 10 + 15 in two calls (the pending update is applied between calls)
    s.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps, rcut=cfg.rcut)
    s.iterate(10, 0.0)
    s.iterate(15, 0.0)
    assert np.array_equal(s.rms_history(), hist1)
    assert np.array_equal(s.get_field("TAU", 1), tau1)


def test_c4_converges_to_a_fixed_point(c4):
    cfg, sv, sol, s = c4
    s.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps, rcut=cfg.rcut)
    n_done, rms = s.iterate(1500, cfg.tol)
    assert rms < cfg.tol and n_done < 1000
    hist = s.rms_history()
    assert len(hist) == n_done and hist[-1] == rms and np.all(hist[:-1] >= cfg.tol)
    mu, site = s.free_energy()
    assert np.isfinite(mu) and abs(site.sum() - mu) < 1e-9 * abs(mu)
    g = s.get_field("G", 0)
    assert g.min() >= 0.0 and abs(np.median(g) - 1.0) < 0.05
    # one more pass of the map from the converged input leaves it (almost) where it is: its residual is < tol too
    tau = [s.get_field_device("TAU", k).clone() for k in range(sv.n_v)]
    for k in range(sv.n_v):
        s.set_tau(k, tau[k])                 # warm start: clears the history, keeps tau
    n2, rms2 = s.iterate(1, 0.0)
    assert n2 == 1 and rms2 < 1.5 * cfg.tol


# ---- C5: 512^3 x 4 sites, 20 000 atoms, 54 GB workspace (the single-GPU memory ceiling of BASELINE.json) ----------
def test_c5_memory_ceiling_setup_and_first_iterations():
    import time
    import torch
    import paper_2403_01039_b200 as lib
    cfg = get_config("C5")
    sv = solvent_by_name(cfg.solvent)
    free, total = torch.cuda.mem_get_info()
    s = None
    try:
        s = lib.Solver(cfg.n, cfg.spacing, sv.n_v, closure=cfg.closure, mdiis_nvec=cfg.mdiis_nvec, mdiis_b=cfg.mdiis_b,
                       mdiis_restart=cfg.mdiis_restart)
    except torch.OutOfMemoryError:
        pytest.skip(f"needs {54} GB of device memory, {free / 1e9:.0f} GB free")
    assert 50e9 < s.workspace.numel() < 60e9             # (2M + 3) field-sets of 4.29 GB + phi, phi~
    sol = make_solute("C5")
    k0, dk, chi = load_chi(sv.name)
    s.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    s.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps, rcut=cfg.rcut)
    # sampled setup fields against the oracle (64-bit offsets: site 3 starts 3.2e9 bytes into the field-set)
    rng = np.random.default_rng(55)
    idx = _sample_points(cfg, sol, rng, 150, 150)
    pts = (idx - cfg.n // 2) * cfg.spacing
    beta = 1.0 / (o3.K_BOLTZMANN * cfg.temperature)
    w_o = o3.w_short_at(pts, sol.xyz, sol.q, sol.sigma, sol.eps, sv.q, sv.sigma, sv.eps, beta, cfg.r_min, cfg.kappa,
                        cfg.rcut)
    phi_o = o3.phi_at(pts, sol.xyz, sol.q, beta, cfg.kappa)
    phi = s.get_field_device("PHI", 0)[idx[:, 0], idx[:, 1], idx[:, 2]].cpu().numpy()
    assert np.max(np.abs(phi - phi_o)) < 1e-10 * np.max(np.abs(phi_o))
    for g in (0, 3):
        w = s.get_field_device("W", g)[idx[:, 0], idx[:, 1], idx[:, 2]].cpu().numpy()
        finite = np.abs(w_o[g]) < 600.0
        assert np.max(np.abs(w - w_o[g])[finite]) < 1e-9 * np.maximum(1.0, np.abs(w_o[g][finite])).max()
    # the loop runs, the residual falls, and G = closure(W + TAU) at sampled points
    n_done, rms = s.iterate(12, 0.0)
    hist = s.rms_history()
    assert n_done == 12 and np.all(np.isfinite(hist)) and hist[-1] < 0.5 * hist[0]
    for g in (1, 2):
        w = s.get_field_device("W", g)[idx[:, 0], idx[:, 1], idx[:, 2]].cpu().numpy()
        t = s.get_field_device("TAU", g)[idx[:, 0], idx[:, 1], idx[:, 2]].cpu().numpy()
        gg = s.get_field_device("G", g)[idx[:, 0], idx[:, 1], idx[:, 2]].cpu().numpy()
        expect = o3.closure_g(w + t, cfg.closure, cfg.pse_order)
        assert np.max(np.abs(gg - expect)) < 1e-12 * max(1.0, expect.max())
    s.close()
