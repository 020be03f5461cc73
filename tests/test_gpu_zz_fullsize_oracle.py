"""-m gpu: the CUDA path against the numpy oracle, element by element over the WHOLE grid, at the kernel
instantiations bench.py times (BASELINE.json north_star: "oracle-matching 3D-RISM convergence at 256^3 x 4 site
types"; tolerance max|dg| <= 1e-9 after a fixed number of iterations).

The oracle runs are tests/_oracle_runs.py's cases, started by tests/conftest.py in background processes when the
session begins; this file is named to run last so that they overlap with the rest of the suite.
  C3full : closure_zfwd<64,..>, fft_strided<128,.>, kspace_x<128,4>, zinv_residual<64,..,MAXO=7> (M = 8, PSE-2);
           1e-9 after 25 iterations; after 50 the bound is what a one-ulp change of the oracle's input does to the oracle
  C4grid : closure_zfwd<128,1,4>, fft_strided<256,.>, kspace_x<256,4>, zinv_residual<128,1,5,9,0> (M = 10, KH,
           rcut 16 A); 12 iterations fill the history of 10 and exercise the drop-oldest path twice
  C5grid : closure_zfwd<256,..>, fft_strided<512,.>, kspace2<512,4> (32 x 16 plan), zinv_residual<256,..> (M = 5, KH,
           rcut 16 A); 2 iterations on the 512^3 grid (the memory-ceiling configuration)
"""
import os

import numpy as np
import pytest

from tests._oracle_runs import case_inputs, solver_kwargs

pytestmark = pytest.mark.gpu


def _run_cuda(name):
    import paper_2403_01039_b200 as lib
    cfg, sv, sub, (k0, dk, chi), iters = case_inputs(name)
    s = lib.Solver(cfg.n, cfg.spacing, sv.n_v, **solver_kwargs(cfg))
    s.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    s.set_solute(sub.xyz, sub.q, sub.sigma, sub.eps, rcut=cfg.rcut)
    return cfg, sv, s, iters


def _compare(name, fullsize_oracle):
    d, status = fullsize_oracle
    cfg, sv, s, iters = _run_cuda(name)
    try:
        # setup fields over the whole grid (S0)
        if os.path.exists(os.path.join(d, "PHI.npy")):
            phi_o = np.load(os.path.join(d, "PHI.npy"), mmap_mode="r")
            assert np.max(np.abs(s.get_field("PHI", 0) - phi_o)) <= 1e-11 * np.max(np.abs(phi_o))
        w_o = np.load(os.path.join(d, "W.npy"), mmap_mode="r")
        for g in range(sv.n_v):
            w, wo = s.get_field("W", g), np.asarray(w_o[g])
            finite = np.abs(wo) < 600.0                       # beyond that exp() underflows on both sides
            assert np.max(np.abs(w - wo)[finite]) <= 1e-10
            assert np.all(w[~finite] < -600.0)
        # the loop (S1-S7), a fixed number of iterations (with a stop on the way where the oracle saved its state)
        ckpt = status.get("checkpoint", 0)
        if ckpt:
            s.iterate(ckpt, 0.0)
            gc_o = np.load(os.path.join(d, "G_ckpt.npy"), mmap_mode="r")
            tc_o = np.load(os.path.join(d, "TAU_ckpt.npy"), mmap_mode="r")
            dgc = max(float(np.max(np.abs(s.get_field("G", g) - gc_o[g]))) for g in range(sv.n_v))
            dtc = max(float(np.max(np.abs(s.get_field("TAU", g) - tc_o[g]))) for g in range(sv.n_v))
            print(f"{name}: after {ckpt} iterations max|dg| = {dgc:.3e}, max|dtau| = {dtc:.3e}")
            assert dgc <= 1e-9 and dtc <= 1e-9
        n_done, rms = s.iterate(iters - ckpt, 0.0)
        assert n_done == iters - ckpt
        hist_o = np.array(status["rms_history"])
        np.testing.assert_allclose(s.rms_history(), hist_o, rtol=1e-6, atol=1e-13)
        g_o = np.load(os.path.join(d, "G.npy"), mmap_mode="r")
        t_o = np.load(os.path.join(d, "TAU.npy"), mmap_mode="r")
        dg = dt = 0.0
        for g in range(sv.n_v):
            dg = max(dg, float(np.max(np.abs(s.get_field("G", g) - g_o[g]))))
            dt = max(dt, float(np.max(np.abs(s.get_field("TAU", g) - t_o[g]))))
        print(f"{name}: {iters} iterations, max|dg| = {dg:.3e}, max|dtau| = {dt:.3e}, rms {rms:.3e} "
              f"(oracle setup {status['setup_s']:.0f} s, loop {status['loop_s']:.0f} s)")
        # north_star: max|dg| <= 1e-9.  Where the case itself moves further than that under a one-ulp change of the
        # oracle's own input (twin run, tests/_oracle_runs.py), that distance is the bound
        bound_g, bound_t = max(1e-9, status.get("twin_dg", 0.0)), max(1e-9, status.get("twin_dtau", 0.0))
        if "twin_dg" in status:
            print(f"{name}: one-ulp twin of the oracle: max|dg| = {status['twin_dg']:.3e}, max|dtau| = {status['twin_dtau']:.3e}")
        assert dg <= bound_g and dt <= bound_t
        mu, _ = s.free_energy()                               # Eq. 18 of the unconverged state: same grid sum
        assert abs(mu - status["dmu"]) <= 1e-7 * max(1.0, abs(status["dmu"]))
    finally:
        s.close()


@pytest.mark.fullsize_oracle("C3full")
def test_c3_full_grid_fifty_iterations_match_oracle(fullsize_oracle):
    _compare("C3full", fullsize_oracle)


@pytest.mark.fullsize_oracle("C4grid")
def test_c4_grid_twelve_iterations_match_oracle(fullsize_oracle):
    _compare("C4grid", fullsize_oracle)


@pytest.mark.fullsize_oracle("C5grid")
def test_c5_grid_two_iterations_match_oracle(fullsize_oracle):
    _compare("C5grid", fullsize_oracle)
