"""-m gpu: edge and degenerate cases of the CUDA path against the oracle -- smallest grid, 1 and 8 site types, HNC,
high PSE order, shifted origin, empty solute, MDIIS restart actually firing, M = 16, divergence reporting, warm
start, and the split-call / trailing-update logic of rism3d_iterate."""
import numpy as np
import pytest

from oracle import rism3d as o3
from tests._gpu_util import make_pair
from tests._util import synthetic_chi
from workloads import Solute, Solvent, make_solute, water

pytestmark = pytest.mark.gpu


def _solvent(n_v, seed=0):
    """made-up neutral solvent of n_v monatomic species (inputs only)"""
    rng = np.random.default_rng(seed)
    q = rng.uniform(-0.6, 0.6, n_v)
    rho = rng.uniform(0.005, 0.02, n_v)
    if n_v == 1:
        q[:] = 0.0
    else:
        q[-1] = -np.dot(rho[:-1], q[:-1]) / rho[-1]          # sum rho q = 0
    return Solvent(name=f"syn{n_v}", type_names=[f"S{i}" for i in range(n_v)], q=q, sigma=rng.uniform(2.5, 3.5, n_v),
                   eps=rng.uniform(0.05, 0.2, n_v), rho=rho, mult=np.ones(n_v, int), site_type=np.arange(n_v),
                   site_species=np.arange(n_v), species_rho=rho, bond=np.zeros((n_v, n_v)))


def _small_solute(seed=1, n=3, charged=True):
    rng = np.random.default_rng(seed)
    xyz = rng.uniform(-1.5, 1.5, (n, 3))
    q = rng.normal(0.0, 0.3, n) if charged else np.zeros(n)
    return Solute("edge", xyz, q, rng.uniform(2.6, 3.4, n), rng.uniform(0.05, 0.2, n))


@pytest.mark.parametrize("n_v,n", [(1, 16), (8, 16), (2, 8), (4, 8), (3, 16), (5, 16), (6, 8), (7, 16)])
def test_site_counts_and_smallest_grids(n_v, n):
    """every site count 1..8 (3, 5, 6, 7 run padded with phantom types inside the library) on the smallest grids"""
    sv = _solvent(n_v, seed=n_v)
    chi = synthetic_chi(n_v, sv.rho, n_k=900, dk=0.02, k0=0.02, seed=n_v, amp=0.5)
    orc, gpu, _, _ = make_pair(n=n, spacing=0.9, solvent=sv, chi=chi, solute=_small_solute(), M=4)
    orc.iterate(20, 0.0)
    nd, rms = gpu.iterate(20, 0.0)
    assert nd == 20 and abs(rms - orc.rms_history[-1]) <= 1e-9 * orc.rms_history[-1] + 1e-13
    assert np.max(np.abs(gpu.get_field("G") - orc.get_field("G"))) <= 1e-9
    mu_o, site_o = orc.free_energy()
    mu_g, site_g = gpu.free_energy()
    assert abs(mu_g - mu_o) <= 1e-9 * max(1.0, abs(mu_o))
    assert site_g.shape == (n_v,) and np.allclose(site_g, site_o, rtol=1e-8, atol=1e-9 * max(1.0, abs(mu_o)))
    assert gpu.get_field("TAU").shape == (n_v, n, n, n)


def test_three_site_solvent_modified_anderson_and_fft_hooks():
    """n_v = 3 (padded to 4): the 1/rho-weighted inner product of the modified Anderson method must ignore the phantom
    type, the rms must be normalised with the caller's site count, and the debug transform hooks pad and unpad."""
    import torch
    from tests._gpu_util import oracle_spectrum_in_gpu_layout
    sv = _solvent(3, seed=3)
    chi = synthetic_chi(3, sv.rho, n_k=900, dk=0.02, k0=0.02, seed=3, amp=0.5)
    orc, gpu, _, _ = make_pair(n=16, spacing=0.9, solvent=sv, chi=chi, solute=_small_solute(), b=0.5, accelerator="ANDERSON")
    orc.iterate(25, 0.0)
    gpu.iterate(25, 0.0)
    np.testing.assert_allclose(gpu.rms_history(), orc.rms_history, rtol=1e-7, atol=1e-14)
    assert np.max(np.abs(gpu.get_field("G") - orc.get_field("G"))) <= 1e-9
    f = np.random.default_rng(5).standard_normal((3, 16, 16, 16))
    spec = gpu.fft_forward(torch.from_numpy(f).cuda())
    ref = oracle_spectrum_in_gpu_layout(f, 0.9)
    assert spec.shape == ref.shape and np.max(np.abs(spec.cpu().numpy() - ref)) < 1e-12 * np.max(np.abs(ref))
    assert np.max(np.abs(gpu.fft_inverse(spec).cpu().numpy() - f)) < 1e-12


@pytest.mark.parametrize("closure,order", [("HNC", 1), ("PSE", 3), ("PSE", 7)])
def test_other_closures(closure, order):
    sol = _small_solute(seed=3, n=4)
    sol = Solute("weak", sol.xyz, 0.3 * sol.q, sol.sigma, sol.eps)        # HNC: keep exp() tame
    orc, gpu, _, _ = make_pair(n=32, spacing=0.5, solvent="water", closure=closure, pse_order=order, solute=sol, M=5)
    orc.iterate(30, 0.0)
    gpu.iterate(30, 0.0)
    g, go = gpu.get_field("G"), orc.get_field("G")
    assert np.max(np.abs(g - go) / np.maximum(1.0, go)) <= 1e-9
    mu_o, _ = orc.free_energy()
    mu_g, _ = gpu.free_energy()
    assert abs(mu_g - mu_o) <= 1e-8 * max(1.0, abs(mu_o))


def test_shifted_origin():
    """origin not at -(n/2) dr and not a multiple of dr: only R_a - r0 enters (Q13)"""
    orc, gpu, _, _ = make_pair(n=32, spacing=0.5, solvent="water", solute=_small_solute(seed=5),
                               origin=(-7.3, -8.1, -8.65))
    orc.iterate(20, 0.0)
    gpu.iterate(20, 0.0)
    assert np.max(np.abs(gpu.get_field("G") - orc.get_field("G"))) <= 1e-9
    assert np.max(np.abs(gpu.get_field("PHI", 0) - orc.phi)) <= 1e-11 * np.max(np.abs(orc.phi))


def test_empty_solute():
    import paper_2403_01039_b200 as lib
    from workloads import load_chi
    sv = water()
    k0, dk, chi = load_chi("water")
    s = lib.Solver(16, 0.5, 2)
    s.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    s.set_solute(np.zeros((0, 3)), [], [], [])
    nd, rms = s.iterate(2, 0.0)
    assert nd == 2 and rms == 0.0 and np.all(s.get_field("G") == 1.0) and s.free_energy()[0] == 0.0
    assert s.iterate(0, 0.0)[0] == 0                    # zero iterations is a valid request


def test_restart_rule_fires_identically():
    """restart factor 0.95: an iteration that improves on the best residual so far by less than 5 % collapses the
    history to its best entry (Q8) -- the rule fires in some iterations and not in others, on both sides alike."""
    sol = make_solute("C2")
    kw = dict(n=32, spacing=0.5, solvent="water", solute=sol, M=6, b=0.5)
    orc, gpu, _, _ = make_pair(restart=0.95, **kw)
    ref, _, _, _ = make_pair(restart=0.0, **kw)
    orc.iterate(40, 0.0)
    ref.iterate(40, 0.0)
    gpu.iterate(40, 0.0)
    ho, hr = np.array(orc.rms_history), np.array(ref.rms_history)
    first = int(np.argmax(np.abs(ho - hr) > 1e-12 * hr))
    assert 2 <= first < 39                               # histories agree until the rule first fires, then part
    np.testing.assert_allclose(gpu.rms_history(), ho, rtol=1e-7)
    assert np.max(np.abs(gpu.get_field("G") - orc.get_field("G"))) <= 1e-9


def test_mdiis_sixteen_vectors_and_no_restart():
    orc, gpu, _, _ = make_pair("C1", n_override=32)
    orc2, gpu2, _, _ = make_pair(n=32, spacing=0.5, solvent="water", solute=make_solute("C1"), M=16, b=0.4, restart=0.0)
    orc2.iterate(40, 0.0)
    gpu2.iterate(40, 0.0)
    np.testing.assert_allclose(gpu2.rms_history(), orc2.rms_history, rtol=1e-5, atol=1e-13)
    assert np.max(np.abs(gpu2.get_field("G") - orc2.get_field("G"))) <= 1e-9


def test_split_calls_equal_one_call():
    """The MDIIS update of an iteration rides on the next closure pass; the last one of a call is applied by a
    trailing pass, so tau is current whenever iterate returns."""
    sol = _small_solute(seed=7)
    _, a, _, _ = make_pair(n=32, spacing=0.5, solvent="water", solute=sol)
    _, b, _, _ = make_pair(n=32, spacing=0.5, solvent="water", solute=sol)
    a.iterate(12, 0.0)
    for k in (1, 4, 2, 5):
        b.iterate(k, 0.0)
    assert np.array_equal(a.rms_history(), b.rms_history())
    assert np.array_equal(a.get_field("TAU"), b.get_field("TAU"))


def test_converged_call_leaves_tau_and_reports_once():
    orc, gpu, _, _ = make_pair("C1", n_override=32)
    n1, r1 = gpu.iterate(500, 1e-7)
    tau = gpu.get_field("TAU")
    assert r1 < 1e-7 and n1 < 500
    n2, r2 = gpu.iterate(500, 1e-7)                      # already converged: one more evaluation, nothing moves
    assert n2 == 1 and r2 < 1e-7
    assert np.array_equal(gpu.get_field("TAU"), tau)
    no, ro = orc.iterate(500, 1e-7)
    assert abs(no - n1) <= 1


def test_divergence_is_reported():
    import paper_2403_01039_b200 as lib
    sol = Solute("hot", np.array([[0.1, 0.2, -0.1]]), np.array([6.0]), np.array([2.0]), np.array([0.1]))
    _, gpu, _, _ = make_pair(n=16, spacing=0.5, solvent="water", closure="HNC", solute=sol, M=1, b=1.0, restart=0.0)
    with pytest.raises(lib.Rism3dError) as e:
        gpu.iterate(200, 0.0)
    assert e.value.status == -8
    assert len(gpu.rms_history()) < 200


def test_warm_start_from_device_and_host():
    sol = _small_solute(seed=9)
    _, a, _, _ = make_pair(n=16, spacing=0.6, solvent="water", solute=sol)
    _, b, _, _ = make_pair(n=16, spacing=0.6, solvent="water", solute=sol)
    a.iterate(7, 0.0)
    for s in range(2):
        b.set_tau(s, a.get_field_device("TAU", s))
    assert np.array_equal(a.get_field("TAU"), b.get_field("TAU"))
    _, c, _, _ = make_pair(n=16, spacing=0.6, solvent="water", solute=sol)
    for s in range(2):
        c.set_tau(s, a.get_field("TAU", s))
    # same input, empty history on both: the next iterate gives identical residuals
    assert b.iterate(1, 0.0) == c.iterate(1, 0.0)


# ---- NEXT-1: the paper's modified Anderson accelerator (Eq. 34-39) -------------------------------------------
@pytest.mark.parametrize("cfg,n,b,s", [("C1", 32, 0.6, (0.2, 0.0)), ("C2", 32, 0.4, (0.2, 0.0)), ("C2", 32, 0.5, (0.1, 0.05))])
def test_modified_anderson_fifty_iterations(cfg, n, b, s):
    sol = make_solute(cfg)
    orc, gpu, _, _ = make_pair(n=n, spacing=0.5, solvent="water", solute=sol, b=b, accelerator="ANDERSON", anderson_s=s)
    orc.iterate(50, 0.0)
    nd, rms = gpu.iterate(50, 0.0)
    assert nd == 50
    np.testing.assert_allclose(gpu.rms_history(), orc.rms_history, rtol=1e-6, atol=1e-13)
    assert np.max(np.abs(gpu.get_field("G") - orc.get_field("G"))) <= 1e-9


def test_modified_anderson_four_sites_converges_to_the_mdiis_fixed_point():
    sol = make_solute("C3")
    keep = np.argsort(np.linalg.norm(sol.xyz, axis=1))[:40]
    sub = Solute("C3_sub40", sol.xyz[keep], sol.q[keep], sol.sigma[keep], sol.eps[keep])
    kw = dict(n=32, spacing=0.75, solvent="water_nacl_0.1M", closure="PSE", pse_order=2, solute=sub)
    orc, gpu, _, _ = make_pair(b=0.5, accelerator="ANDERSON", **kw)
    _, ref, _, _ = make_pair(M=8, b=0.5, **kw)
    no, ro = orc.iterate(3000, 1e-9)
    ng, rg = gpu.iterate(3000, 1e-9)
    nr, rr = ref.iterate(3000, 1e-9)
    # (300 iterations amplify rounding differences: the two paths cross the threshold a few iterations apart)
    assert ro < 1e-9 and rg < 1e-9 and rr < 1e-9 and abs(ng - no) <= 0.1 * no
    mu_o, mu_g, mu_r = orc.free_energy()[0], gpu.free_energy()[0], ref.free_energy()[0]
    assert abs(mu_g - mu_o) <= 1e-7 * abs(mu_o)
    assert abs(mu_g - mu_r) <= 1e-6 * abs(mu_r)          # the fixed point does not depend on the accelerator
    gg, gr = gpu.get_field("G"), ref.get_field("G")      # (slowly converging case: rms 1e-9 leaves ~1e-6 in g)
    assert np.max(np.abs(gg - gr) / np.maximum(1.0, gr)) <= 1e-5


# ---- NEXT-2 (first item): partial molar volume, Eq. 19 ---------------------------------------------------------
@pytest.mark.parametrize("cfg,n", [("C1", 32), ("C2", 32)])
def test_partial_molar_volume_matches_oracle(cfg, n):
    orc, gpu, _, _ = make_pair(cfg, n_override=n)
    orc.iterate(400, 1e-9)
    gpu.iterate(400, 1e-9)
    chi_t = 0.55                                         # A^3 mol/kcal; any number: it multiplies both sides alike
    v_o, c_o = orc.pmv(chi_t)
    v_g, c_g = gpu.pmv(chi_t)
    assert abs(v_g - v_o) <= 1e-7 * abs(v_o)
    np.testing.assert_allclose(c_g, c_o, rtol=1e-6, atol=1e-7 * np.max(np.abs(c_o)))


# ---- NEXT-2: solvent-induced gradient on the solute atoms --------------------------------------
@pytest.mark.parametrize("case", ["C2", "sub40", "ion_offcentre"])
def test_gradient_matches_oracle(case):
    if case == "C2":
        orc, gpu, sol, _ = make_pair("C2", n_override=32)
    elif case == "sub40":
        full = make_solute("C3")
        keep = np.argsort(np.linalg.norm(full.xyz, axis=1))[:40]
        sol = Solute("C3_sub40", full.xyz[keep], full.q[keep], full.sigma[keep], full.eps[keep])
        orc, gpu, _, _ = make_pair(n=32, spacing=0.75, solvent="water_nacl_0.1M", closure="PSE", pse_order=2, M=8,
                                   solute=sol)
    else:
        sol = Solute("ion", np.array([[0.5, 0.0, 0.0]]), np.array([1.0]), np.array([2.35]), np.array([0.13]))   # on a grid point
        orc, gpu, _, _ = make_pair(n=32, spacing=0.5, solvent="water", solute=sol)
    orc.iterate(60, 0.0)
    gpu.iterate(60, 0.0)
    tau_before = gpu.get_field("TAU")
    go, gg = orc.solvation_gradient(), gpu.gradient()
    assert gg.shape == (sol.n_atoms, 3)
    assert np.max(np.abs(gg - go)) <= 1e-8 * max(1.0, np.max(np.abs(go)))
    # the gradient borrowed the k-space work array and a free history slot: the state is untouched and the loop goes on
    # exactly as it would have without the call (compared bit for bit with a second solver that never asked for it)
    assert np.array_equal(gpu.get_field("TAU"), tau_before)
    if case == "C2":
        _, twin, _, _ = make_pair("C2", n_override=32)
    elif case == "sub40":
        _, twin, _, _ = make_pair(n=32, spacing=0.75, solvent="water_nacl_0.1M", closure="PSE", pse_order=2, M=8, solute=sol)
    else:
        _, twin, _, _ = make_pair(n=32, spacing=0.5, solvent="water", solute=sol)
    twin.iterate(63, 0.0)
    gpu.iterate(3, 0.0)
    assert np.array_equal(gpu.rms_history(), twin.rms_history())
    assert np.array_equal(gpu.get_field("G"), twin.get_field("G"))


# ---- NEXT-2: pressure correction, Eq. 21, with the bulk chi_T and P stored beside the chi table (Eq. 19-20) --------
@pytest.mark.parametrize("cfg,n", [("C1", 32), ("C2", 32)])
def test_pressure_correction_matches_oracle(cfg, n):
    from workloads import load_solvent_thermo
    orc, gpu, _, _ = make_pair(cfg, n_override=n)
    chi_t, pressure = load_solvent_thermo("water")
    assert chi_t > 0.0 and np.isfinite(pressure)
    orc.iterate(400, 1e-9)
    gpu.iterate(400, 1e-9)
    pc_o, v_o = orc.pressure_correction(chi_t, pressure)
    pc_g, v_g = gpu.pressure_correction(chi_t, pressure)
    assert abs(v_g - v_o) <= 1e-7 * abs(v_o)
    assert abs(pc_g - pc_o) <= 1e-7 * abs(pc_o)
    assert pc_g == -pressure * v_g


# ---- NEXT-4: dynamic damping b = -0.2 log10(rms) (Q18) -----------------------------------
@pytest.mark.parametrize("cfg,n,M", [("C1", 32, 5), ("C2", 32, 5), ("C2", 32, 10)])
def test_dynamic_damping_fifty_iterations(cfg, n, M):
    sol = make_solute(cfg)
    orc, gpu, _, _ = make_pair(n=n, spacing=0.5, solvent="water", solute=sol, M=M, mdiis_dynamic_b=(0.1, 1.0))
    orc.iterate(50, 0.0)
    nd, rms = gpu.iterate(50, 0.0)
    assert nd == 50
    np.testing.assert_allclose(gpu.rms_history(), orc.rms_history, rtol=1e-6, atol=1e-13)
    assert np.max(np.abs(gpu.get_field("G") - orc.get_field("G"))) <= 1e-9
    # split calls: the trailing update pass applies the same dynamic b
    _, twin, _, _ = make_pair(n=n, spacing=0.5, solvent="water", solute=sol, M=M, mdiis_dynamic_b=(0.1, 1.0))
    for k in (7, 1, 30, 12):
        twin.iterate(k, 0.0)
    assert np.array_equal(twin.rms_history(), gpu.rms_history())
    assert np.array_equal(twin.get_field("TAU"), gpu.get_field("TAU"))


# ---- boxes that are not cubes: (nx, ny, nz) powers of two with one spacing (rism3d.h "grid") ------------------
@pytest.mark.parametrize("shape,nv", [((8, 16, 32), 2), ((32, 16, 8), 4), ((64, 32, 16), 1), ((16, 64, 128), 4),
                                      ((128, 32, 64), 2), ((256, 16, 16), 4)])
def test_fft_pair_on_non_cubic_grids(shape, nv):
    import torch
    import paper_2403_01039_b200 as lib
    from tests._gpu_util import oracle_spectrum_in_gpu_layout
    rng = np.random.default_rng(sum(shape) + nv)
    f = rng.standard_normal((nv,) + shape)
    s = lib.Solver(shape, 0.5, nv)
    spec = s.fft_forward(torch.from_numpy(f).cuda()).cpu().numpy()
    ref = oracle_spectrum_in_gpu_layout(f, 0.5)
    assert spec.shape == ref.shape == (shape[0], shape[1], shape[2] // 2, nv)
    tol = 2e-14 * np.log2(max(shape))
    assert np.max(np.abs(spec - ref)) < tol * np.max(np.abs(ref))
    back = s.fft_inverse(torch.from_numpy(ref).cuda()).cpu().numpy()
    assert np.max(np.abs(back - f)) < tol * np.max(np.abs(f))
    s.close()


@pytest.mark.parametrize("shape,rcut", [((32, 64, 16), 0.0), ((16, 32, 64), 7.0), ((64, 16, 32), 0.0)])
def test_fifty_iterations_on_a_non_cubic_grid(shape, rcut):
    """A small charged solute in water in a box that is not a cube (the |k| shells of the three axes then differ by factors of
    4 in the shell index): setup fields, 50 fixed iterations, free energy, gradient."""
    sol = _small_solute(seed=sum(shape), n=4)                # fits the shortest axis (8 A)
    orc, gpu, _, _ = make_pair(n=shape, spacing=0.5, solvent="water", M=5, solute=sol, rcut=rcut)
    W, Wo = gpu.get_field("W"), orc.get_field("W")
    assert W.shape == (2,) + shape
    finite = np.abs(Wo) < 600.0
    assert np.max(np.abs(W - Wo)[finite]) < 1e-10
    assert np.max(np.abs(gpu.get_field("PHI", 0) - orc.phi)) < 1e-11 * np.max(np.abs(orc.phi))
    orc.iterate(50, 0.0)
    nd, rms = gpu.iterate(50, 0.0)
    assert nd == 50
    np.testing.assert_allclose(gpu.rms_history(), orc.rms_history, rtol=1e-6, atol=1e-12)
    assert np.max(np.abs(gpu.get_field("G") - orc.get_field("G"))) <= 1e-9
    assert np.max(np.abs(gpu.get_field("TAU") - orc.get_field("TAU"))) <= 1e-9
    mu, _ = gpu.free_energy()
    mu_o, _ = orc.free_energy()
    assert abs(mu - mu_o) <= 1e-7 * abs(mu_o)
    if rcut == 0.0:
        go = orc.solvation_gradient()
        assert np.max(np.abs(gpu.gradient() - go)) <= 1e-8 * max(1.0, np.max(np.abs(go)))
    gpu.close()


def test_non_cubic_four_sites_pse2():
    """4 site types, PSE-2, M = 8 on (64, 32, 32) with a 40-atom subset of C3's solute."""
    from workloads import Solute, make_solute
    sol = make_solute("C3")
    keep = np.argsort(np.linalg.norm(sol.xyz, axis=1))[:40]
    sub = Solute("C3_sub40", sol.xyz[keep], sol.q[keep], sol.sigma[keep], sol.eps[keep])
    orc, gpu, _, _ = make_pair(n=(64, 32, 32), spacing=0.75, solvent="water_nacl_0.1M", closure="PSE", pse_order=2,
                               M=8, solute=sub)
    orc.iterate(30, 0.0)
    gpu.iterate(30, 0.0)
    np.testing.assert_allclose(gpu.rms_history(), orc.rms_history, rtol=1e-6, atol=1e-12)
    assert np.max(np.abs(gpu.get_field("G") - orc.get_field("G"))) <= 1e-9
    gpu.close()


@pytest.mark.parametrize("shape,nv,M", [((512, 8, 16), 2, 3), ((8, 512, 16), 4, 3), ((16, 8, 512), 2, 3), ((512, 16, 8), 8, 2),
                                        ((256, 8, 8), 2, 5), ((8, 256, 8), 2, 4), ((8, 8, 256), 4, 4), ((128, 64, 8), 3, 6)])
def test_longest_lines_on_thin_grids(shape, nv, M):
    """the 256- and 512-point instantiations of every pass (two-pass k-space kernels, the TMA y pass, the strided y pass
    at 512, the 256-point z lines) on grids that are thin in the other directions, whole grid against the oracle"""
    sv = _solvent(nv, seed=nv + sum(shape))
    chi = synthetic_chi(nv, sv.rho, n_k=3000, dk=0.02, k0=0.02, seed=nv, amp=0.5)
    sol = _small_solute(seed=shape[0], n=3)
    orc, gpu, _, _ = make_pair(n=shape, spacing=0.4, solvent=sv, chi=chi, M=M, solute=sol)
    W, Wo = gpu.get_field("W"), orc.get_field("W")
    finite = np.abs(Wo) < 600.0
    assert np.max(np.abs(W - Wo)[finite]) < 1e-10
    orc.iterate(12, 0.0)
    gpu.iterate(12, 0.0)
    np.testing.assert_allclose(gpu.rms_history(), orc.rms_history, rtol=1e-6, atol=1e-12)
    assert np.max(np.abs(gpu.get_field("G") - orc.get_field("G"))) <= 1e-9
    assert np.max(np.abs(gpu.get_field("TAU") - orc.get_field("TAU"))) <= 1e-9
    gpu.close()
