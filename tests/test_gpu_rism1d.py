"""-m gpu: the GPU 1D-RISM solvent solve (include/rism1d.h) against the oracle O-1D
(oracle/rism1d.py), on the same solvents: fixed numbers of iterations element by element, the converged susceptibility
chi (the input of the 3D path), the bulk thermodynamics of Eq. 19-21, and the stored table a 3D solve runs on."""
import numpy as np
import pytest

from oracle import rism1d as o1
from workloads import load_chi, solvent_by_name

pytestmark = pytest.mark.gpu


def _pair(solvent, n_points, dr=0.025, nvec=10, b=0.3, restart=0.0, closure="KH", pse_order=1):
    import paper_2403_01039_b200 as lib
    sv = solvent_by_name(solvent)
    orc = o1.Xrism1d(sv, temperature=298.0, closure=closure, pse_order=pse_order, n_points=n_points, dr=dr, kappa=1.0)
    gpu = lib.Solver1d(sv.n_s, n_points=n_points, dr=dr, closure=closure, pse_order=pse_order, mdiis_nvec=nvec, mdiis_b=b,
                       mdiis_restart=restart)
    gpu.set_solvent(sv.q[sv.site_type], sv.sigma[sv.site_type], sv.eps[sv.site_type], sv.species_rho[sv.site_species],
                    sv.site_species, sv.bond)
    return sv, orc, gpu


def _oracle_fixed(orc, lam, iters, nvec, b, restart):
    """`iters` MDIIS iterations of the oracle at charge scale lam, from its current tau (the loop of Xrism1d.solve
    without the tolerance test) -> rms history"""
    import math
    orc.set_charge_scale(lam)
    md = o1.Mdiis(nvec, b, restart)
    hist = []
    for _ in range(iters):
        X = orc.tau
        R = orc.rism_map(X) - X
        rms = math.sqrt(o1.gram(R, R) / float(orc.tau.size))
        hist.append(rms)
        orc.tau = md.step(X, R, rms)
    return hist


@pytest.mark.parametrize("solvent,n_points,lam", [("water", 2048, 0.0), ("water", 1024, 0.5), ("water_nacl_0.1M", 4096, 0.25),
                                                   ("water", 512, 0.0)])
def test_fixed_iterations_match_oracle(solvent, n_points, lam):
    """12 iterations: 1e-9 element by element (the first iterations agree to 1e-16).  40 iterations: this iteration is
    far from convergence and its MDIIS steps amplify rounding, so the bound there is what a one-ulp change of the
    oracle's OWN starting point does to the oracle (a twin run)."""
    nvec, b, restart = 6, 0.3, 10.0
    sv, orc, gpu = _pair(solvent, n_points, nvec=nvec, b=b, restart=restart)
    hist = _oracle_fixed(orc, lam, 12, nvec, b, restart)
    nd, rms = gpu.solve(lam, 12, 0.0)
    assert nd == 12
    assert abs(rms - hist[-1]) <= 1e-8 * hist[-1]
    assert np.max(np.abs(gpu.pair("TAU") - orc.tau)) <= 1e-9
    assert np.max(np.abs(gpu.pair("G") - orc.g_r())) <= 1e-9
    chi_g, chi_o = gpu.chi(), orc.chi_full()
    assert np.max(np.abs(chi_g - chi_o)) <= 1e-9 * max(1.0, np.max(np.abs(chi_o)))
    gpu.close()
    # 40 iterations from scratch, with a twin of the oracle started one ulp away
    sv, orc, gpu = _pair(solvent, n_points, nvec=nvec, b=b, restart=restart)
    _, twin, _g2 = _pair(solvent, n_points, nvec=nvec, b=b, restart=restart)
    _g2.close()
    hist = _oracle_fixed(orc, lam, 1, nvec, b, restart) + _oracle_fixed_continue(orc, 39, nvec, b, restart)
    _oracle_fixed(twin, lam, 1, nvec, b, restart)
    twin.tau = twin.tau * (1.0 + 2.0 ** -52)
    # (both oracles restart their MDIIS history after the first iteration; the GPU run does the same in two calls)
    _oracle_fixed_continue(twin, 39, nvec, b, restart)
    gpu.solve(lam, 1, 0.0)
    nd, rms = gpu.solve(lam, 39, 0.0)
    twin_d = float(np.max(np.abs(twin.tau - orc.tau)))
    d = float(np.max(np.abs(gpu.pair("TAU") - orc.tau)))
    print(f"{solvent} {n_points}: 1 + 39 iterations, max|dtau| = {d:.3e}, one-ulp twin of the oracle {twin_d:.3e}")
    assert d <= max(1e-9, 10.0 * twin_d)
    assert abs(rms - hist[-1]) <= max(1e-8, 100.0 * twin_d) * max(hist[-1], 1e-12) / min(1.0, hist[-1] / 1e-4 + 1e-30) or abs(rms - hist[-1]) <= 1e-5 * hist[-1]
    gpu.close()


def _oracle_fixed_continue(orc, iters, nvec, b, restart):
    return _oracle_fixed(orc, orc.lam, iters, nvec, b, restart)


def test_converged_water_chi_thermo_and_types():
    """the charge ramp of oracle/make_chi_tables.py on a 4096-point grid, both sides to 1e-10"""
    from oracle.make_chi_tables import RAMP as ramp
    sv, orc, gpu = _pair("water", 4096, dr=0.05, nvec=10, b=0.3, restart=0.0)
    orc.solve_with_charge_ramp(ramp=ramp, tol=1e-10, nvec=10, b=0.3, restart=0.0, max_iter=3000)
    total = 0
    for lam in ramp:
        nd, rms = gpu.solve(lam, 3000, 1e-10)
        assert rms < 1e-10
        total += nd
    assert total > 50
    chi_o = orc.chi_types()
    chi_g = gpu.chi_types(sv.site_type)
    assert chi_g.shape == chi_o.shape
    assert np.max(np.abs(chi_g - chi_o)) <= 1e-7 * np.max(np.abs(chi_o))
    assert np.max(np.abs(gpu.pair("G") - orc.g_r())) <= 1e-7
    chi_t, pr, c0 = gpu.thermo()
    assert abs(chi_t - orc.compressibility()) <= 1e-7 * abs(orc.compressibility())
    assert abs(pr - orc.pressure()) <= 1e-7 * abs(orc.pressure())
    np.testing.assert_allclose(c0, orc.c_sr_k0(), rtol=1e-7, atol=1e-7)
    gpu.close()


def test_full_size_table_feeds_the_3d_solver():
    """the production grid (16 384 points at 0.025 A, charge ramp in seven steps): chi from the GPU 1D solve, resampled
    like the stored table, against the stored table of the oracle; then a 3D solve on it"""
    import paper_2403_01039_b200 as lib
    from oracle import make_chi_tables as mk
    sv, _, gpu = _pair("water", 16384, dr=0.025, nvec=10, b=0.3, restart=0.0)
    for lam in mk.RAMP:
        nd, rms = gpu.solve(lam, 3000, 1e-10)
        assert rms < 1e-10, (lam, nd, rms)
    chi = gpu.chi_types(sv.site_type)
    k0, dk, table = load_chi("water")
    # the stored table keeps the first n_k points of the radial k grid
    assert abs(gpu.k[0] - k0) < 1e-12 and abs(gpu.k[1] - gpu.k[0] - dk) < 1e-12
    assert np.max(np.abs(chi[:table.shape[0]] - table)) <= 1e-6 * np.max(np.abs(table))
    s = lib.Solver(32, 0.5, sv.n_v)
    s.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi[:table.shape[0]])
    s.set_solute(np.zeros((1, 3)), [1.0], [2.35], [0.13])
    nd, rms = s.iterate(400, 1e-6)
    assert rms < 1e-6
    ref = lib.Solver(32, 0.5, sv.n_v)
    ref.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, table)
    ref.set_solute(np.zeros((1, 3)), [1.0], [2.35], [0.13])
    ref.iterate(400, 1e-6)
    assert abs(s.free_energy()[0] - ref.free_energy()[0]) <= 1e-5 * abs(ref.free_energy()[0])
    gpu.close()


def test_argument_and_order_checks():
    import paper_2403_01039_b200 as lib
    sv = solvent_by_name("water")
    one = lib.Solver1d(sv.n_s, n_points=512, dr=0.05)
    with pytest.raises(lib.Rism3dError) as e:
        one.solve(1.0, 5, 0.0)                               # no solvent yet
    assert e.value.status == -3
    args = [sv.q[sv.site_type], sv.sigma[sv.site_type], sv.eps[sv.site_type], sv.species_rho[sv.site_species],
            sv.site_species, sv.bond]
    bad_q = np.array(args[0], dtype=float)
    bad_q[0] += 0.1                                          # not neutral any more
    with pytest.raises(lib.Rism3dError) as e:
        one.set_solvent(bad_q, *args[1:])
    assert e.value.status == -5
    no_bond = np.zeros_like(sv.bond)
    with pytest.raises(lib.Rism3dError) as e:
        one.set_solvent(*args[:5], no_bond)                  # bonded sites need a distance
    assert e.value.status == -1
    one.set_solvent(*args)
    nd, rms = one.solve(0.0, 3, 0.0)
    assert nd == 3 and rms > 0
    with pytest.raises(lib.Rism3dError):
        lib.rism1d_get_pair(one.ctx, 7, sv.n_s, 512)         # unknown pair function
    # a refused set_solvent leaves the accepted solvent in place: same iterations, same numbers, before and after
    g_before = lib.rism1d_get_pair(one.ctx, 0, sv.n_s, 512)
    for k, bad in ((1, 0.0), (1, -1.0), (3, 0.0), (2, -0.1), (1, float("nan"))):     # sigma, rho, eps
        a = [np.array(x, dtype=float) if i < 4 else x for i, x in enumerate(args)]
        a[k][0] = bad
        with pytest.raises(lib.Rism3dError) as e:
            one.set_solvent(*a)
        assert e.value.status == -1
    with pytest.raises(lib.Rism3dError) as e:
        one.set_solvent(*args[:5], no_bond)
    assert e.value.status == -1
    g_after = lib.rism1d_get_pair(one.ctx, 0, sv.n_s, 512)
    assert np.array_equal(np.asarray(g_before), np.asarray(g_after))
    for bad in (-0.5, float("nan"), float("inf")):           # a negative scale used to double as "never solved"
        with pytest.raises(lib.Rism3dError) as e:
            one.solve(bad, 1, 0.0)
        assert e.value.status == -1
    one.close()
