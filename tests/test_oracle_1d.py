"""Pins for the O-1D oracle (oracle/rism1d.py; SURVEY.md §8(c) "O-1D" step 5) and pin P10 of the 3D oracle:
the radial Fourier pair against a closed form, the low-density limit, the index conventions and limits of the
stored chi tables, and the 3D loop for a spherical ion against the independent radial (1D) discretisation."""
import math

import numpy as np
import pytest

from oracle import rism1d as o1
from oracle import rism3d as o3
from workloads import Solvent, load_chi, make_solute, solvent_by_name, water
from workloads.solvents import L_HH, L_OH


# ------------------------------------------------------------------------------------------------
# radial transform pair: exp(-a r^2)  <->  (pi/a)^{3/2} exp(-k^2 / (4a))   (textbook closed form)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("a", [1.0, 0.35])
def test_radial_transform_gaussian_pair(a):
    g = o1.RadialGrid(2048, 0.02)
    f = np.exp(-a * g.r ** 2)
    F = g.forward(f)
    exact = (math.pi / a) ** 1.5 * np.exp(-g.k ** 2 / (4.0 * a))
    assert np.max(np.abs(F - exact)) < 1e-10 * exact.max()
    back = g.inverse(exact)
    assert np.max(np.abs(back - f)) < 1e-10
    # and the pair is an exact inverse of itself on the grid (DST-I is an involution up to scale)
    assert np.max(np.abs(g.inverse(F) - f)) < 1e-12


def test_radial_grid_spacing_relation():
    g = o1.RadialGrid(1024, 0.05)
    assert abs(g.dr * g.dk - math.pi / 1024) < 1e-15
    assert g.r[0] == g.dr and g.k[0] == g.dk and len(g.r) == 1023


def test_long_range_pair_1d_is_a_fourier_pair():
    """f(r) = beta C qq (1 - exp(-kappa r))/r minus the bare Coulomb beta C qq / r is short ranged:
    its radial transform must equal 4 pi beta C qq [kappa^2/(k^2(k^2+kappa^2)) - 1/k^2] = -4 pi beta C qq/(k^2+kappa^2)
    (Eq. 29-30)."""
    g = o1.RadialGrid(4096, 0.01)
    beta, qq, kappa = 1.7, -0.36, 1.0
    short = o1.f_long_r(g.r, qq, beta, kappa) - beta * o3.COULOMB * qq / g.r          # = -beta C qq exp(-kappa r)/r
    lhs = g.forward(short)
    rhs = o1.f_long_k(g.k, qq, beta, kappa) - 4.0 * math.pi * beta * o3.COULOMB * qq / g.k ** 2
    sel = g.k < 20.0
    assert np.max(np.abs(lhs - rhs)[sel]) < 2e-3 * np.max(np.abs(rhs))
    assert np.allclose(rhs, -4.0 * math.pi * beta * o3.COULOMB * qq / (g.k ** 2 + kappa ** 2), rtol=1e-12)


def test_omega_matrix():
    sv = water()
    k = np.array([0.5, 2.0, 7.0])
    W = o1.omega_k(k, sv.bond, sv.site_species)
    assert np.allclose(W[:, 0, 0], 1.0) and np.allclose(W, np.swapaxes(W, 1, 2))
    assert np.allclose(W[:, 0, 1], np.sin(k * L_OH) / (k * L_OH))
    assert np.allclose(W[:, 1, 2], np.sin(k * L_HH) / (k * L_HH))
    sv2 = solvent_by_name("water_nacl_0.1M")
    W2 = o1.omega_k(k, sv2.bond, sv2.site_species)
    assert np.all(W2[:, 3, :3] == 0.0) and np.all(W2[:, 3, 4] == 0.0) and np.all(W2[:, 4, 4] == 1.0)


# ------------------------------------------------------------------------------------------------
# low-density limit of the solvent-solvent solve: a one-site LJ fluid at rho -> 0 has g = exp(-beta u) + O(rho)
# ------------------------------------------------------------------------------------------------
def _one_site_fluid(rho, q=0.0):
    return Solvent(name="lj", type_names=["A"], q=np.array([q]), sigma=np.array([3.4]), eps=np.array([0.24]),
                   rho=np.array([rho]), mult=np.array([1]), site_type=np.array([0]), site_species=np.array([0]),
                   species_rho=np.array([rho]), bond=np.zeros((1, 1)))


def test_low_density_limit_is_the_boltzmann_factor():
    x = o1.Xrism1d(_one_site_fluid(1e-7), temperature=298.0, closure="HNC", n_points=1024, dr=0.03)
    x.solve(tol=1e-12, nvec=5, b=0.7)
    g = x.g_r()[0, 0]
    boltz = np.exp(-x.beta * o1.lj_pair(x.grid.r, 3.4, 0.24, 3.4, 0.24))
    assert np.max(np.abs(g - boltz)) < 1e-5
    # at a moderate density the first-order correction has the right sign at contact for a repulsive core: g > e^{-beta u}
    x2 = o1.Xrism1d(_one_site_fluid(0.01), temperature=298.0, closure="HNC", n_points=1024, dr=0.03)
    x2.solve(tol=1e-10, nvec=5, b=0.5)
    i = int(np.argmax(boltz))
    assert x2.g_r()[0, 0][i] > boltz[i]
    # chi of a one-site fluid is the structure factor S(k) = 1 + rho h(k): compressibility limit S(0) < 1 for this state
    chi = x2.chi_types()[:, 0, 0]
    assert 0.0 < chi[0] < 1.0 and abs(chi[-1] - 1.0) < 1e-3


# ------------------------------------------------------------------------------------------------
# the stored chi tables (workloads/chi/*.npz, written by oracle/make_chi_tables.py): conventions and limits
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["water", "water_nacl_0.1M", "water_nacl_0.15M"])
def test_stored_chi_density_weighted_symmetry(name):
    """chi_{g'g} = omega_{g'g} + rho_{g'} h_{g'g} reduced to site types is NOT symmetric, but
    rho_g chi_{g'g} is (Q15); a transposed table fails this."""
    sv = solvent_by_name(name)
    k0, dk, chi = load_chi(name)
    assert chi.shape[1:] == (sv.n_v, sv.n_v)
    w = chi * sv.rho[None, None, :]
    scale = np.max(np.abs(w), axis=0)
    # 1e-8 of each entry's own scale: the 1D solve stops at rms 1e-10 and the ion entries are ~1e-4; a transposed
    # table is off by O(1)
    assert np.max(np.abs(w - np.swapaxes(w, 1, 2)) / scale[None]) < 1e-8
    # and the water block really is asymmetric: chi_HO = 2 chi_OH
    assert np.allclose(chi[:, 1, 0], 2.0 * chi[:, 0, 1], rtol=1e-9, atol=1e-12)


def test_stored_chi_large_k_limit_is_the_reduced_intramolecular_matrix():
    k0, dk, chi = load_chi("water_nacl_0.1M")
    k = k0 + dk * np.arange(chi.shape[0])
    sel = k > 14.0
    s_oh = np.sin(k * L_OH) / (k * L_OH)
    s_hh = np.sin(k * L_HH) / (k * L_HH)
    expect = np.zeros_like(chi)
    expect[:, 0, 0] = 1.0
    expect[:, 1, 1] = 1.0 + s_hh            # sum over a in H of omega_{a,H1}
    expect[:, 0, 1] = s_oh                  # a = O, b = H
    expect[:, 1, 0] = 2.0 * s_oh            # a = H1, H2, b = O
    expect[:, 2, 2] = 1.0
    expect[:, 3, 3] = 1.0
    dev = np.max(np.abs(chi - expect)[sel], axis=0)     # what is left is rho h(k), decaying like 1/k^2
    assert np.max(dev[:2, :2]) < 1e-2                   # water block: |s_oh| reaches 0.07 here, so a lost factor 2 shows
    assert np.max(dev[:2, 2:]) < 2e-2                   # rho_water h(water-ion)
    assert np.max(dev[2:, :]) < 1e-3                    # rows of the dilute ions: rho_ion h ~ 1e-4


def test_stored_chi_neutral_molecule_sum_rule():
    """Pure water: sum_{g'} q_{g'} chi_{g'g}(k) -> 0 like k^2 as k -> 0 (neutral molecules, perfect screening)."""
    sv = water()
    k0, dk, chi = load_chi("water")
    k = k0 + dk * np.arange(chi.shape[0])
    s = np.einsum("a,kab->kb", sv.q, chi)
    assert np.max(np.abs(s[0])) < 1e-3
    for g in range(2):
        ratio = s[7, g] / s[3, g]           # k_7 / k_3 = 2  ->  ratio 4 for a k^2 law
        assert 3.5 < ratio < 4.5


def test_stored_chi_covers_every_config_grid():
    from workloads import CONFIGS
    for cfg in CONFIGS.values():
        k0, dk, chi = load_chi(cfg.solvent)
        dkg = 2.0 * math.pi / (cfg.n * cfg.spacing)
        kmin, kmax = dkg * math.sqrt(0.75), math.sqrt(3.0) * (math.pi / cfg.spacing - dkg / 2.0)
        assert k0 <= kmin and kmax <= k0 + (chi.shape[0] - 1) * dk
        assert dk <= kmin / 2.0             # table at least twice finer than the smallest 3D |k|


# ------------------------------------------------------------------------------------------------
# a fresh (coarser) water solve: physical sanity of g, and the stored table is what the script produces
# ------------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def coarse_water():
    x = o1.Xrism1d(water(), temperature=298.0, closure="KH", n_points=2048, dr=0.05, kappa=1.0)
    x.solve_with_charge_ramp(ramp=(0.0, 0.25, 0.5, 0.75, 0.85, 0.95, 1.0), tol=1e-9, nvec=10, b=0.3, restart=0.0,
                             max_iter=3000)
    return x


def test_water_pair_functions_are_sane(coarse_water):
    x = coarse_water
    g = x.g_r()
    assert g.min() >= 0.0
    assert np.max(np.abs(g[:, :, x.grid.r > 40.0] - 1.0)) < 1e-3          # g -> 1 at large r
    assert np.max(g[:, :, x.grid.r < 0.8]) < 1e-6 or g[0, 0, x.grid.r < 2.0].max() < 1e-3   # cores are empty
    assert np.max(np.abs(g - np.swapaxes(g, 0, 1))) < 1e-10               # g_ab = g_ba
    assert np.max(np.abs(g[1, 1] - g[2, 2])) < 1e-8 and np.max(np.abs(g[0, 1] - g[0, 2])) < 1e-8   # H1 == H2
    # O-H hydrogen-bond peak sits inside the O-O first peak
    r = x.grid.r
    r_oh = r[np.argmax(g[0, 1] * (r < 2.5))]
    r_oo = r[np.argmax(g[0, 0] * (r < 4.0))]
    assert 1.4 < r_oh < 2.2 and 2.5 < r_oo < 3.5


def test_stored_water_table_matches_a_coarser_solve(coarse_water):
    """The stored table comes from 16384 points at 0.025 A; 2048 points at 0.05 A must give the same chi to the
    accuracy of the coarser radial grid (a table written by anything else than this solve would be off by O(1))."""
    x = coarse_water
    k0, dk, chi = load_chi("water")
    k_tab = k0 + dk * np.arange(chi.shape[0])
    fresh = x.chi_types()
    kf = x.grid.k
    sel = kf < 10.0
    for a in range(2):
        for b in range(2):
            ref = np.interp(kf[sel], k_tab, chi[:, a, b])
            assert np.max(np.abs(fresh[sel, a, b] - ref)) < 2e-2 * max(1.0, np.max(np.abs(ref)))


def test_reduced_types_equal_full_site_sums(coarse_water):
    x = coarse_water
    full = x.chi_full()
    red = x.chi_types()
    assert np.allclose(red[:, 0, 0], full[:, 0, 0])
    assert np.allclose(red[:, 1, 1], full[:, 1, 1] + full[:, 2, 1])
    assert np.allclose(red[:, 0, 1], full[:, 0, 1])
    assert np.allclose(red[:, 1, 0], full[:, 1, 0] + full[:, 2, 0])
    # chi_full = omega + rho h with h symmetric and one density: symmetric
    assert np.max(np.abs(full - np.swapaxes(full, 1, 2))) < 1e-8


# ------------------------------------------------------------------------------------------------
# P10: a single spherical ion.  Spherical symmetry reduces 3D-RISM to the 1D solute-solvent equation (Eq. 8,
# PAPER.md:107, with one solute site): the 3D oracle on a 32 A box against the independent radial discretisation,
# same chi table, closure and kappa.  A discretisation / box check, hence loose.
# ------------------------------------------------------------------------------------------------
@pytest.mark.slow
def test_p10_spherical_ion_3d_matches_radial_1d():
    sv = water()
    k0, dk, chi = load_chi("water")
    sol = make_solute("C1")                       # Na+ at the origin
    n, dr = 64, 0.5
    orc = o3.Rism3dOracle(n, dr, sv.n_v, closure="KH", mdiis_nvec=5)
    orc.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    orc.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps)
    nd, rms = orc.iterate(500, 1e-7)
    assert rms < 1e-7
    g3 = orc.get_field("G")
    mu3, _ = orc.free_energy()

    grid = o1.RadialGrid(4096, 0.0125)            # r to 51 A, k to 251 1/A
    k_hi = k0 + (chi.shape[0] - 1) * dk
    chi_on = np.moveaxis(o3.interp_chi(np.clip(grid.k, k0, k_hi), k0, dk, chi), -1, 0)
    beyond = grid.k > k_hi                        # past the table (16 1/A): the intramolecular limit of chi
    s_oh, s_hh = (np.sin(grid.k * l) / (grid.k * l) for l in (L_OH, L_HH))
    chi_on[beyond] = np.stack([np.stack([np.ones_like(s_oh), s_oh], -1),
                               np.stack([2.0 * s_oh, 1.0 + s_hh], -1)], -2)[beyond]
    ion = o1.IonRism1d(grid, chi_on, sv.q, sv.sigma, sv.eps, sv.rho, sol.q[0], sol.sigma[0], sol.eps[0])
    ion.solve(tol=1e-9)
    g1 = ion.g_r()
    mu1, _ = ion.free_energy()

    rr = np.sqrt(np.sum(orc.points ** 2, axis=1)).reshape(n, n, n)
    for s in range(sv.n_v):
        # radius, tolerance of the shell mean against the radial solution, tolerance of the spread over the shell
        for r_c, tol, spread in [(2.5, 0.08, 0.25), (3.0, 0.05, 0.30), (5.0, 0.015, 0.08), (6.0, 0.01, 0.03),
                                 (10.0, 0.005, 0.01), (12.0, 0.005, 0.01)]:
            shell = np.abs(rr - r_c) < 1e-9       # grid points at exactly this distance (axes and permutations)
            assert shell.sum() >= 6
            vals = g3[s][shell]
            # different orbits of the cubic group at one radius agree to the grid's discretisation error ...
            assert vals.max() - vals.min() < spread * max(1.0, vals.mean()), (s, r_c, vals.min(), vals.max())
            i1 = int(round(r_c / grid.dr)) - 1
            assert abs(vals.mean() - g1[s][i1]) < tol * max(1.0, g1[s][i1]), (s, r_c, vals.mean(), g1[s][i1])
        # ... and the points of one orbit (+-x, +-y, +-z axis at 3 A; index n/2 is the origin) agree to rounding
        c, o = n // 2, 6
        axis = [g3[s][c + o, c, c], g3[s][c - o, c, c], g3[s][c, c + o, c], g3[s][c, c - o, c], g3[s][c, c, c + o],
                g3[s][c, c, c - o]]
        assert max(axis) - min(axis) < 1e-6
        inside = rr < 1.5
        assert g3[s][inside].max() < 1e-6 and g1[s][grid.r < 1.5].max() < 1e-6      # empty core in both
    assert abs(mu3 - mu1) < 0.01 * abs(mu1)       # measured: -80.44 (3D, 0.5 A grid) vs -80.64 (radial) kcal/mol


# ------------------------------------------------------------------------------------------------
# Bulk thermodynamics of the solvent: compressibility (for Eq. 19) and pressure (Eq. 20)
# ------------------------------------------------------------------------------------------------
def _lj_fluid(rho, sigma=3.4, eps=0.24):
    """one-site Lennard-Jones fluid (inputs only)"""
    return Solvent(name="lj", type_names=["A"], q=np.zeros(1), sigma=np.array([sigma]), eps=np.array([eps]),
                   rho=np.array([rho]), mult=np.ones(1, int), site_type=np.zeros(1, int), site_species=np.zeros(1, int),
                   species_rho=np.array([rho]), bond=np.zeros((1, 1)))


def test_compressibility_and_pressure_low_density_limits_and_second_virial_coefficient():
    """Ideal gas: chi_T = 1/(rho kT), P = rho kT.  To second order in the density (textbook virial expansion, B_2 from an
    independent radial quadrature of the Mayer function):  P = kT (rho + B_2 rho^2),  1/(kT chi_T) = rho + 2 B_2 rho^2."""
    T = 298.0
    kT = o3.K_BOLTZMANN * T
    sig, eps = 3.4, 0.24
    r = np.linspace(1e-3, 60.0, 600001)
    mayer = np.exp(-4.0 * eps * ((sig / r) ** 12 - (sig / r) ** 6) / kT) - 1.0
    b2 = -2.0 * math.pi * np.trapezoid(mayer * r * r, r)
    for rho in (1e-7, 2e-5):                               # (third virial term: B_3 rho^3 / |B_2| rho^2 ~ 2e-3 at 2e-5)
        x = o1.Xrism1d(_lj_fluid(rho, sig, eps), temperature=T, closure="HNC", n_points=4096, dr=0.02)
        x.solve(tol=1e-12, nvec=5, b=1.0)
        chi_t, p = x.compressibility(), x.pressure()
        assert abs(chi_t * rho * kT - 1.0) < 3.0 * abs(2 * b2 * rho) + 1e-9          # -> ideal gas
        assert abs(p / (rho * kT) - 1.0) < 3.0 * abs(b2 * rho) + 1e-9
        # second virial level: the remainders are O(rho^2) relative
        assert abs(p / kT - (rho + b2 * rho * rho)) < 1e-2 * abs(b2) * rho * rho
        assert abs(1.0 / (kT * chi_t) - (rho + 2.0 * b2 * rho * rho)) < 1e-2 * abs(2.0 * b2) * rho * rho


def test_compressibility_equals_structure_factor_at_k_zero():
    """One-site fluid: rho kT chi_T = S(0) = 1 + rho h(k -> 0) (the textbook compressibility equation) -- h from the
    converged g(r) by direct integration, against the c-route the oracle uses."""
    T, rho = 298.0, 0.018
    kT = o3.K_BOLTZMANN * T
    x = o1.Xrism1d(_lj_fluid(rho), temperature=T, closure="KH", n_points=8192, dr=0.02)
    x.solve(tol=1e-12, nvec=8, b=0.7)
    g = x.g_r()[0, 0]
    h0 = 4.0 * math.pi * x.grid.dr * np.sum((g - 1.0) * x.grid.r ** 2)
    assert abs(rho * kT * x.compressibility() - (1.0 + rho * h0)) < 2e-4 * (1.0 + rho * h0)


def test_water_thermodynamics_sanity_and_site_sum_convention(coarse_water):
    """Water (3 sites, one species): rho kT chi_T = 1/(1 - rho sum_ab c_ab(0)) with the sum over ALL NINE site pairs, and
    Eq. 20 with n_Gamma = 3.  Coarse radial grid (the stored tables use 16384 points): sanity of sign and size only."""
    sv = water()
    x = coarse_water
    kT = 1.0 / x.beta
    c0 = x.c_sr_k0()
    assert c0.shape == (3, 3) and np.allclose(c0, c0.T, rtol=1e-9, atol=1e-9)
    rho = sv.species_rho[0]
    chi_t = x.compressibility()
    assert abs(rho * kT * chi_t - 1.0 / (1.0 - rho * c0.sum())) < 1e-12
    assert 0.0 < rho * kT * chi_t < 1.0                                  # a dense liquid is far less compressible than a gas
    p = x.pressure()
    assert abs(p - kT * (rho * (3 + 1) / 2.0 - 0.5 * rho * rho * c0.sum())) < 1e-12 * abs(p)


def test_pressure_correction_is_minus_p_v():
    """Eq. 21 on top of Eq. 19: a null solute has V = kT chi_T and dmu_PC = -P kT chi_T."""
    sv = water()
    from tests._util import synthetic_chi
    k0, dk, chi = synthetic_chi(2, sv.rho)
    orc = o3.Rism3dOracle(16, 0.6, 2)
    orc.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    orc.set_solute(np.array([[0.1, 0.0, 0.2]]), [0.0], [3.0], [0.0])
    orc.iterate(1, 0.0)
    pc, v = orc.pressure_correction(0.7, 0.01)
    assert v == orc.kT * 0.7 and pc == -0.01 * v
