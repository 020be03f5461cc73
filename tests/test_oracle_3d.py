"""Pins for the O-3D oracle: each checks the oracle against something other
than itself -- brute-force sums, closed forms, invariants, textbook special cases."""
import itertools
import math

import numpy as np
import pytest

from oracle import rism3d as o3
from tests._util import identity_chi, synthetic_chi
from workloads import water, make_solute

BETA = 1.0 / (o3.K_BOLTZMANN * 298.0)


# ------------------------------------------------------------------------------------------------
# P1: shifted DFT pair vs the O(N^2) triple sum written from the definition
# ------------------------------------------------------------------------------------------------
def _brute_forward(f, dr, origin):
    nx, ny, nz = f.shape
    L = [nx * dr, ny * dr, nz * dr]
    out = np.zeros(f.shape, dtype=complex)
    for jx, jy, jz in itertools.product(range(nx), range(ny), range(nz)):
        k = []
        for j, n, l in zip((jx, jy, jz), (nx, ny, nz), L):
            dk = 2 * math.pi / l
            k.append(dk * (j + 0.5) if j < n // 2 else dk * (j + 0.5 - n))
        acc = 0j
        for ix, iy, iz in itertools.product(range(nx), range(ny), range(nz)):
            r = (origin[0] + ix * dr, origin[1] + iy * dr, origin[2] + iz * dr)
            acc += f[ix, iy, iz] * np.exp(-1j * (k[0] * r[0] + k[1] * r[1] + k[2] * r[2]))
        out[jx, jy, jz] = acc * dr ** 3
    return out


@pytest.mark.parametrize("shape", [(4, 4, 4), (2, 4, 8), (8, 8, 8)])
def test_p1_shifted_dft_matches_brute_force(shape):
    rng = np.random.default_rng(1)
    f = rng.standard_normal(shape)
    dr = 0.4
    origin = (-0.7, 0.3, -1.1)          # deliberately not a multiple of dr
    F = o3.shifted_dft_forward(f, dr, origin)
    Fb = _brute_forward(f, dr, origin)
    assert np.max(np.abs(F - Fb)) < 1e-13 * np.max(np.abs(Fb))
    # round trip and reality
    back = o3.shifted_dft_inverse(F, dr, origin)
    assert np.max(np.abs(back.imag)) < 1e-14
    assert np.max(np.abs(back.real - f)) < 1e-13
    # Parseval: dV sum |f|^2 = (1/V) sum |F|^2
    V = np.prod(shape) * dr ** 3
    assert abs(dr ** 3 * np.sum(f * f) - np.sum(np.abs(F) ** 2) / V) < 1e-12
    # conjugate symmetry of a real field on the half-integer grid: F[n-1-j] = conj F[j] on all three axes
    # (holds up to the origin phase; check with the default, grid-aligned origin)
    o0 = tuple(-(n // 2) * dr for n in shape)
    F0 = o3.shifted_dft_forward(f, dr, o0)
    assert np.max(np.abs(F0[::-1, ::-1, ::-1] - np.conj(F0))) < 1e-13 * np.max(np.abs(F0))


def test_k_axis_is_symmetric_half_integer_set():
    k = o3.k_axis(8, 0.5)
    dk = 2 * math.pi / 4.0
    assert np.allclose(np.sort(k) / dk, [-3.5, -2.5, -1.5, -0.5, 0.5, 1.5, 2.5, 3.5])
    assert np.allclose(k[:4] / dk, [0.5, 1.5, 2.5, 3.5])


# ------------------------------------------------------------------------------------------------
# Eq. 29 <-> Eq. 30 are a Fourier pair (Q5): radial quadrature of the continuous transform
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kappa", [1.0, 0.7])
def test_long_range_pair_is_a_fourier_pair(kappa):
    # FT[(1-exp(-kappa r))/r](k) = 4 pi kappa^2/(k^2 (k^2+kappa^2)); verify through the convergent
    # difference with a second screening length: FT[(exp(-a r) - exp(-kappa r))/r] = 4pi/(k^2+a^2) - 4pi/(k^2+kappa^2)
    a = 0.05
    r = np.linspace(1e-6, 400.0, 4_000_001)
    for k in (0.3, 1.0, 2.5):
        integrand = 4 * math.pi * r * np.sin(k * r) / k * (np.exp(-a * r) - np.exp(-kappa * r)) / r
        num = np.trapezoid(integrand, r)
        # oracle formula with 1/r -> exp(-a r)/r regularisation removed analytically:
        xyz = np.zeros((1, 3))
        pt = o3.phi_tilde_at(np.array([[k, 0.0, 0.0]]), xyz, np.array([1.0]), 1.0, kappa)[0].real / o3.COULOMB
        exact_reg = pt - (4 * math.pi / k ** 2 - 4 * math.pi / (k ** 2 + a ** 2))
        assert abs(num - exact_reg) < 2e-6 * abs(exact_reg) + 1e-7


def test_phi_limits_and_values():
    xyz = np.array([[0.0, 0.0, 0.0]])
    q = np.array([2.0])
    pts = np.array([[0.0, 0.0, 0.0], [1e-10, 0.0, 0.0], [0.0, 3.0, 4.0]])
    phi = o3.phi_at(pts, xyz, q, 1.5, 0.8)
    assert phi[0] == pytest.approx(1.5 * o3.COULOMB * 2.0 * 0.8, rel=1e-15)
    assert phi[1] == pytest.approx(phi[0], rel=1e-9)
    assert phi[2] == pytest.approx(1.5 * o3.COULOMB * 2.0 * (1 - math.exp(-4.0)) / 5.0, rel=1e-14)
    # structure factor phase: atom displaced along x
    kv = np.array([[0.4, -0.2, 0.9]])
    R = np.array([[1.0, 2.0, -0.5]])
    pt = o3.phi_tilde_at(kv, R, np.array([1.0]), 1.0, 1.0)[0]
    k2 = 0.16 + 0.04 + 0.81
    mag = 4 * math.pi * o3.COULOMB / (k2 * (k2 + 1))
    ph = -(0.4 * 1.0 - 0.2 * 2.0 - 0.9 * 0.5)
    assert pt == pytest.approx(mag * complex(math.cos(ph), math.sin(ph)), rel=1e-14)


def test_potential_hand_values():
    # one atom, one solvent site: LJ zero at r = sigma, minimum -eps at 2^(1/6) sigma, Coulomb C q q / r
    xyz = np.zeros((1, 3))
    s_u, e_u, s_v, e_v = 3.0, 0.2, 2.0, 0.05
    s = 2.5
    e = math.sqrt(0.2 * 0.05)
    pts = np.array([[s, 0, 0], [0, 2 ** (1 / 6) * s, 0], [0, 0, 7.0], [0, 0, 0]])
    bu = o3.beta_u_at(pts, xyz, np.array([0.5]), np.array([s_u]), np.array([e_u]),
                      np.array([-0.8]), np.array([s_v]), np.array([e_v]), BETA, 1e-3)[0]
    assert bu[0] == pytest.approx(BETA * o3.COULOMB * 0.5 * -0.8 / s, rel=1e-12)
    assert bu[1] == pytest.approx(BETA * (o3.COULOMB * 0.5 * -0.8 / (2 ** (1 / 6) * s) - e), rel=1e-12)
    lj7 = 4 * e * ((s / 7) ** 12 - (s / 7) ** 6)
    assert bu[2] == pytest.approx(BETA * (o3.COULOMB * 0.5 * -0.8 / 7.0 + lj7), rel=1e-12)
    assert bu[3] > 1e30                 # clamped at r_min, still astronomically repulsive (Q11)
    # cut-off short-range remainder + f reproduces Eq. 22 when the cutoff includes the atom
    w = o3.w_short_at(pts[:3], xyz, np.array([0.5]), np.array([s_u]), np.array([e_u]), np.array([-0.8]),
                      np.array([s_v]), np.array([e_v]), BETA, 1e-3, 1.0, 50.0)[0]
    f = -0.8 * o3.phi_at(pts[:3], xyz, np.array([0.5]), BETA, 1.0)
    assert np.allclose(w - f, -bu[:3], rtol=1e-12)
    # and drops it when it does not
    w2 = o3.w_short_at(pts[2:3], xyz, np.array([0.5]), np.array([s_u]), np.array([e_u]), np.array([-0.8]),
                       np.array([s_v]), np.array([e_v]), BETA, 1e-3, 1.0, 6.9)[0]
    assert w2[0] == 0.0


# ------------------------------------------------------------------------------------------------
# P9: closure limits (Q1, Q2)
# ------------------------------------------------------------------------------------------------
def test_p9_closure_limits():
    d = np.linspace(-6, 6, 2401)
    kh = o3.closure_g(d, "KH")
    assert np.array_equal(kh, o3.closure_g(d, "PSE", 1))                    # PSE-1 == KH bit for bit
    assert np.allclose(kh[d <= 0], np.exp(d[d <= 0]), rtol=0, atol=0)
    assert np.allclose(kh[d > 0], 1 + d[d > 0], rtol=1e-16)
    assert np.all(kh >= 0)                                                  # the reading of Q1: g >= 0
    # continuity and C^n at 0
    eps = 1e-7
    for n in (1, 2, 3):
        gm = o3.closure_g(np.array([-eps]), "PSE", n)[0]
        gp = o3.closure_g(np.array([+eps]), "PSE", n)[0]
        assert abs(gp - gm - 2 * eps) < 1e-13
    # PSE-2 value: 1 + d + d^2/2 ; PSE-3 adds d^3/6
    assert o3.closure_g(np.array([2.0]), "PSE", 2)[0] == pytest.approx(5.0, rel=1e-15)
    assert o3.closure_g(np.array([2.0]), "PSE", 3)[0] == pytest.approx(5.0 + 8.0 / 6.0, rel=1e-15)
    # n -> infinity: HNC
    dd = np.linspace(-5, 5, 101)
    assert np.allclose(o3.closure_g(dd, "PSE", 30), o3.closure_g(dd, "HNC"), rtol=1e-12)
    # free-energy extra term: PSE-1 == KH where they overlap (d = h on the linear branch)
    h = kh - 1
    assert np.allclose(o3.closure_sfe_extra(d, h, "KH"), o3.closure_sfe_extra(d, h, "PSE", 1), rtol=1e-15, atol=0)
    assert np.all(o3.closure_sfe_extra(d, h, "HNC") == 0)
    # no overflow warnings on the unused branch
    with np.errstate(over="raise"):
        o3.closure_g(np.array([1e4, -1e40]), "KH")


# ------------------------------------------------------------------------------------------------
# chi interpolation (Q6): cubic Lagrange reproduces cubics exactly, including the shifted end stencils
# ------------------------------------------------------------------------------------------------
def test_interp_chi_reproduces_cubics():
    k0, dk, n_k = 0.1, 0.05, 50
    k = k0 + dk * np.arange(n_k)
    poly = lambda x: 1.0 - 2.0 * x + 0.5 * x ** 2 + 0.3 * x ** 3
    chi = np.zeros((n_k, 2, 2))
    chi[:, 0, 1] = poly(k)
    chi[:, 1, 0] = 7.0
    kq = np.array([0.1, 0.1201, 0.333, 1.0, 2.549, 2.55])      # first/last intervals included
    out = o3.interp_chi(kq, k0, dk, chi)
    assert np.allclose(out[0, 1], poly(kq), rtol=1e-13)
    assert np.allclose(out[1, 0], 7.0, rtol=1e-14)
    assert np.all(out[0, 0] == 0)
    # nodes are reproduced exactly enough and the interpolant is continuous across a node
    a = o3.interp_chi(np.array([k[10] - 1e-12, k[10] + 1e-12]), k0, dk, chi)[0, 1]
    assert abs(a[0] - a[1]) < 1e-10
    with pytest.raises(ValueError):
        o3.interp_chi(np.array([2.56]), k0, dk, chi)
    with pytest.raises(ValueError):
        o3.interp_chi(np.array([0.09]), k0, dk, chi)


# ------------------------------------------------------------------------------------------------
# MDIIS (Q7, Q8): small solve vs LAPACK, KKT conditions, affine-map special case (P8), M = 1 limit
# ------------------------------------------------------------------------------------------------
def test_mdiis_coefficients_match_lapack_and_kkt():
    rng = np.random.default_rng(3)
    for m in (1, 2, 5, 10):
        Rm = rng.standard_normal((m, 40))
        S = Rm @ Rm.T * 3.7e-5
        c = o3.mdiis_coefficients(S)
        A = np.zeros((m + 1, m + 1))
        A[:m, :m] = S / S.diagonal().max()
        A[:m, m] = A[m, :m] = 1
        rhs = np.zeros(m + 1)
        rhs[m] = 1
        ref = np.linalg.solve(A, rhs)[:m]
        assert np.allclose(c, ref, rtol=1e-9, atol=1e-12)
        assert abs(c.sum() - 1) < 1e-12
        # minimiser: any feasible perturbation increases c^T S c
        base = c @ S @ c
        for _ in range(5):
            dlt = rng.standard_normal(m)
            dlt -= dlt.mean()
            assert (c + 1e-3 * dlt) @ S @ (c + 1e-3 * dlt) >= base - 1e-18
    assert np.array_equal(o3.mdiis_coefficients(np.zeros((3, 3))), [0, 0, 1])       # degenerate: last entry


def test_p8_mdiis_exact_on_affine_map():
    # Y = A X + y0 in d = 3 dimensions, b = 1, M >= d + 1: exact fixed point within d + 1 steps
    rng = np.random.default_rng(5)
    A = 0.5 * rng.standard_normal((3, 3))
    y0 = rng.standard_normal(3)
    xstar = np.linalg.solve(np.eye(3) - A, y0)
    md = o3.Mdiis(nvec=5, b=1.0, restart=0.0)
    X = np.zeros(3)
    for step in range(4):
        R = A @ X + y0 - X
        X = md.step(X, R, float(np.sqrt(R @ R / 3)))
    assert np.max(np.abs(X - xstar)) < 1e-10


def test_mdiis_m1_is_damped_picard_and_b1_is_diis():
    rng = np.random.default_rng(6)
    X, R = rng.standard_normal(7), rng.standard_normal(7)
    assert np.allclose(o3.Mdiis(1, 0.3, 0.0).step(X, R, 1.0), X + 0.3 * R, rtol=1e-15)
    # b = 1 ("becomes the original DIIS"): X_new = sum c_i Y_i
    md = o3.Mdiis(3, 1.0, 0.0)
    X1, R1 = rng.standard_normal(7), rng.standard_normal(7)
    md.step(X, R, 1.0)
    out = md.step(X1, R1, 1.0)
    S = np.array([[R @ R, R @ R1], [R @ R1, R1 @ R1]])
    c = o3.mdiis_coefficients(S)
    assert np.allclose(out, c[0] * (X + R) + c[1] * (X1 + R1), rtol=1e-13)


def test_mdiis_circular_overwrite_and_restart():
    md = o3.Mdiis(2, 0.5, 10.0)
    e = np.eye(4)
    md.step(e[0], 0.1 * e[0], 0.1)
    md.step(e[1], 0.1 * e[1], 0.1)
    md.step(e[2], 0.1 * e[2], 0.1)
    assert len(md.X) == 2 and np.array_equal(md.X[0], e[1])                  # oldest dropped
    out = md.step(e[3], 5.0 * e[3], 5.0)                                    # rms jumps > 10 x min: restart
    assert len(md.X) == 1 and np.array_equal(md.X[0], e[2])
    assert np.allclose(out, e[2] + 0.5 * 0.1 * e[2])


# ------------------------------------------------------------------------------------------------
# Whole-loop pins
# ------------------------------------------------------------------------------------------------
def _water_oracle(n=16, dr=0.5, **kw):
    w = water()
    orc = o3.Rism3dOracle(n, dr, w.n_v, **kw)
    return w, orc


def test_p2_null_solute_gives_exact_zero():
    w, orc = _water_oracle()
    orc.set_solvent_chi(w.q, w.sigma, w.eps, w.rho, *synthetic_chi(2, w.rho))
    orc.set_solute(np.array([[0.3, -0.2, 0.1], [1.5, 0, 0]]), np.zeros(2), np.array([3.0, 2.0]), np.zeros(2))
    n_done, rms = orc.iterate(3)
    assert rms == 0.0
    assert np.all(orc.get_field("G") == 1.0) and np.all(orc.get_field("C_SR") == 0.0)
    assert orc.free_energy()[0] == 0.0


@pytest.mark.parametrize("closure,order", [("KH", 1), ("PSE", 2), ("HNC", 1)])
def test_p3_identity_chi_closed_form(closure, order):
    # chi = I (ideal gas of sites), uncharged LJ solute: fixed point t = 0, g = closure(-beta u) pointwise,
    # dmu = kT dV sum rho [ -h - ... ] evaluated directly from the closed form.
    w, orc = _water_oracle(closure=closure, pse_order=order, mdiis_nvec=3, mdiis_b=1.0)
    orc.set_solvent_chi(w.q, w.sigma, w.eps, w.rho, *identity_chi(2))
    xyz = np.array([[0.1, 0.2, -0.3], [1.9, 0.2, -0.3]])
    orc.set_solute(xyz, np.zeros(2), np.array([3.0, 2.6]), np.array([0.15, 0.4]))
    # one pass from a NON-zero start must already land on t' = 0 (h~ = c~  =>  t' = h - c_sr = 0)
    rng = np.random.default_rng(0)
    t0 = 0.1 * rng.standard_normal(orc.t.shape)
    t1, _, _ = orc.rism_map(t0)
    assert np.max(np.abs(t1)) < 1e-12
    orc.iterate(4)
    bu = o3.beta_u_at(orc.points, xyz, np.zeros(2), np.array([3.0, 2.6]), np.array([0.15, 0.4]),
                      w.q, w.sigma, w.eps, orc.beta, orc.r_min).reshape(orc.t.shape)
    d = -bu
    if closure == "HNC":
        g_exact = np.exp(d)
    elif closure == "KH":
        g_exact = np.where(d > 0, 1 + d, np.exp(np.minimum(d, 0)))
    else:
        g_exact = np.where(d > 0, 1 + d + d * d / 2, np.exp(np.minimum(d, 0)))
    g = orc.get_field("G")
    assert np.max(np.abs(g - g_exact)) < 1e-12
    # closed-form SFE: c = h - t = h (t = 0)  =>  integrand = -h - h^2/2 + h^2/2 - B = -h - B
    h = g_exact - 1
    if closure == "HNC":
        integrand = -h
    elif closure == "KH":
        integrand = -h - np.where(h > 0, 0.5 * h * h, 0.0)
    else:
        integrand = -h - np.where(d > 0, d ** 3 / 6.0, 0.0)
    dmu_exact = orc.kT * orc.dr ** 3 * sum(w.rho[gm] * integrand[gm].sum() for gm in range(2))
    assert orc.free_energy()[0] == pytest.approx(dmu_exact, rel=1e-12)


def test_p4_identity_chi_charged_solute_measures_only_tail_aliasing():
    # chi = I with a charged solute: t' = f(r) - DFT^-1[f~(k)], the aliasing / anti-periodic image error of
    # the analytic tail; must shrink when the box grows (loose, reported).
    errs = []
    for n in (16, 32):
        w, orc = _water_oracle(n=n, dr=0.5)
        orc.set_solvent_chi(w.q, w.sigma, w.eps, w.rho, *identity_chi(2))
        orc.set_solute(np.zeros((1, 3)), np.array([1.0]), np.array([2.35]), np.array([0.13]))
        t1, g, c_sr = orc.rism_map(orc.t)
        # Y = X + h + 1 - g with h = DFT^-1[c~_sr - f~] = c_sr - DFT^-1[f~]  =>  Y = f - DFT^-1[f~]
        direct = orc.f - o3.shifted_dft_inverse(orc.f_tilde, orc.dr, orc.origin).real
        assert np.max(np.abs(t1 - direct)) < 1e-9 * np.max(np.abs(orc.f))
        c = n // 2
        errs.append(np.max(np.abs(direct[:, c - 4:c + 4, c - 4:c + 4, c - 4:c + 4])))
    assert errs[1] < errs[0]


def _run_converged(orc, tol=1e-10, max_iter=400):
    n_done, rms = orc.iterate(max_iter, tol)
    assert rms < tol, (n_done, rms)
    return n_done


def test_p5_site_splitting_invariance():
    # (O,H,H) with a symmetric full-site susceptibility vs (O,H) with the reduced, asymmetric one (Q15):
    # chi_red[g'][g] = sum_{a in g'} chi_full[a][b], b any member of g.
    w = water()
    k0, dk, n_k = 0.03, 0.03, 600
    k = k0 + dk * np.arange(n_k)
    bump = np.exp(-(k / 2.0) ** 2)
    rho = 0.0334
    # full-site chi = omega-like + rho h-like, symmetric, H1 <-> H2 equivalent
    hOO, hOH, hHH, wOH, wHH = -8.0, 5.0, -3.0, 0.6, 0.4
    full = np.zeros((n_k, 3, 3))
    for a in range(3):
        full[:, a, a] = 1.0
    full[:, 0, 0] += rho * hOO * bump
    for hsite in (1, 2):
        full[:, 0, hsite] = full[:, hsite, 0] = wOH * bump + rho * hOH * bump
        full[:, hsite, hsite] += rho * hHH * bump
    full[:, 1, 2] = full[:, 2, 1] = wHH * bump + rho * hHH * bump
    red = np.zeros((n_k, 2, 2))
    red[:, 0, 0] = full[:, 0, 0]
    red[:, 0, 1] = full[:, 0, 1]
    red[:, 1, 0] = full[:, 1, 0] + full[:, 2, 0]
    red[:, 1, 1] = full[:, 1, 1] + full[:, 2, 1]
    sol = make_solute("C2")
    xyz = sol.xyz[:4] * 0.5
    qs = np.array([0.3, -0.2, 0.1, -0.2])
    kw = dict(mdiis_nvec=5, mdiis_b=0.5)
    a = o3.Rism3dOracle(16, 0.5, 3, **kw)
    a.set_solvent_chi(w.q[[0, 1, 1]], w.sigma[[0, 1, 1]], w.eps[[0, 1, 1]], np.full(3, rho), k0, dk, full)
    a.set_solute(xyz, qs, sol.sigma[:4], sol.eps[:4])
    b = o3.Rism3dOracle(16, 0.5, 2, **kw)
    b.set_solvent_chi(w.q, w.sigma, w.eps, w.rho, k0, dk, red)
    b.set_solute(xyz, qs, sol.sigma[:4], sol.eps[:4])
    _run_converged(a, 1e-11)
    _run_converged(b, 1e-11)
    ga, gb = a.get_field("G"), b.get_field("G")
    assert np.max(np.abs(ga[0] - gb[0])) < 1e-9
    assert np.max(np.abs(ga[1] - gb[1])) < 1e-9 and np.max(np.abs(ga[2] - gb[1])) < 1e-9
    assert a.free_energy()[0] == pytest.approx(b.free_energy()[0], rel=1e-9)
    # a transposed chi must NOT pass (the pin has teeth)
    c = o3.Rism3dOracle(16, 0.5, 2, **kw)
    c.set_solvent_chi(w.q, w.sigma, w.eps, w.rho, k0, dk, np.swapaxes(red, 1, 2).copy())
    c.set_solute(xyz, qs, sol.sigma[:4], sol.eps[:4])
    c.iterate(400, 1e-11)
    assert np.max(np.abs(c.get_field("G")[0] - gb[0])) > 1e-4


def test_p6_axis_permutation_and_reflection():
    w = water()
    chi = synthetic_chi(2, w.rho, seed=4)
    sol = make_solute("C2")
    xyz, qs = sol.xyz[:3] * 0.4, np.array([0.4, -0.1, -0.3])

    def run(coords):
        orc = o3.Rism3dOracle(16, 0.5, 2, mdiis_nvec=5)
        orc.set_solvent_chi(w.q, w.sigma, w.eps, w.rho, *chi)
        orc.set_solute(coords, qs, sol.sigma[:3], sol.eps[:3])
        orc.iterate(12)
        return orc.get_field("G")

    g = run(xyz)
    gp = run(xyz[:, [1, 2, 0]])                  # new x = old y, new y = old z, new z = old x
    assert np.max(np.abs(gp - np.transpose(g, (0, 2, 3, 1)))) < 1e-10
    # Reflection: the r-grid {origin + i dr} maps onto itself under i -> n-1-i, i.e. x -> -dr - x (mirror plane
    # at the grid's own centre -dr/2).  The convolution kernel chi(|k|) is real and even on the symmetric
    # half-integer k set, so this symmetry is exact.  (Mirroring about the grid POINT at 0 is NOT a symmetry of
    # the discrete problem: the unpaired -L/2 plane feeds the anti-periodic convolution.)
    refl = xyz.copy()
    refl[:, 0] = -0.5 - refl[:, 0]
    gr = run(refl)
    assert np.max(np.abs(gr - g[:, ::-1])) < 1e-10


def test_p7_accelerator_independence_and_p11_threshold_protocol():
    w = water()
    chi = synthetic_chi(2, w.rho, seed=2)
    sol = make_solute("C2")
    xyz, qs = sol.xyz[:5] * 0.5, np.array([0.3, -0.3, 0.2, -0.1, -0.1])
    res = []
    for M, b, restart in ((1, 0.3, 0.0), (5, 0.5, 10.0), (10, 0.5, 0.0)):
        orc = o3.Rism3dOracle(16, 0.5, 2, mdiis_nvec=M, mdiis_b=b, mdiis_restart=restart)
        orc.set_solvent_chi(w.q, w.sigma, w.eps, w.rho, *chi)
        orc.set_solute(xyz, qs, sol.sigma[:5], sol.eps[:5])
        n1 = orc.iterate(3000, 1e-6)[0]
        mu6 = orc.free_energy()[0]
        orc.iterate(3000, 1e-8)
        mu8 = orc.free_energy()[0]
        orc.iterate(3000, 1e-10)
        res.append((orc.get_field("G"), orc.free_energy()[0], n1))
        assert abs(mu6 - mu8) < 2e-6 * abs(mu8) + 1e-7          # P11
    for g, mu, _ in res[1:]:
        assert np.max(np.abs(g - res[0][0])) < 1e-8
        assert mu == pytest.approx(res[0][1], rel=1e-8)
    assert res[1][2] < res[0][2]                                 # MDIIS beats damped Picard
    # log-linear decay: rms falls by orders of magnitude, monotone on a coarse scale
    h = orc.rms_history
    assert h[-1] < 1e-3 * h[0]


# ------------------------------------------------------------------------------------------------
# Modified Anderson (Eq. 34-39; Q17)
# ------------------------------------------------------------------------------------------------
def test_anderson_two_histories_is_exact_on_a_2d_affine_map():
    """Textbook property: Anderson mixing with m histories solves a linear fixed-point problem of dimension m exactly
    at step m + 1 (s = 0, b = 1 is the original method)."""
    rng = np.random.default_rng(0)
    A = rng.uniform(-0.4, 0.4, (2, 2))
    y0 = rng.standard_normal(2)
    exact = np.linalg.solve(np.eye(2) - A, y0)
    acc = o3.ModifiedAnderson(1.0, (0.0, 0.0), np.ones(1))
    X = np.zeros((1, 2))
    errs = []
    for _ in range(4):
        R = (A @ X[0] + y0)[None] - X
        errs.append(np.abs(X[0] - exact).max())
        X = acc.step(X, R, 0.0)
    assert errs[2] > 1e-3 and errs[3] < 1e-13
    # the first two steps are Picard steps X + b R
    acc = o3.ModifiedAnderson(0.6, (0.2, 0.0), np.ones(1))
    X0 = np.array([[0.3, -0.1]])
    R0 = np.array([[0.5, 0.25]])
    assert np.allclose(acc.step(X0, R0, 0.0), X0 + 0.6 * R0)


def test_anderson_theta_solves_the_least_squares_problem_and_uses_the_weights():
    rng = np.random.default_rng(3)
    R = rng.standard_normal((3, 2, 50))                  # R0, R1, R2 as [gamma][r]
    w = np.array([1.0 / 0.0334, 1.0 / 0.0668])
    S = np.array([[o3.gram_weighted(R[i], R[j], w) for j in range(3)] for i in range(3)])
    th = o3.anderson_theta(S)
    # brute force: minimise sum_g w_g |R0 - th1 (R0 - R1) - th2 (R0 - R2)|^2 with a library least-squares routine
    sw = np.sqrt(w)[:, None]
    D = np.stack([((R[0] - R[1]) * sw).ravel(), ((R[0] - R[2]) * sw).ravel()], axis=1)
    ref = np.linalg.lstsq(D, (R[0] * sw).ravel(), rcond=None)[0]
    assert np.allclose(th, ref, rtol=1e-10)
    assert not np.allclose(th, o3.anderson_theta(np.array([[o3.gram(R[i], R[j]) for j in range(3)] for i in range(3)])))
    assert np.all(o3.anderson_theta(np.zeros((3, 3))) == 0.0)


def test_anderson_update_is_the_combination_of_z_entries():
    """Eq. 34-39 collapse to X_new = (1 - a1 - a2) Z0 + a1 Z1 + a2 Z2 with Z_k = X_k + b R_k, a_i = theta_i + s_i --
    the form the CUDA path uses."""
    rng = np.random.default_rng(5)
    b, s = 0.6, (0.2, 0.05)
    acc = o3.ModifiedAnderson(b, s, np.array([2.0, 0.5]))
    Xs = [rng.standard_normal((2, 30)) for _ in range(3)]
    Rs = [rng.standard_normal((2, 30)) for _ in range(3)]
    for X, R in zip(Xs[:2], Rs[:2]):
        acc.step(X, R, 0.0)
    out = acc.step(Xs[2], Rs[2], 0.0)
    S = np.array([[o3.gram_weighted(Rs[2 - i], Rs[2 - j], acc.w) for j in range(3)] for i in range(3)])
    a = o3.anderson_theta(S) + np.array(s)
    Z = [Xs[2 - k] + b * Rs[2 - k] for k in range(3)]
    assert np.allclose(out, (1 - a[0] - a[1]) * Z[0] + a[0] * Z[1] + a[1] * Z[2], rtol=1e-12, atol=1e-12)


def test_anderson_reaches_the_same_fixed_point_as_mdiis():
    sv = water()
    k0, dk, chi = synthetic_chi(2, sv.rho)
    sol = make_solute("C1")
    res = []
    for kw in (dict(mdiis_nvec=5), dict(accelerator="ANDERSON", mdiis_b=0.6, anderson_s=(0.2, 0.0))):
        orc = o3.Rism3dOracle(16, 0.6, 2, **kw)
        orc.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
        orc.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps)
        n, rms = orc.iterate(2000, 1e-10)
        assert rms < 1e-10
        res.append((orc.get_field("G"), orc.free_energy()[0]))
    assert np.max(np.abs(res[0][0] - res[1][0])) < 1e-8
    assert abs(res[0][1] - res[1][1]) < 1e-8 * abs(res[0][1])


# ------------------------------------------------------------------------------------------------
# Partial molar volume, Eq. 19
# ------------------------------------------------------------------------------------------------
def test_pmv_ideal_gas_solvent_is_the_second_virial_coefficient():
    """One-site ideal-gas solvent (chi = 1, rho kT chi_T = 1), HNC, LJ solute: the fixed point is g = exp(-beta u)
    (pin P3), so Eq. 19 gives V - 1/rho = -int (exp(-beta u) - 1) dr = 2 B_2(T), the textbook second virial
    coefficient of the pair, here from an independent radial quadrature."""
    rho, T = 0.02, 298.0
    kT = o3.K_BOLTZMANN * T
    sig_v, eps_v, sig_u, eps_u = 3.0, 0.15, 3.4, 0.2
    n, dr = 64, 0.3
    orc = o3.Rism3dOracle(n, dr, 1, closure="HNC", mdiis_nvec=3, origin=(-9.45, -9.45, -9.45))   # atom between grid points
    orc.set_solvent_chi([0.0], [sig_v], [eps_v], [rho], *identity_chi(1, n_k=1300, dk=0.015, k0=0.015))
    orc.set_solute(np.zeros((1, 3)), [0.0], [sig_u], [eps_u])
    orc.iterate(3, 0.0)
    chi_t = 1.0 / (rho * kT)
    v, c_int = orc.pmv(chi_t)
    r = np.linspace(1e-4, 9.6 * np.sqrt(3), 400001)
    s, e = 0.5 * (sig_v + sig_u), np.sqrt(eps_v * eps_u)
    mayer = np.exp(-4.0 * e * ((s / r) ** 12 - (s / r) ** 6) / kT) - 1.0
    # the cubic box cuts the integration domain; beyond the inscribed sphere the integrand is ~1e-4 r^2, so compare
    # with the radial integral over the box's volume-equivalent region by integrating the same function on the grid
    # of the oracle directly (closed form on the grid) and, loosely, against the radial quadrature to 9.6 A
    rr = np.sqrt(np.sum(orc.points ** 2, axis=1))
    on_grid = dr ** 3 * np.sum(np.exp(-4.0 * e * ((s / rr) ** 12 - (s / rr) ** 6) / kT) - 1.0)
    assert abs(c_int[0] - on_grid) < 1e-9 * abs(on_grid)
    assert abs(v - (1.0 / rho - on_grid)) < 1e-9 * abs(v)
    sel = r < 9.6
    radial = np.trapezoid(4.0 * np.pi * r[sel] ** 2 * mayer[sel], r[sel])
    shell = dr ** 3 * np.sum((np.exp(-4.0 * e * ((s / rr) ** 12 - (s / rr) ** 6) / kT) - 1.0)[rr < 9.6])
    assert abs(shell - radial) < 2e-2 * abs(radial)      # 0.3 A grid against the exact radial integral


def test_pmv_null_solute_and_sign():
    sv = water()
    k0, dk, chi = synthetic_chi(2, sv.rho)
    orc = o3.Rism3dOracle(16, 0.6, 2)
    orc.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    orc.set_solute(np.array([[0.1, 0.0, 0.2]]), [0.0], [3.0], [0.0])
    orc.iterate(2, 0.0)
    v, c_int = orc.pmv(0.7)
    assert np.all(c_int == 0.0) and v == orc.kT * 0.7    # nothing there: the ideal term kT chi_T alone
    sol = make_solute("C1")
    orc.set_solute(sol.xyz, 0.0 * sol.q, sol.sigma, sol.eps)
    orc.iterate(200, 1e-9)
    v2, c2 = orc.pmv(0.7)
    assert v2 > v and np.dot(sv.rho, c2) < 0.0           # a repulsive core excludes solvent: c integrates to < 0


# ------------------------------------------------------------------------------------------------
# Solvent-induced gradient on the solute atoms
# ------------------------------------------------------------------------------------------------
def test_gradient_closed_form_in_an_ideal_gas_solvent():
    """chi = I, HNC: g = exp(-beta u) pointwise and dmu = -kT rho dV sum_r (exp(-beta u) - 1), so the gradient formula
    must equal the derivative of that grid sum with respect to the atom position -- taken here by central
    differences of the closed form, which is built from the potential alone."""
    rho, sig_v, eps_v = 0.02, 3.0, 0.15
    n, dr = 24, 0.5
    xyz = np.array([[0.37, -0.21, 0.13], [2.9, 0.4, -0.6]])
    q, sig, eps = np.array([0.0, 0.0]), np.array([3.2, 2.8]), np.array([0.2, 0.1])
    orc = o3.Rism3dOracle(n, dr, 1, closure="HNC", mdiis_nvec=2)
    orc.set_solvent_chi([0.0], [sig_v], [eps_v], [rho], *identity_chi(1, n_k=1000, dk=0.02, k0=0.02))
    orc.set_solute(xyz, q, sig, eps)
    orc.iterate(3, 0.0)
    grad = orc.solvation_gradient()

    def closed_form(pos):
        bu = o3.beta_u_at(orc.points, pos, q, sig, eps, np.array([0.0]), np.array([sig_v]), np.array([eps_v]), orc.beta, 1e-3)
        return -orc.kT * rho * dr ** 3 * float(np.sum(np.exp(-bu[0]) - 1.0))

    assert abs(orc.free_energy()[0] - closed_form(xyz)) < 1e-10
    h = 1e-5
    for a in range(2):
        for k in range(3):
            p1, p2 = xyz.copy(), xyz.copy()
            p1[a, k] += h
            p2[a, k] -= h
            fd = (closed_form(p1) - closed_form(p2)) / (2 * h)
            assert abs(grad[a, k] - fd) < 1e-6 * max(1.0, abs(fd)), (a, k, grad[a, k], fd)


def test_gradient_vanishes_by_symmetry_and_matches_finite_differences_of_the_solve():
    sv = water()
    k0, dk, chi = synthetic_chi(2, sv.rho)
    # one ion at the centre of a grid whose points are symmetric about it (origin at -(n-1)/2 dr: the default grid
    # has an unpaired -L/2 face, which leaves a net pull on a finite box)
    orc = o3.Rism3dOracle(16, 0.6, 2, mdiis_nvec=5, origin=(-4.5, -4.5, -4.5))
    orc.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    sol = make_solute("C1")
    orc.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps)
    orc.iterate(500, 1e-10)
    assert np.max(np.abs(orc.solvation_gradient())) < 1e-9 * np.max(np.abs(orc.get_field("G"))) * 1e3
    # an off-centre LJ pair: the stationarity of the free-energy functional makes the gradient formula the derivative
    # of the converged dmu; on the grid this holds to discretisation accuracy
    xyz = np.array([[0.31, 0.17, -0.23], [2.6, 0.5, 0.4]])
    qs, sig, eps = np.zeros(2), np.array([3.0, 2.7]), np.array([0.15, 0.1])

    def dmu(pos):
        o = o3.Rism3dOracle(16, 0.6, 2, mdiis_nvec=5)
        o.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
        o.set_solute(pos, qs, sig, eps)
        o.iterate(2000, 1e-11)
        return o, o.free_energy()[0]

    o0, _ = dmu(xyz)
    grad = o0.solvation_gradient()
    h = 1e-3
    for a, k in ((0, 0), (1, 2)):
        p1, p2 = xyz.copy(), xyz.copy()
        p1[a, k] += h
        p2[a, k] -= h
        fd = (dmu(p1)[1] - dmu(p2)[1]) / (2 * h)
        assert abs(grad[a, k] - fd) < 2e-2 * max(abs(fd), 0.05), (a, k, grad[a, k], fd)


def test_gradient_coulomb_and_lj_terms_against_the_differenced_potential():
    """Pins du/dR term by term, INCLUDING C q_a q_g / r^3 (PAPER.md:188-190 with u of Eq. 22): with g held fixed, the
    gradient is the g-weighted sum of d(beta u)/dR_a, taken here by central differences of beta_u_at (itself pinned
    by hand values in test_potential_hand_values) -- a charged solute in a charged solvent, so that a wrong sign,
    factor or power in the Coulomb term fails."""
    sv = water()
    k0, dk, chi = synthetic_chi(2, sv.rho)
    xyz = np.array([[0.31, 0.17, -0.23], [2.4, -0.5, 0.6], [-1.1, 1.9, 0.35]])
    q, sig, eps = np.array([0.7, -0.4, 0.25]), np.array([3.0, 2.7, 3.3]), np.array([0.15, 0.1, 0.2])
    orc = o3.Rism3dOracle(16, 0.6, 2, mdiis_nvec=5)
    orc.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    orc.set_solute(xyz, q, sig, eps)
    orc.iterate(30, 0.0)
    g = orc.get_field("G").reshape(2, -1)
    grad = orc.solvation_gradient()
    assert np.max(np.abs(grad)) > 1.0                                     # a non-trivial case
    h = 1e-5
    for a in range(3):
        for k in range(3):
            p1, p2 = xyz.copy(), xyz.copy()
            p1[a, k] += h
            p2[a, k] -= h
            u1 = o3.beta_u_at(orc.points, p1, q, sig, eps, sv.q, sv.sigma, sv.eps, orc.beta, orc.r_min)
            u2 = o3.beta_u_at(orc.points, p2, q, sig, eps, sv.q, sv.sigma, sv.eps, orc.beta, orc.r_min)
            fd = orc.kT * orc.dr ** 3 * float(np.sum(sv.rho[:, None] * g * (u1 - u2))) / (2 * h)
            assert abs(grad[a, k] - fd) < 1e-6 * max(1.0, abs(fd)), (a, k, grad[a, k], fd)
    # the Coulomb part alone: LJ switched off (eps = 0) leaves only C q_a q_g (r - R_a) / r^3
    orc.set_solute(xyz, q, sig, np.zeros(3))
    gc = orc.solvation_gradient()                                         # t = f: g = closure(-beta u_coul)
    gg = orc.get_field("G").reshape(2, -1)
    for a in range(3):
        d = orc.points - xyz[a]
        r3 = np.sum(d * d, axis=1) ** 1.5
        expect = sum(sv.rho[gam] * orc.dr ** 3 * o3.COULOMB * q[a] * sv.q[gam] * np.sum(gg[gam][:, None] * d / r3[:, None], axis=0)
                     for gam in range(2))
        assert np.max(np.abs(gc[a] - expect)) < 1e-10 * max(1.0, np.max(np.abs(expect)))


def test_gradient_of_a_charged_pair_matches_finite_differences_of_the_converged_free_energy():
    """The finite-difference pin of the LJ pair above repeated with a CHARGED off-centre pair in charged water: the
    converged dmu (Eq. 18) differentiated numerically against the gradient formula, Coulomb term included.  The solve
    sees the long-range part of c through the anti-periodic images of the half-integer k grid (pin P4) while the
    formula uses the image-free u of Eq. 22, so the two agree up to a box effect: it must be small on a 19 A box and
    shrink with the box (measured: 4.4 % at 9.6 A, 0.45 % at 19.2 A; a wrong Coulomb sign or factor is off by O(1))."""
    sv = water()
    k0, dk, chi = synthetic_chi(2, sv.rho)
    xyz = np.array([[0.31, 0.17, -0.23], [2.6, 0.5, 0.4]])
    qs, sig, eps = np.array([0.5, -0.5]), np.array([3.0, 2.7]), np.array([0.15, 0.1])

    def dmu(pos, n):
        o = o3.Rism3dOracle(n, 0.6, 2, mdiis_nvec=5)
        o.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
        o.set_solute(pos, qs, sig, eps)
        _, rms = o.iterate(3000, 1e-11)
        assert rms < 1e-11
        return o, o.free_energy()[0]

    h, err = 1e-3, {}
    for n in (16, 32):
        grad = dmu(xyz, n)[0].solvation_gradient()
        p1, p2 = xyz.copy(), xyz.copy()
        p1[0, 0] += h
        p2[0, 0] -= h
        fd = (dmu(p1, n)[1] - dmu(p2, n)[1]) / (2 * h)
        assert abs(fd) > 100.0                                            # Coulomb dominated
        err[n] = abs(grad[0, 0] - fd) / abs(fd)
    assert err[32] < 1e-2 and err[32] < 0.25 * err[16], err


# ------------------------------------------------------------------------------------------------
# Dynamic damping b = -0.2 log R (Q18)
# ------------------------------------------------------------------------------------------------
def test_dynamic_damping_values_and_update_formula():
    assert o3.dynamic_damping(1e-1, 0.1, 1.0) == pytest.approx(0.2, abs=1e-15)
    assert o3.dynamic_damping(1e-3, 0.1, 1.0) == pytest.approx(0.6, abs=1e-15)
    assert o3.dynamic_damping(10.0 ** -2.5, 0.1, 1.0) == pytest.approx(0.5, abs=1e-15)
    assert o3.dynamic_damping(5.0, 0.1, 1.0) == 0.1            # R >= 1 would give b <= 0: clamped from below
    assert o3.dynamic_damping(1e-9, 0.1, 1.0) == 1.0           # plain DIIS (b = 1) near convergence
    # the CURRENT b multiplies every stored residual (Eq. 40: b stands in front of the sum)
    rng = np.random.default_rng(3)
    md = o3.Mdiis(3, 0.5, 0.0, dynamic_b=(0.1, 1.0))
    Xs, Rs, rs = [rng.standard_normal(7) for _ in range(3)], [rng.standard_normal(7) for _ in range(3)], [1e-1, 1e-2, 1e-4]
    for X, R, r in zip(Xs, Rs, rs):
        out = md.step(X, R, r)
    S = np.array([[np.dot(a, b) for b in Rs] for a in Rs])
    c = o3.mdiis_coefficients(S)
    b_now = 0.8                                                # -0.2 log10(1e-4)
    assert np.allclose(out, sum(c[i] * (Xs[i] + b_now * Rs[i]) for i in range(3)), rtol=1e-12, atol=1e-12)


def test_dynamic_damping_reaches_the_same_fixed_point_faster():
    """The fixed point does not depend on the damping schedule (invariant P7); on the small ion case the dynamic rule
    needs fewer iterations than the static b = 0.5 (the paper's claim)."""
    sv = water()
    k0, dk, chi = synthetic_chi(2, sv.rho)
    sol = make_solute("C1")
    out = []
    for dyn in (None, (0.1, 1.0)):
        orc = o3.Rism3dOracle(16, 0.6, 2, mdiis_nvec=5, mdiis_b=0.5, mdiis_dynamic_b=dyn)
        orc.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
        orc.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps)
        n, rms = orc.iterate(3000, 1e-10)
        assert rms < 1e-10
        out.append((n, orc.get_field("G"), orc.free_energy()[0]))
    assert np.max(np.abs(out[0][1] - out[1][1])) < 1e-8
    assert abs(out[0][2] - out[1][2]) < 1e-8 * abs(out[0][2])
    assert out[1][0] <= out[0][0]
