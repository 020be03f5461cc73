"""-m gpu parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Tolerances: BASELINE.json north_star -- max|dg| <= 1e-9 after 50 fixed iterations,
converged solvation free energy to 1e-7 relative."""
import numpy as np
import pytest

from oracle import rism3d as o3
from tests._gpu_util import make_pair, oracle_spectrum_in_gpu_layout
from tests._util import synthetic_chi
from workloads import make_solute, solvent_by_name, water

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    return torch


# ---- the shifted 3D transform pair alone -----------------------------------------
@pytest.mark.parametrize("n,nv", [(8, 2), (16, 1), (16, 4), (32, 2), (64, 4), (128, 2), (128, 4), (256, 4)])
def test_fft_pair_matches_oracle(n, nv):
    """element by element, up to the transform size and site count of the benchmarked configuration (256, 4)"""
    torch = _torch()
    import paper_2403_01039_b200 as lib
    rng = np.random.default_rng(n + nv)
    f = rng.standard_normal((nv, n, n, n))
    s = lib.Solver(n, 0.5, nv)
    spec = s.fft_forward(torch.from_numpy(f).cuda()).cpu().numpy()
    ref = oracle_spectrum_in_gpu_layout(f, 0.5)
    scale = np.max(np.abs(ref))
    assert np.max(np.abs(spec - ref)) < 2e-14 * scale * np.log2(n)
    back = s.fft_inverse(torch.from_numpy(ref).cuda()).cpu().numpy()
    assert np.max(np.abs(back - f)) < 2e-14 * np.log2(n) * np.max(np.abs(f))


@pytest.mark.parametrize("n,nv", [(256, 1), (512, 2)])
def test_fft_round_trip_and_sampled_lines_large(n, nv):
    """Full-size lines: round trip = identity, Parseval, and sampled k points against the defining sum."""
    torch = _torch()
    import paper_2403_01039_b200 as lib
    g = torch.Generator(device="cuda").manual_seed(n)
    f = torch.randn((nv, n, n, n), dtype=torch.float64, device="cuda", generator=g)
    s = lib.Solver(n, 0.5, nv, mdiis_nvec=1)
    spec = s.fft_forward(f)
    back = s.fft_inverse(spec)
    assert float((back - f).abs().max()) < 1e-12
    # Parseval on the half spectrum: sum |f|^2 = (2 / N) sum_half |F|^2
    lhs = float((f * f).sum())
    rhs = 2.0 * float((spec.abs() ** 2).sum()) / n ** 3
    assert abs(lhs - rhs) < 1e-10 * lhs
    # sampled outputs from the definition F(j) = sum_r f(r) exp(-2 pi i ((jx+1/2) x + (jy+1/2) y + (jz+1/2) z)/n)
    rng = np.random.default_rng(7)
    idx = torch.arange(n, device="cuda", dtype=torch.float64)
    for _ in range(4):
        jx, jy, p = (int(v) for v in rng.integers(0, [n, n, n // 2]))
        ex = torch.exp(-2j * np.pi * (jx + 0.5) * idx / n)
        ey = torch.exp(-2j * np.pi * (jy + 0.5) * idx / n)
        ez = torch.exp(-2j * np.pi * (2 * p + 0.5) * idx / n)
        val = torch.einsum("xyz,x,y,z->", f[0].to(torch.complex128), ex, ey, ez)
        assert abs(complex(spec[jx, jy, p, 0]) - complex(val)) < 1e-9 * n ** 1.5


# ---- setup kernels: potential, phi, phi~ through one map evaluation ----------------------------------------
@pytest.mark.parametrize("cfg,n", [("C1", 32), ("C2", 32)])
def test_setup_fields_match_oracle(cfg, n):
    orc, gpu, _, _ = make_pair(cfg, n_override=n)
    W = gpu.get_field("W")
    Wo = orc.get_field("W")
    finite = np.abs(Wo) < 600.0                       # beyond that exp() underflows on both sides
    assert np.max(np.abs(W - Wo)[finite]) < 1e-10
    assert np.all(W[~finite] < -600.0)
    assert np.max(np.abs(gpu.get_field("PHI", 0) - orc.phi)) < 1e-11 * np.max(np.abs(orc.phi)) + 1e-13


def test_setup_with_cutoff_matches_oracle_pair_set():
    sol = make_solute("C3")
    orc, gpu, _, _ = make_pair(n=32, spacing=1.5, solvent="water_nacl_0.1M", solute=sol, rcut=9.0, M=4)
    W, Wo = gpu.get_field("W"), orc.get_field("W")
    finite = np.abs(Wo) < 600.0
    assert np.max(np.abs(W - Wo)[finite]) < 1e-10     # a single differing pair would show up at >= 1e-6


@pytest.mark.parametrize("n,spacing,kappa,rcut", [(64, 1.0, 1.0, 50.0), (32, 1.5, 3.0, 16.0), (32, 1.5, 4.0, 12.0)])
def test_cutoff_beyond_the_screening_range_keeps_lennard_jones(n, spacing, kappa, rcut):
    """rcut > 40/kappa: between the distance where exp(-kappa r) vanishes in double precision and the cutoff, a
    pair still contributes its Lennard-Jones term (~1e-7 each at these distances) -- Eq. 22 with the cutoff of Q12."""
    sol = make_solute("C3")
    orc, gpu, _, _ = make_pair(n=n, spacing=spacing, solvent="water_nacl_0.1M", solute=sol, rcut=rcut, M=4, kappa=kappa)
    assert rcut > 40.0 / kappa
    W, Wo = gpu.get_field("W"), orc.get_field("W")
    finite = np.abs(Wo) < 600.0
    assert np.max(np.abs(W - Wo)[finite]) < 1e-10
    assert np.max(np.abs(gpu.get_field("PHI", 0) - orc.phi)) < 1e-11 * np.max(np.abs(orc.phi))


# ---- the loop: 50 fixed iterations, max |dg| <= 1e-9 -------------------------------------------------------
@pytest.mark.parametrize("cfg,n", [("C1", 32), ("C2", 64)])
def test_fifty_iterations_match_oracle(cfg, n):
    orc, gpu, _, _ = make_pair(cfg, n_override=n)
    orc.iterate(50, 0.0)
    nd, rms = gpu.iterate(50, 0.0)
    assert nd == 50
    assert abs(rms - orc.rms_history[-1]) <= 1e-9 * max(orc.rms_history[-1], 1e-3)
    hist = gpu.rms_history()
    assert len(hist) == 50
    np.testing.assert_allclose(hist, orc.rms_history, rtol=1e-6, atol=1e-12)
    g, go = gpu.get_field("G"), orc.get_field("G")
    assert np.max(np.abs(g - go)) <= 1e-9
    assert np.max(np.abs(gpu.get_field("TAU") - orc.get_field("TAU"))) <= 1e-9


def test_fifty_iterations_pse2_four_sites():
    """C3's settings (PSE-2, 4 site types, M = 8) on a 32^3 grid with a 40-atom subset of its solute."""
    sol = make_solute("C3")
    keep = np.argsort(np.linalg.norm(sol.xyz, axis=1))[:40]
    from workloads import Solute
    sub = Solute("C3_sub40", sol.xyz[keep], sol.q[keep], sol.sigma[keep], sol.eps[keep])
    orc, gpu, _, _ = make_pair(n=32, spacing=0.75, solvent="water_nacl_0.1M", closure="PSE", pse_order=2, M=8,
                               solute=sub)
    orc.iterate(50, 0.0)
    gpu.iterate(50, 0.0)
    assert np.max(np.abs(gpu.get_field("G") - orc.get_field("G"))) <= 1e-9


def test_picard_m1_fifty_iterations():
    """M = 1 (damped Picard): no small solve involved -- the strict fallback comparison of DESIGN.md."""
    orc, gpu, _, _ = make_pair("C1", n_override=32)
    orc2 = o3.Rism3dOracle(32, 0.5, 2, mdiis_nvec=1, mdiis_b=0.3)
    sv = water()
    from workloads import load_chi
    k0, dk, chi = load_chi("water")
    orc2.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    sol = make_solute("C1")
    orc2.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps)
    import paper_2403_01039_b200 as lib
    g2 = lib.Solver(32, 0.5, 2, mdiis_nvec=1, mdiis_b=0.3)
    g2.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    g2.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps)
    orc2.iterate(50, 0.0)
    g2.iterate(50, 0.0)
    assert np.max(np.abs(g2.get_field("G") - orc2.get_field("G"))) <= 1e-10


# ---- convergence and free energy ---------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,n", [("C1", 32), ("C2", 64)])
def test_converged_free_energy_matches_oracle(cfg, n):
    orc, gpu, _, _ = make_pair(cfg, n_override=n)
    no, ro = orc.iterate(2000, 1e-8)
    ng, rg = gpu.iterate(2000, 1e-8)
    assert ro < 1e-8 and rg < 1e-8
    assert abs(ng - no) <= 2                          # same path up to rounding; may cross the threshold one step apart
    mu_o, site_o = orc.free_energy()
    mu_g, site_g = gpu.free_energy()
    assert abs(mu_g - mu_o) <= 1e-7 * abs(mu_o)
    np.testing.assert_allclose(site_g, site_o, rtol=1e-6, atol=1e-7 * abs(mu_o))
    assert np.max(np.abs(gpu.get_field("G") - orc.get_field("G"))) <= 1e-6


def test_null_solute_is_exact_zero():
    from workloads import Solute
    sol = Solute("null", np.array([[0.3, -0.2, 0.1]]), np.zeros(1), np.array([3.0]), np.zeros(1))
    orc, gpu, _, _ = make_pair(n=16, spacing=0.5, solvent="water", solute=sol)
    nd, rms = gpu.iterate(3, 0.0)
    assert rms == 0.0
    assert np.all(gpu.get_field("G") == 1.0)
    assert gpu.free_energy()[0] == 0.0


def test_identity_chi_closed_form():
    """chi = I, uncharged LJ solute: g = closure(-beta u) pointwise after any number of iterations (pin P3)."""
    from tests._util import identity_chi
    from workloads import Solute
    sv = water()
    sol = Solute("lj", np.array([[0.2, 0.1, -0.3], [2.5, 0.0, 0.4]]), np.zeros(2), np.array([3.0, 2.8]),
                 np.array([0.15, 0.1]))
    orc, gpu, _, _ = make_pair(n=32, spacing=0.5, solvent=sv, chi=identity_chi(2), solute=sol)
    gpu.iterate(5, 0.0)
    g = gpu.get_field("G")
    bu = o3.beta_u_at(orc.points, sol.xyz, sol.q, sol.sigma, sol.eps, sv.q, sv.sigma, sv.eps, orc.beta, 1e-3)
    expect = o3.closure_g(-bu, "KH").reshape(g.shape)
    assert np.max(np.abs(g - expect)) < 1e-12


def test_error_paths():
    import paper_2403_01039_b200 as lib
    sv = water()
    s = lib.Solver(16, 0.5, 2)
    with pytest.raises(lib.Rism3dError) as e:
        s.set_solute(np.zeros((1, 3)), [1.0], [2.0], [0.1])
    assert e.value.status == -3                       # order
    k0, dk, chi = synthetic_chi(2, sv.rho, n_k=50, dk=0.03)
    with pytest.raises(lib.Rism3dError) as e:
        s.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    assert e.value.status == -4                       # chi range
    k0, dk, chi = synthetic_chi(2, sv.rho)
    with pytest.raises(lib.Rism3dError) as e:
        s.set_solvent_chi([1.0, 1.0], sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    assert e.value.status == -5                       # neutrality
    with pytest.raises(lib.Rism3dError):
        lib.Solver(24, 0.5, 2)                        # not a power of two
    with pytest.raises(lib.Rism3dError):
        lib.Solver(16, 0.5, 9)                        # more than 8 site types
    with pytest.raises(lib.Rism3dError):
        lib.Solver(16, 0.5, 2, r_min=0.0)             # a zero clamp would put 1/0 into w (Q11)
    with pytest.raises(lib.Rism3dError):
        lib.Solver(16, 0.5, 2, mdiis_b=0.0)
    with pytest.raises(ValueError):
        s.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho[:1], k0, dk, chi)      # array lengths are checked before the C call
    with pytest.raises(ValueError):
        s.set_solute(np.zeros((2, 3)), [1.0], [2.0], [0.1])
