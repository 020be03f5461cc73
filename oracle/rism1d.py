"""O-1D: the 1D XRISM solvent solve that produces the solvent susceptibility chi, and the 1D
solute-solvent solve for a single spherical site (pin P10).

TEST INFRASTRUCTURE (see oracle/__init__.py).  The paper gives only the equations -- the 1D-RISM
equation (Eq. 4), the closures (Eq. 5-7, with the KH branches read as
in DESIGN.md Q1), the definition X = omega + rho h and the solute-solvent equation
(Eq. 8) -- and defers the numerical procedure to its ref. 7.  The
procedure below is the reading of DESIGN.md "O-1D": full-site formulation, the same analytic
long-range split as the 3D path (Eq. 29-30), radial sine transforms, MDIIS.

Plain numpy float64; the only library steps are a type-I discrete sine transform and a batched small
dense solve.  Units: Angstrom, e, kcal/mol, K.
"""
from __future__ import annotations

import math

import numpy as np
from scipy.fft import dst

from .rism3d import COULOMB, K_BOLTZMANN, Mdiis, closure_g, closure_sfe_extra, gram


# ----------------------------------------------------------------------------------------------
# Radial grid and the radial Fourier pair
#   F(k) = 4 pi int f(r) r sin(kr)/k dr        f(r) = 1/(2 pi^2) int F(k) k sin(kr)/r dk
# on r_i = i dr, k_j = j dk, i, j = 1..M-1, dr dk = pi / M  (so sin(k_j r_i) = sin(pi i j / M)).
# ----------------------------------------------------------------------------------------------
class RadialGrid:
    def __init__(self, n_points: int, dr: float):
        self.M = int(n_points)
        self.dr = float(dr)
        self.dk = math.pi / (self.M * self.dr)
        i = np.arange(1, self.M)
        self.r = i * self.dr
        self.k = i * self.dk

    def forward(self, f: np.ndarray) -> np.ndarray:
        """f[..., M-1] on r -> F[..., M-1] on k:  F(k_j) = (4 pi dr / k_j) sum_i r_i f(r_i) sin(k_j r_i)."""
        return (2.0 * math.pi * self.dr / self.k) * dst(f * self.r, type=1, axis=-1)   # dst-I = 2 sum sin

    def inverse(self, F: np.ndarray) -> np.ndarray:
        """F[..., M-1] on k -> f on r:  f(r_i) = (dk / (2 pi^2 r_i)) sum_j k_j F(k_j) sin(k_j r_i)."""
        return (self.dk / (4.0 * math.pi ** 2 * self.r)) * dst(F * self.k, type=1, axis=-1)


# ----------------------------------------------------------------------------------------------
# Pair functions
# ----------------------------------------------------------------------------------------------
def lj_pair(r, sig_a, eps_a, sig_b, eps_b):
    """4 eps_ab ((s_ab/r)^12 - (s_ab/r)^6), Lorentz-Berthelot (Q4)."""
    s = 0.5 * (sig_a + sig_b)
    e = math.sqrt(eps_a * eps_b)
    sr6 = (s / r) ** 6
    return 4.0 * e * (sr6 * sr6 - sr6)


def f_long_r(r, qq, beta, kappa):
    """beta C q_a q_b (1 - exp(-kappa r)) / r   (Eq. 29 for one pair)."""
    return beta * COULOMB * qq * (-np.expm1(-kappa * r)) / r


def f_long_k(k, qq, beta, kappa):
    """4 pi beta C q_a q_b kappa^2 / (k^2 (k^2 + kappa^2))   (Eq. 30 for one pair)."""
    return 4.0 * math.pi * beta * COULOMB * qq * kappa ** 2 / (k * k * (k * k + kappa ** 2))


def omega_k(k, bond, species):
    """Intramolecular matrix w_ab(k): 1 on the diagonal, sin(k l)/(k l) for bonded sites of the same
    species, 0 across species  -> [M-1][n_s][n_s]."""
    n_s = len(species)
    W = np.zeros((len(k), n_s, n_s))
    for a in range(n_s):
        for b in range(n_s):
            if a == b:
                W[:, a, b] = 1.0
            elif species[a] == species[b]:
                x = k * bond[a, b]
                W[:, a, b] = np.sin(x) / x
    return W


# ----------------------------------------------------------------------------------------------
# Solvent-solvent XRISM  (Eq. 4)
# ----------------------------------------------------------------------------------------------
class Xrism1d:
    """Full-site solvent-solvent RISM.  Iteration variable tau_ab(r) = t_ab - f_ab (t = h - c),
    symmetric in (a, b); one pass:
        g = closure(w + tau),  w = -beta u + f          (Eq. 5-7)
        c_sr = g - 1 - tau ;  C(k) = C_sr(k) - F(k)      (long-range split, Eq. 29-30)
        H(k) = (I - W C R)^-1 W C W ,  R = diag(rho_a)   (Eq. 4 solved for h at each k)
        tau' (k) = H - C_sr ,  back to r."""

    def __init__(self, solvent, temperature=298.0, closure="KH", pse_order=1, n_points=16384,
                 dr=0.025, kappa=1.0):
        self.sv = solvent
        self.grid = RadialGrid(n_points, dr)
        self.beta = 1.0 / (K_BOLTZMANN * temperature)
        self.closure, self.pse_order, self.kappa = closure, pse_order, float(kappa)
        sv = solvent
        self.n_s = sv.n_s
        self.q = sv.q[sv.site_type]
        self.sig = sv.sigma[sv.site_type]
        self.eps = sv.eps[sv.site_type]
        self.rho_site = sv.species_rho[sv.site_species]          # species number density per full site
        self.W = omega_k(self.grid.k, sv.bond, sv.site_species)   # [k][a][b]
        self.tau = np.zeros((self.n_s, self.n_s, self.grid.M - 1))
        self.set_charge_scale(1.0)

    def set_charge_scale(self, lam: float):
        """w_ab(r) = -beta [LJ + C q_a q_b exp(-kappa r)/r] and F_ab(k) with charges scaled by lam."""
        g, n_s = self.grid, self.n_s
        self.lam = float(lam)
        self.w = np.empty((n_s, n_s, g.M - 1))
        self.Fk = np.empty((n_s, n_s, g.M - 1))
        self.fr = np.empty((n_s, n_s, g.M - 1))
        for a in range(n_s):
            for b in range(n_s):
                qq = lam * lam * self.q[a] * self.q[b]
                lj = lj_pair(g.r, self.sig[a], self.eps[a], self.sig[b], self.eps[b])
                self.w[a, b] = -self.beta * (lj + COULOMB * qq * np.exp(-self.kappa * g.r) / g.r)
                self.Fk[a, b] = f_long_k(g.k, qq, self.beta, self.kappa)
                self.fr[a, b] = f_long_r(g.r, qq, self.beta, self.kappa)

    def closure_step(self, tau):
        d = self.w + tau
        gr = closure_g(d, self.closure, self.pse_order)
        return gr, gr - 1.0 - tau

    def h_of_k(self, c_sr):
        """H(k) from C_sr(r) by Eq. 4: returns (H[k][a][b], C_sr(k)[k][a][b])."""
        Csr_k = np.moveaxis(self.grid.forward(c_sr), -1, 0)                # [k][a][b]
        Ck = Csr_k - np.moveaxis(self.Fk, -1, 0)
        WC = self.W @ Ck
        A = np.eye(self.n_s)[None] - WC * self.rho_site[None, None, :]     # I - W C R
        Hk = np.linalg.solve(A, WC @ self.W)
        return Hk, Csr_k

    def rism_map(self, tau):
        gr, c_sr = self.closure_step(tau)
        Hk, Csr_k = self.h_of_k(c_sr)
        tau_new = self.grid.inverse(np.moveaxis(Hk - Csr_k, 0, -1))
        return 0.5 * (tau_new + np.swapaxes(tau_new, 0, 1))                # keep exact (a,b) symmetry

    def solve(self, tol=1e-10, max_iter=5000, nvec=10, b=0.5, restart=10.0, verbose=False):
        md = Mdiis(nvec, b, restart)
        npts = float(self.tau.size)
        rms = float("nan")
        for it in range(max_iter):
            X = self.tau
            R = self.rism_map(X) - X
            rms = math.sqrt(gram(R, R) / npts)
            if verbose and it % 50 == 0:
                print(f"    1D lam={self.lam:.2f} it={it} rms={rms:.3e}", flush=True)
            if not math.isfinite(rms):
                raise FloatingPointError("1D-RISM diverged")
            if rms < tol:
                return it + 1, rms
            self.tau = md.step(X, R, rms)
        raise RuntimeError(f"1D-RISM not converged: rms={rms:.3e} after {max_iter} iterations")

    def solve_with_charge_ramp(self, ramp=(0.0, 0.25, 0.5, 0.75, 1.0), **kw):
        total = 0
        for lam in ramp:
            self.set_charge_scale(lam)
            n, _ = self.solve(**kw)
            total += n
        return total

    # -- results -------------------------------------------------------------------------------
    def g_r(self):
        return self.closure_step(self.tau)[0]

    def chi_full(self):
        """chi^full_ab(k) = w_ab(k) + rho_a H_ab(k)   (X of PAPER.md:109) -> [k][a][b]."""
        _, c_sr = self.closure_step(self.tau)
        Hk, _ = self.h_of_k(c_sr)
        return self.W + self.rho_site[None, :, None] * Hk

    # -- bulk thermodynamics of the solvent -------------------------------------
    def c_sr_k0(self):
        """int c_sr,ab(r) dr = 4 pi dr sum_i r_i^2 c_sr,ab(r_i)  -> [a][b]  (the k = 0 value of the short-range part of the
        site-site direct correlation function of the bulk solvent)."""
        _, c_sr = self.closure_step(self.tau)
        g = self.grid
        return 4.0 * math.pi * g.dr * np.sum(c_sr * g.r ** 2, axis=-1)

    def _rho_rho_c(self):
        """sum_ab rho_a rho_b int c_ab(r) dr over all solvent sites (rho_a = number density of the species site a
        belongs to).  c_ab = c_sr,ab - f_ab; the long-range parts sum to (sum_a rho_a q_a)^2 int(...) = 0 for a neutral
        solvent (the same cancellation as in Eq. 18-19 of the 3D path, Q10), so only c_sr enters."""
        if abs(float(np.dot(self.rho_site, self.q))) > 1e-12:
            raise ValueError("solvent not neutral")
        return float(self.rho_site @ self.c_sr_k0() @ self.rho_site)

    def compressibility(self):
        """Isothermal compressibility chi_T of the bulk solvent, A^3 mol / kcal, 'obtained by the RISM calculation for a
        pure solvent system': the compressibility route,
            1 / (k_B T chi_T) = sum_Gamma rho_Gamma - sum_ab rho_a rho_b int c_ab(r) dr
        (Gamma: species, a, b: sites).  One species: rho k_B T chi_T = 1 / (1 - rho sum_ab c_ab(k = 0))."""
        kT = 1.0 / self.beta
        return 1.0 / (kT * (float(np.sum(self.sv.species_rho)) - self._rho_rho_c()))

    def pressure(self):
        """Bulk pressure of Eq. 20, kcal / (mol A^3):
            P = sum_Gamma rho_Gamma (n_Gamma + 1) / (2 beta) - sum_{gamma lambda} (2 pi rho_gamma rho_lambda / beta) int c r^2 dr
        n_Gamma = number of sites of species Gamma (the paper prints rho_gamma rho_gamma in the second sum: read as
        rho_gamma rho_lambda).  2 pi int c r^2 dr = (1/2) int c dr."""
        kT = 1.0 / self.beta
        n_sites = np.bincount(self.sv.site_species, minlength=len(self.sv.species_rho))
        ideal = float(np.sum(self.sv.species_rho * (n_sites + 1))) / 2.0
        return kT * (ideal - 0.5 * self._rho_rho_c())

    def chi_types(self):
        """Reduce to site TYPES (Q15): chi_{g'g}(k) = sum_{a in g'} chi^full_ab, b any member of g."""
        sv = self.sv
        full = self.chi_full()
        out = np.zeros((full.shape[0], sv.n_v, sv.n_v))
        for gp in range(sv.n_v):
            for gm in range(sv.n_v):
                b = int(np.nonzero(sv.site_type == gm)[0][0])
                for a in np.nonzero(sv.site_type == gp)[0]:
                    out[:, gp, gm] += full[:, a, b]
        return out


# ----------------------------------------------------------------------------------------------
# 1D solute-solvent RISM for ONE spherical solute site  (Eq. 8 with omega_aa' = 1)  -- pin P10
# ----------------------------------------------------------------------------------------------
class IonRism1d:
    """h_g(k) = sum_g' c_g'(k) chi_{g'g}(k) on the radial grid, same closure, kappa and chi table
    as the 3D solve; SFE by Eq. 10 (KH) / Eq. 9 (HNC), the radial form of Eq. 17-18."""

    def __init__(self, grid: RadialGrid, chi_on_grid, q_v, sig_v, eps_v, rho_v, q_u, sig_u, eps_u,
                 temperature=298.0, closure="KH", pse_order=1, kappa=1.0):
        self.grid, self.chi = grid, np.asarray(chi_on_grid)                # chi [k][g'][g] at grid.k
        self.beta = 1.0 / (K_BOLTZMANN * temperature)
        self.kT = K_BOLTZMANN * temperature
        self.closure, self.pse_order = closure, pse_order
        self.rho_v = np.asarray(rho_v, float)
        n_v = len(q_v)
        r, k = grid.r, grid.k
        self.w = np.empty((n_v, len(r)))
        self.fr = np.empty((n_v, len(r)))
        self.Fk = np.empty((n_v, len(k)))
        for g in range(n_v):
            qq = q_u * q_v[g]
            lj = lj_pair(r, sig_u, eps_u, sig_v[g], eps_v[g])
            self.w[g] = -self.beta * (lj + COULOMB * qq * np.exp(-kappa * r) / r)
            self.fr[g] = f_long_r(r, qq, self.beta, kappa)
            self.Fk[g] = f_long_k(k, qq, self.beta, kappa)
        self.tau = np.zeros((n_v, len(r)))

    def closure_step(self, tau):
        d = self.w + tau
        g = closure_g(d, self.closure, self.pse_order)
        return d, g, g - 1.0 - tau

    def rism_map(self, tau):
        _, _, c_sr = self.closure_step(tau)
        Csr_k = self.grid.forward(c_sr)
        Ck = Csr_k - self.Fk
        Hk = np.einsum("ak,kab->bk", Ck, self.chi)                         # Eq. 8 / Eq. 13
        return self.grid.inverse(Hk - Csr_k)

    def solve(self, tol=1e-10, max_iter=3000, nvec=10, b=0.5, restart=10.0):
        md = Mdiis(nvec, b, restart)
        npts = float(self.tau.size)
        for it in range(max_iter):
            X = self.tau
            R = self.rism_map(X) - X
            rms = math.sqrt(gram(R, R) / npts)
            if rms < tol:
                return it + 1, rms
            self.tau = md.step(X, R, rms)
        raise RuntimeError("1D solute-solvent RISM not converged")

    def g_r(self):
        return self.closure_step(self.tau)[1]

    def free_energy(self):
        d, g, c_sr = self.closure_step(self.tau)
        h = g - 1.0
        c = c_sr - self.fr
        B = closure_sfe_extra(d, h, self.closure, self.pse_order)
        integrand = -c_sr - 0.5 * h * c + 0.5 * h * h - B     # the f part of -c drops: sum rho q = 0
        r = self.grid.r
        per_site = self.kT * self.rho_v * 4.0 * math.pi * self.grid.dr * np.sum(integrand * r * r, axis=1)
        return float(per_site.sum()), per_site
