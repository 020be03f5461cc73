"""O-3D: the 3D-RISM self-consistent loop, step by step, in plain numpy float64.

TEST INFRASTRUCTURE (see oracle/__init__.py).  Follows PAPER.md:222-254 (numerical procedure),
PAPER.md:300-310 (MDIIS), PAPER.md:264-298 (modified Anderson), PAPER.md:374-379 (residual), PAPER.md:148-158 (free
energy, partial molar volume) in the paper's own variable t = h - c, with
the readings Q1..Q16 listed in DESIGN.md (the paper prints the KH branches, Eq. 40 and Eq. 41 in
garbled form).  Nothing here is blocked, fused or reordered: every array op is one line of a
formula.  Arrays are indexed [gamma][ix][iy][iz].

Units: Angstrom, e, kcal/mol, K.
"""
from __future__ import annotations

import math

import numpy as np

# Physical constants (paper silent; reading Q3).  Typed here independently of the CUDA side.
K_BOLTZMANN = 0.001987204259      # kcal / (mol K)
COULOMB = 332.06371               # kcal A / (mol e^2)


# ----------------------------------------------------------------------------------------------
# Grid  (r-space at integer points, k-space at half-integer points)
# ----------------------------------------------------------------------------------------------
def r_axis(n: int, spacing: float, origin: float) -> np.ndarray:
    """r_i = origin + i * spacing, i = 0..n-1."""
    return origin + spacing * np.arange(n)


def k_axis(n: int, spacing: float) -> np.ndarray:
    """k_j = dk (j + 1/2) for j < n/2, dk (j + 1/2 - n) for j >= n/2 (principal alias); dk = 2 pi / (n spacing).

    The set is +-1/2, +-3/2, ... +-(n-1)/2 times dk: symmetric, no zero."""
    dk = 2.0 * math.pi / (n * spacing)
    j = np.arange(n)
    return dk * np.where(j < n // 2, j + 0.5, j + 0.5 - n)


# ----------------------------------------------------------------------------------------------
# Shifted discrete Fourier pair  (steps 3 and 5 of PAPER.md:242-247; reading Q13)
#   F(k_j) = dV sum_n f(r_n) exp(-i k_j . r_n)        f(r_n) = (1/V) sum_j F(k_j) exp(+i k_j . r_n)
# Separable; per axis  sum_m f_m exp(-i k_j (x0 + m dr)) = exp(-i k_j x0) FFT[f_m exp(-i pi m / n)]_j .
# ----------------------------------------------------------------------------------------------
def shifted_dft_forward(f: np.ndarray, spacing: float, origin) -> np.ndarray:
    """f: real or complex [..., nx, ny, nz] -> complex F on the half-integer k grid (index j per axis)."""
    F = f.astype(np.complex128)
    for ax, x0 in zip((-3, -2, -1), origin):
        n = F.shape[ax]
        shape = [1, 1, 1]
        shape[ax] = n
        m = np.arange(n)
        pre = np.exp(-1j * math.pi * m / n).reshape(shape)
        F = np.fft.fft(F * pre, axis=ax)
        F = F * np.exp(-1j * k_axis(n, spacing) * x0).reshape(shape)
    return F * spacing ** 3


def shifted_dft_inverse(F: np.ndarray, spacing: float, origin) -> np.ndarray:
    """complex F [..., nx, ny, nz] on the half-integer k grid -> complex f(r_n) (imaginary part ~1e-17
    when F has the symmetry of a real field)."""
    f = F.astype(np.complex128)
    for ax, x0 in zip((-3, -2, -1), origin):
        n = f.shape[ax]
        shape = [1, 1, 1]
        shape[ax] = n
        m = np.arange(n)
        f = f * np.exp(+1j * k_axis(n, spacing) * x0).reshape(shape)
        f = np.fft.ifft(f, axis=ax)            # includes 1/n
        f = f * np.exp(+1j * math.pi * m / n).reshape(shape)
    return f / spacing ** 3                    # 1/V = 1/(N dV)


# ----------------------------------------------------------------------------------------------
# Closures  (Eq. 14-16; readings Q1, Q2)
# ----------------------------------------------------------------------------------------------
def closure_g(d: np.ndarray, closure: str, pse_order: int = 1) -> np.ndarray:
    """g(d).  HNC: exp(d).  KH: exp(d) for d <= 0, 1 + d for d > 0.  PSE-n: exp(d) for d <= 0,
    sum_{i=0..n} d^i / i! for d > 0 (n = 1 is KH)."""
    if closure == "HNC":
        return np.exp(d)
    if closure == "KH":
        n = 1
    elif closure == "PSE":
        n = int(pse_order)
    else:
        raise ValueError(closure)
    dneg = np.minimum(d, 0.0)                  # keeps exp() from overflowing on the unused branch
    dpos = np.maximum(d, 0.0)
    series = np.ones_like(d)
    for i in range(n, 0, -1):                  # Horner: 1 + d/1 (1 + d/2 (1 + ... (1 + d/n)))
        series = 1.0 + series * dpos / i
    return np.where(d > 0.0, series, np.exp(dneg))


def closure_sfe_extra(d: np.ndarray, h: np.ndarray, closure: str, pse_order: int = 1) -> np.ndarray:
    """The term B subtracted inside the SFE integrand  -c - hc/2 + h^2/2 - B:
    HNC: 0 (Eq. 17).  KH: h^2/2 Theta(h) (Eq. 18: the h^2 term survives only where h < 0).
    PSE-n: Theta(d) d^(n+1)/(n+1)!  (n = 1: d = h on that branch, so identical to KH)."""
    if closure == "HNC":
        return np.zeros_like(d)
    if closure == "KH":
        return np.where(h > 0.0, 0.5 * h * h, 0.0)
    if closure == "PSE":
        n = int(pse_order)
        dpos = np.maximum(d, 0.0)
        return np.where(d > 0.0, dpos ** (n + 1) / math.factorial(n + 1), 0.0)
    raise ValueError(closure)


# ----------------------------------------------------------------------------------------------
# Potential and long-range functions at arbitrary points (Eq. 22; 226-231 Eq. 29-30)
# ----------------------------------------------------------------------------------------------
def beta_u_at(points, xyz, q_u, sig_u, eps_u, q_v, sig_v, eps_v, beta, r_min):
    """beta * u_gamma(r) of Eq. 22 at `points` [P][3] -> [n_v][P].  All atoms, no images, distance
    clamped at r_min (Q11); Lorentz-Berthelot mixing (Q4)."""
    out = np.zeros((len(q_v), len(points)))
    for a in range(len(q_u)):
        r = np.sqrt(np.sum((points - xyz[a]) ** 2, axis=1))
        r = np.maximum(r, r_min)
        for g in range(len(q_v)):
            s = 0.5 * (sig_u[a] + sig_v[g])
            e = math.sqrt(eps_u[a] * eps_v[g])
            sr6 = (s / r) ** 6
            out[g] += beta * (COULOMB * q_u[a] * q_v[g] / r + 4.0 * e * (sr6 * sr6 - sr6))
    return out


def w_short_at(points, xyz, q_u, sig_u, eps_u, q_v, sig_v, eps_v, beta, r_min, kappa, rcut):
    """w_gamma(r) = -beta sum_{r_a < rcut} [C q_a q_g exp(-kappa r_a)/r_a + LJ]  (Q12): the short-range
    remainder -beta u + f with a sharp cutoff.  Only used when rcut > 0."""
    out = np.zeros((len(q_v), len(points)))
    for a in range(len(q_u)):
        dx = points[:, 0] - xyz[a, 0]
        dy = points[:, 1] - xyz[a, 1]
        dz = points[:, 2] - xyz[a, 2]
        r2 = dx * dx + dy * dy + dz * dz
        inside = r2 < rcut * rcut
        if not inside.any():
            continue
        r = np.maximum(np.sqrt(r2[inside]), r_min)
        for g in range(len(q_v)):
            s = 0.5 * (sig_u[a] + sig_v[g])
            e = math.sqrt(eps_u[a] * eps_v[g])
            sr6 = (s / r) ** 6
            out[g, inside] -= beta * (COULOMB * q_u[a] * q_v[g] * np.exp(-kappa * r) / r
                                      + 4.0 * e * (sr6 * sr6 - sr6))
    return out


def phi_at(points, xyz, q_u, beta, kappa):
    """phi(r) = beta C sum_a q_a (1 - exp(-kappa r_a)) / r_a ;  f_gamma = q_gamma phi  (Eq. 29).
    Finite limit beta C q_a kappa at r_a -> 0.  Never cut off."""
    out = np.zeros(len(points))
    for a in range(len(q_u)):
        r = np.sqrt(np.sum((points - xyz[a]) ** 2, axis=1))
        small = r * kappa < 1e-8
        rs = np.where(small, 1.0, r)
        val = np.where(small, kappa, -np.expm1(-kappa * rs) / rs)
        out += beta * COULOMB * q_u[a] * val
    return out


def phi_tilde_at(kvecs, xyz, q_u, beta, kappa):
    """phi~(k) = 4 pi beta C sum_a q_a exp(-i k.R_a) kappa^2 / (k^2 (k^2 + kappa^2)) ; f~_gamma = q_gamma phi~
    (Eq. 30 with general kappa, Q5).  kvecs [P][3] -> complex [P]."""
    k2 = np.sum(kvecs ** 2, axis=1)
    sfac = np.zeros(len(kvecs), dtype=np.complex128)
    for a in range(len(q_u)):
        sfac += q_u[a] * np.exp(-1j * (kvecs @ xyz[a]))
    return 4.0 * math.pi * beta * COULOMB * sfac * kappa ** 2 / (k2 * (k2 + kappa ** 2))


# ----------------------------------------------------------------------------------------------
# chi(|k|) from the radial table  (reading Q6: 4-point Lagrange cubic)
# ----------------------------------------------------------------------------------------------
def interp_chi(kmag: np.ndarray, k0: float, dk: float, chi: np.ndarray) -> np.ndarray:
    """chi [n_k][n_v][n_v] on k_m = k0 + m dk  ->  [n_v][n_v][...kmag.shape].
    m = floor((|k| - k0)/dk); cubic Lagrange on nodes m-1..m+2, stencil shifted inward at the ends."""
    n_k = chi.shape[0]
    x = (kmag - k0) / dk
    if x.min() < 0.0 or x.max() > n_k - 1:
        raise ValueError("chi table does not cover the 3D |k| range")
    m = np.floor(x).astype(np.int64)
    first = np.clip(m - 1, 0, n_k - 4)         # first node of the 4-point stencil
    u = x - first                              # position in node units, in [0, 3]
    l0 = -(u - 1.0) * (u - 2.0) * (u - 3.0) / 6.0
    l1 = u * (u - 2.0) * (u - 3.0) / 2.0
    l2 = -u * (u - 1.0) * (u - 3.0) / 2.0
    l3 = u * (u - 1.0) * (u - 2.0) / 6.0
    n_v = chi.shape[1]
    out = np.empty((n_v, n_v) + kmag.shape)
    for a in range(n_v):
        for b in range(n_v):
            t = chi[:, a, b]
            out[a, b] = l0 * t[first] + l1 * t[first + 1] + l2 * t[first + 2] + l3 * t[first + 3]
    return out


# ----------------------------------------------------------------------------------------------
# MDIIS small solve  (readings Q7, Q8)
# ----------------------------------------------------------------------------------------------
def mdiis_coefficients(S: np.ndarray) -> np.ndarray:
    """Minimise c^T S c subject to sum c = 1 over m stored residuals: bordered system
    [[S/smax, 1], [1^T, 0]] [c; lambda] = [0; 1], Gaussian elimination with partial pivoting,
    written out (no library call) so that the CUDA side can take the same steps in the same order.
    Degenerate input (smax <= 0 or a zero pivot): c = unit vector on the LAST entry."""
    m = S.shape[0]
    smax = max(S[i, i] for i in range(m))
    fallback = np.zeros(m)
    fallback[m - 1] = 1.0
    if not (smax > 0.0):
        return fallback
    n = m + 1
    A = [[0.0] * (n + 1) for _ in range(n)]
    for i in range(m):
        for j in range(m):
            A[i][j] = float(S[i, j]) / smax
        A[i][m] = 1.0
        A[m][i] = 1.0
    A[m][n] = 1.0                              # right-hand side column
    for col in range(n):
        piv = col
        for r in range(col + 1, n):
            if abs(A[r][col]) > abs(A[piv][col]):
                piv = r
        if A[piv][col] == 0.0:
            return fallback
        A[col], A[piv] = A[piv], A[col]
        for r in range(col + 1, n):
            fac = A[r][col] / A[col][col]
            for c in range(col, n + 1):
                A[r][c] = A[r][c] - fac * A[col][c]
    x = [0.0] * n
    for r in range(n - 1, -1, -1):
        acc = A[r][n]
        for c in range(r + 1, n):
            acc = acc - A[r][c] * x[c]
        x[r] = acc / A[r][r]
    return np.array(x[:m])


def gram(a: np.ndarray, b: np.ndarray) -> float:
    """sum_{n,gamma} a b, accumulated in extended precision (x86 80-bit) so that the rounded result
    does not depend on the summation order ('correctly rounded Gram entries')."""
    return float(np.sum(a.astype(np.longdouble) * b.astype(np.longdouble), dtype=np.longdouble))


def dynamic_damping(rms: float, b_min: float, b_max: float) -> float:
    """b = -0.2 log(R), R the rms residual ('when this parameter was changed dynamically ... the 3D-RISM
    calculation is stable and converges quickly').  The paper gives neither the base of the logarithm nor what happens
    for R >= 1 (b <= 0) or R < 1e-5 (b > 1): read as the decimal logarithm, clamped to [b_min, b_max] (Q18)."""
    return min(b_max, max(b_min, -0.2 * math.log10(rms)))


class Mdiis:
    """History of (X_i, R_i) pairs, circular over M slots, with the restart rule of Q8.
    dynamic_b = (b_min, b_max): the damping parameter of Eq. 40 follows the residual (dynamic_damping) instead of being
    the static b; it multiplies the whole sum of Eq. 40, i.e. the CURRENT b applies to every stored residual."""

    def __init__(self, nvec: int, b: float, restart: float, dynamic_b=None):
        self.M, self.b, self.restart = int(nvec), float(b), float(restart)
        self.dynamic_b = None if dynamic_b is None else (float(dynamic_b[0]), float(dynamic_b[1]))
        self.X, self.R, self.rms = [], [], []      # oldest first
        self.S = np.zeros((0, 0))

    def step(self, X: np.ndarray, R: np.ndarray, rms: float) -> np.ndarray:
        """Store (X, R), return the next input X_new = sum_i c_i (X_i + b R_i)."""
        if self.dynamic_b is not None:
            self.b = dynamic_damping(rms, *self.dynamic_b)
        if len(self.X) == self.M:                  # overwrite the oldest
            self.X.pop(0); self.R.pop(0); self.rms.pop(0)
            self.S = self.S[1:, 1:]
        self.X.append(X); self.R.append(R); self.rms.append(rms)
        m = len(self.X)
        S = np.zeros((m, m))
        S[:m - 1, :m - 1] = self.S
        for i in range(m):
            S[m - 1, i] = S[i, m - 1] = gram(R, self.R[i])
        self.S = S
        if self.restart > 0.0 and rms > self.restart * min(self.rms):
            best = int(np.argmin(self.rms))        # first minimum
            self.X, self.R, self.rms = [self.X[best]], [self.R[best]], [self.rms[best]]
            self.S = self.S[best:best + 1, best:best + 1].copy()
            m = 1
        c = mdiis_coefficients(self.S)
        Xn = np.zeros_like(X)
        for i in range(m):
            Xn = Xn + c[i] * (self.X[i] + self.b * self.R[i])
        return Xn


# ----------------------------------------------------------------------------------------------
# Modified Anderson with two histories  (Eq. 34-39; reading Q17)
# ----------------------------------------------------------------------------------------------
def gram_weighted(a: np.ndarray, b: np.ndarray, w: np.ndarray) -> float:
    """(a, b) = sum_gamma w_gamma sum_r a b  (Eq. 38; a, b are [gamma][...]), extended precision like gram()."""
    tot = np.longdouble(0.0)
    for g in range(a.shape[0]):
        tot += np.longdouble(w[g]) * np.sum(a[g].astype(np.longdouble) * b[g].astype(np.longdouble), dtype=np.longdouble)
    return float(tot)


def anderson_theta(S: np.ndarray) -> np.ndarray:
    """theta_1, theta_2 of Eq. 36, read as the normal equations of min |R0 - sum_j theta_j dR_j|^2 with
    dR_j = R^(n-1) - R^(n-j-1):   sum_j (dR_i, dR_j) theta_j = (R0, dR_i),  i = 1, 2.
    S is the 3x3 weighted Gram matrix of (R0 = newest, R1, R2).  2x2 solve by Cramer's rule on the system scaled by
    its largest diagonal entry; a singular system gives theta = 0 (plain mixing)."""
    A = [[0.0, 0.0], [0.0, 0.0]]
    rhs = [0.0, 0.0]
    for i in (1, 2):
        rhs[i - 1] = S[0, 0] - S[0, i]
        for j in (1, 2):
            A[i - 1][j - 1] = S[0, 0] - S[0, i] - S[0, j] + S[i, j]
    amax = max(A[0][0], A[1][1])
    if not (amax > 0.0):
        return np.zeros(2)
    a, b_, c, d = A[0][0] / amax, A[0][1] / amax, A[1][0] / amax, A[1][1] / amax
    r0, r1 = rhs[0] / amax, rhs[1] / amax
    det = a * d - b_ * c
    if det == 0.0:
        return np.zeros(2)
    return np.array([(r0 * d - b_ * r1) / det, (a * r1 - r0 * c) / det])


class ModifiedAnderson:
    """Two histories.  With X_k, R_k the inputs and residuals of the newest (k = 0) and the two previous (k = 1, 2)
    evaluations, Y_k = X_k + R_k:
        u = X_0 + sum_i (theta_i + s_i)(X_i - X_0)              Eq. 34
        v = Y_0 + sum_i (theta_i + s_i)(Y_i - Y_0)              Eq. 35
        X_new = u + b (v - u)                                   Eq. 39
    Picard steps X + b R until two histories exist."""

    def __init__(self, b: float, s, weights):
        self.b, self.s, self.w = float(b), (float(s[0]), float(s[1])), np.asarray(weights, float)
        self.X, self.R = [], []                    # newest first

    def step(self, X: np.ndarray, R: np.ndarray, rms: float) -> np.ndarray:
        self.X.insert(0, X)
        self.R.insert(0, R)
        del self.X[3:], self.R[3:]
        if len(self.X) < 3:
            return X + self.b * R
        S = np.zeros((3, 3))
        for i in range(3):
            for j in range(i, 3):
                S[i, j] = S[j, i] = gram_weighted(self.R[i], self.R[j], self.w)
        th = anderson_theta(S)
        u = self.X[0].copy()
        v = self.X[0] + self.R[0]
        for i in (1, 2):
            a = th[i - 1] + self.s[i - 1]
            u = u + a * (self.X[i] - self.X[0])
            v = v + a * ((self.X[i] + self.R[i]) - (self.X[0] + self.R[0]))
        return u + self.b * (v - u)


# ----------------------------------------------------------------------------------------------
# The solver
# ----------------------------------------------------------------------------------------------
class Rism3dOracle:
    """Same five calls as the C ABI (include/rism3d.h): init / set_solvent_chi / set_solute /
    iterate / free_energy, plus get_field."""

    def __init__(self, n, spacing, n_sites, closure="KH", pse_order=1, temperature=298.0,
                 mdiis_nvec=5, mdiis_b=0.5, mdiis_restart=10.0, kappa=1.0, r_min=1e-3, origin=None,
                 accelerator="MDIIS", anderson_s=(0.2, 0.0), mdiis_dynamic_b=None):
        self.mdiis_dynamic_b = mdiis_dynamic_b
        self.n = (n, n, n) if np.isscalar(n) else tuple(n)
        self.dr = float(spacing)
        self.origin = tuple(-(m // 2) * self.dr for m in self.n) if origin is None else tuple(origin)
        self.n_v = int(n_sites)
        self.closure, self.pse_order = closure, int(pse_order)
        self.beta = 1.0 / (K_BOLTZMANN * temperature)
        self.kT = K_BOLTZMANN * temperature
        self.M, self.b, self.restart = mdiis_nvec, mdiis_b, mdiis_restart
        self.kappa, self.r_min = float(kappa), float(r_min)
        self.accelerator, self.anderson_s = accelerator, tuple(anderson_s)
        ax = [r_axis(m, self.dr, o) for m, o in zip(self.n, self.origin)]
        gx, gy, gz = np.meshgrid(*ax, indexing="ij")
        self.points = np.stack([gx.ravel(), gy.ravel(), gz.ravel()], axis=1)
        kx, ky, kz = np.meshgrid(*[k_axis(m, self.dr) for m in self.n], indexing="ij")
        self.kvecs = np.stack([kx.ravel(), ky.ravel(), kz.ravel()], axis=1)
        self.kmag = np.sqrt(kx * kx + ky * ky + kz * kz)
        self.chi_grid = None
        self.t = None

    # -- solvent ---------------------------------------------------------------------------
    def set_solvent_chi(self, q, sigma, eps, rho, k0, dk, chi):
        self.q_v, self.sig_v, self.eps_v, self.rho_v = (np.asarray(a, float) for a in (q, sigma, eps, rho))
        if abs(np.dot(self.rho_v, self.q_v)) > 1e-12:
            raise ValueError("solvent not neutral: sum rho_gamma q_gamma != 0")
        self.chi_grid = interp_chi(self.kmag, k0, dk, np.asarray(chi, float))   # [g'][g][kx][ky][kz]

    # -- solute: steps 1-3 of SURVEY 8(c) --------------------------------------------------
    def set_solute(self, xyz, q, sigma, eps, rcut=0.0):
        xyz, q, sigma, eps = (np.asarray(a, float) for a in (xyz, q, sigma, eps))
        shp = (self.n_v,) + self.n
        phi = phi_at(self.points, xyz, q, self.beta, self.kappa)
        self.phi = phi.reshape(self.n)
        self.f = self.q_v[:, None, None, None] * self.phi[None]                        # Eq. 29
        self.phi_tilde = phi_tilde_at(self.kvecs, xyz, q, self.beta, self.kappa).reshape(self.n)
        self.f_tilde = self.q_v[:, None, None, None] * self.phi_tilde[None]            # Eq. 30
        if rcut > 0.0:
            w = w_short_at(self.points, xyz, q, sigma, eps, self.q_v, self.sig_v, self.eps_v,
                           self.beta, self.r_min, self.kappa, rcut).reshape(shp)
            self.minus_beta_u = w - self.f                                             # Q12
        else:
            self.minus_beta_u = -beta_u_at(self.points, xyz, q, sigma, eps, self.q_v, self.sig_v,
                                           self.eps_v, self.beta, self.r_min).reshape(shp)  # Eq. 22
        self._solute = (xyz, q, sigma, eps)
        self.t = self.f.copy()                                                         # step 1
        if self.accelerator == "ANDERSON":          # weight 1/rho_gamma; b is the mixing parameter
            self.mdiis = ModifiedAnderson(self.b, self.anderson_s, 1.0 / self.rho_v)
        else:
            self.mdiis = Mdiis(self.M, self.b, self.restart, self.mdiis_dynamic_b)
        self.rms_history = []

    # -- one pass of steps 2-5 ---------------------------------------------------------------
    def closure_step(self, t):
        """step 2: g from the closure, c_sr by Eq. 31."""
        d = self.minus_beta_u + t                                                      # Eq. 16 with t = h - c
        g = closure_g(d, self.closure, self.pse_order)
        c_sr = g - 1.0 - t + self.f                                                    # Eq. 31
        return d, g, c_sr

    def rism_map(self, t):
        """steps 2-5: t -> t' (Eq. 33).  Returns (t', g, c_sr)."""
        d, g, c_sr = self.closure_step(t)
        c_sr_k = shifted_dft_forward(c_sr, self.dr, self.origin)                       # step 3
        c_k = c_sr_k - self.f_tilde                                                    # Eq. 32
        h_k = np.zeros_like(c_k)
        for gam in range(self.n_v):                                                    # Eq. 13 (step 4)
            for gp in range(self.n_v):
                h_k[gam] += c_k[gp] * self.chi_grid[gp, gam]
        h = shifted_dft_inverse(h_k, self.dr, self.origin).real                        # step 5
        t_new = t + h + 1.0 - g                                                        # Eq. 33
        return t_new, g, c_sr

    def iterate(self, max_iter, tol=0.0):
        """steps 2-7.  tol <= 0: exactly max_iter passes.  Returns (n_done, last rms)."""
        n_done, rms = 0, float("nan")
        npts = float(np.prod(self.n) * self.n_v)
        for _ in range(max_iter):
            X = self.t
            Y, _, _ = self.rism_map(X)
            R = Y - X
            rms = math.sqrt(gram(R, R) / npts)                                         # Q9
            n_done += 1
            self.rms_history.append(rms)
            if not math.isfinite(rms):
                raise FloatingPointError("3D-RISM diverged")
            if tol > 0.0 and rms < tol:
                break                                                                  # step 7; X unchanged
            self.t = self.mdiis.step(X, R, rms)                                        # step 6
        return n_done, rms

    # -- results -------------------------------------------------------------------------------
    def get_field(self, which):
        d, g, c_sr = self.closure_step(self.t)
        return {"G": g, "H": g - 1.0, "C_SR": c_sr, "T": self.t, "TAU": self.t - self.f,
                "W": self.minus_beta_u + self.f, "C": c_sr - self.f, "D": d}[which]

    def free_energy(self):
        """Eq. 18 (KH) / Eq. 17 (HNC) / PSE-n, plain grid sum (Q10):
        dmu = kT dV sum_n sum_gamma rho_gamma [ -c_sr - h c / 2 + h^2 / 2 - B ],  c = c_sr - f."""
        d, g, c_sr = self.closure_step(self.t)
        h = g - 1.0
        c = c_sr - self.f
        B = closure_sfe_extra(d, h, self.closure, self.pse_order)
        integrand = -c_sr - 0.5 * h * c + 0.5 * h * h - B
        per_site = np.array([self.kT * self.dr ** 3 * self.rho_v[gam] *
                             float(np.sum(integrand[gam], dtype=np.longdouble))
                             for gam in range(self.n_v)])
        return float(per_site.sum()), per_site

    def pmv(self, chi_t):
        """Partial molar volume, Eq. 19:  V = kT chi_T (1 - sum_gamma rho_gamma int c_gamma dr), plain
        grid sum.  The long-range part -f_gamma of c drops out of the density-weighted sum (sum rho q = 0), as in the
        free energy (Q10).  Returns (V in A^3, per-site dV sum_r c_sr)."""
        _, _, c_sr = self.closure_step(self.t)
        c_int = np.array([self.dr ** 3 * float(np.sum(c_sr[gam], dtype=np.longdouble)) for gam in range(self.n_v)])
        return float(self.kT * chi_t * (1.0 - np.dot(self.rho_v, c_int))), c_int

    def pressure_correction(self, chi_t, pressure):
        """PC term of the solvation free energy, Eq. 21:  dmu_PC = -P V, with the partial molar volume of
        Eq. 19 and the bulk pressure of Eq. 20 (both bulk quantities come from the solvent's own 1D solve).
        Returns (dmu_PC in kcal/mol, V in A^3)."""
        v, _ = self.pmv(chi_t)
        return -pressure * v, v

    def solvation_gradient(self):
        """d(dmu)/dR_alpha = sum_gamma rho_gamma dV sum_r g_gamma(r) du_gamma(r)/dR_alpha  (the
        equation after Eq. 23; 'common for both HNC and KH'), kcal/(mol A), all pairs, u of Eq. 22 with the distance
        clamp of Q11 (inside the clamp the potential is flat: no contribution).  -> [n_atoms][3].
        d/dR_alpha [1/r] = (r - R_alpha)/r^3 ;  d/dR_alpha [(s/r)^12 - (s/r)^6] = (12 s^12/r^14 - 6 s^6/r^8)(r - R_alpha)."""
        _, g, _ = self.closure_step(self.t)
        xyz, q_u, sig_u, eps_u = self._solute
        out = np.zeros((len(q_u), 3))
        gw = [self.rho_v[gam] * self.dr ** 3 * g[gam].ravel() for gam in range(self.n_v)]
        for a in range(len(q_u)):
            d = self.points - xyz[a]
            r2 = np.sum(d * d, axis=1)
            inside = r2 < self.r_min ** 2
            r2 = np.where(inside, 1.0, r2)
            coef = np.zeros(len(r2))
            for gam in range(self.n_v):
                s = 0.5 * (sig_u[a] + self.sig_v[gam])
                e = math.sqrt(eps_u[a] * self.eps_v[gam])
                s6 = (s * s / r2) ** 3
                du = COULOMB * q_u[a] * self.q_v[gam] / (r2 * np.sqrt(r2)) + 4.0 * e * (12.0 * s6 * s6 - 6.0 * s6) / r2
                coef += gw[gam] * du
            coef = np.where(inside, 0.0, coef)
            out[a] = [float(np.sum(coef * d[:, k], dtype=np.longdouble)) for k in range(3)]
        return out

