// setup_kernels.cu -- everything outside the iteration loop:
//   potential_kernel   : w_g(r) = -beta u_g(r) + f_g(r) and phi(r)       (Eq. 22 + Eq. 29)
//   phase / phi_tilde  : phi~(k) exp(+i k.r0)/dV on the stored half of the half-integer k grid (Eq. 30)
//   chi_shell_kernel   : chi_{g'g}(|k|) for every distinct |k| of the grid, by 4-point Lagrange interpolation of
//                        the radial table (Q6)
//   free_energy_kernel : Eq. 17 / 18 / PSE-n grid sum (Q2, Q10)
//   get_field_kernel   : g, h, c_sr, t, tau, w, phi of one site
#include "rism3d_internal.h"

namespace r3d {

// ------------------------------------------------------------------------------------------------
// Grid potential, all pairs (optionally with the sharp cutoff of Q12 on the short-range remainder).
// One thread per grid point, atoms staged through shared memory in chunks.
// atoms: [n_atoms] (x, y, z, beta*C*q_a);  pair: [n_atoms][nv] (beta C q_a q_g, sigma_ag^2, 4 beta eps_ag)
// ------------------------------------------------------------------------------------------------
constexpr int ATOM_CHUNK = 64;

template <int NV>
__global__ void __launch_bounds__(128)
    potential_kernel(double* __restrict__ w, double* __restrict__ phi, const double4* __restrict__ atoms,
                     const double* __restrict__ pair, int n_atoms, int n, double h, double ox, double oy, double oz,
                     double kappa, double r_min, double rcut2, size_t npts) {
  __shared__ double4 s_atom[ATOM_CHUNK];
  __shared__ double s_pair[ATOM_CHUNK * NV * 3];
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;   // npts is a multiple of blockDim
  const int iz = (int)(idx % n), iy = (int)((idx / n) % n), ix = (int)(idx / ((size_t)n * n));
  // r_n = origin + spacing * index, each operation rounded separately (the pair set of a cutoff must not depend
  // on contraction)
  const double x = __dadd_rn(ox, __dmul_rn(h, (double)ix));
  const double y = __dadd_rn(oy, __dmul_rn(h, (double)iy));
  const double z = __dadd_rn(oz, __dmul_rn(h, (double)iz));
  double acc[NV];
#pragma unroll
  for (int g = 0; g < NV; ++g) acc[g] = 0.0;
  double ph = 0.0;
  const bool cut = rcut2 > 0.0;
  const double rmin2 = r_min * r_min, far2 = 1600.0 / (kappa * kappa);
  for (int a0 = 0; a0 < n_atoms; a0 += ATOM_CHUNK) {
    const int na = min(ATOM_CHUNK, n_atoms - a0);
    __syncthreads();
    for (int i = threadIdx.x; i < na; i += blockDim.x) s_atom[i] = atoms[a0 + i];
    for (int i = threadIdx.x; i < na * NV * 3; i += blockDim.x) s_pair[i] = pair[(size_t)a0 * NV * 3 + i];
    __syncthreads();
    for (int a = 0; a < na; ++a) {
      const double4 at = s_atom[a];
      const double dx = x - at.x, dy = y - at.y, dz = z - at.z;
      const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
      // The common case first.  1/r: float rsqrt seed + two Newton steps in double (~2 ulp; r^2 is far inside the
      // float range).  Beyond kappa r = 40, exp(-kappa r) < 5e-18 vanishes against 1 in double precision: (1 -
      // exp(-kappa r))/r is 1/r to the last bit and the short-range Coulomb term is 0, so far pairs (most of them
      // on the large grids) need no exp at all.
      if (r2 >= rmin2) {
        double rinv = (double)rsqrtf((float)r2);
        rinv = rinv * fma(-0.5 * r2, rinv * rinv, 1.5);
        rinv = rinv * fma(-0.5 * r2, rinv * rinv, 1.5);
        if (r2 > far2) {
          ph = fma(at.w, rinv, ph);
          if (!cut) {                                         // all-pairs mode: LJ reaches further than exp(-kappa r)
            const double inv2 = rinv * rinv;
            const double* pp = s_pair + a * NV * 3;
#pragma unroll
            for (int g = 0; g < NV; ++g) {
              const double s2 = pp[g * 3 + 1] * inv2;
              const double s6 = s2 * s2 * s2;
              acc[g] -= pp[g * 3 + 2] * (s6 * s6 - s6);
            }
          }
        } else {
          const double kr = kappa * (r2 * rinv);
          // 1 - exp(-kappa r): expm1 where the subtraction would cancel, exp elsewhere
          const double ex = (kr < 0.5) ? 1.0 + expm1(-kr) : exp(-kr);
          const double om = (kr < 0.5) ? -expm1(-kr) : 1.0 - ex;
          ph = fma(at.w, om * rinv, ph);
          if (!cut || r2 < rcut2) {
            const double sc = ex * rinv;                      // exp(-kappa r)/r = 1/r - (1 - exp(-kappa r))/r
            const double inv2 = rinv * rinv;
            const double* pp = s_pair + a * NV * 3;
#pragma unroll
            for (int g = 0; g < NV; ++g) {
              const double s2 = pp[g * 3 + 1] * inv2;
              const double s6 = s2 * s2 * s2;
              acc[g] -= pp[g * 3 + 0] * sc + pp[g * 3 + 2] * (s6 * s6 - s6);
            }
          }
        }
      } else {
        // grid point (almost) on an atom: distance clamped at r_min (Q11), phi at its finite limit
        const double rt = sqrt(r2);
        const double kr = kappa * rt;
        const double em = expm1(-kr);
        const double lr = (kr < 1e-8) ? kappa : -em / rt;     // (1 - exp(-kappa r)) / r and its limit
        ph += at.w * lr;
        if (!cut || r2 < rcut2) {
          const double rc = fmax(rt, r_min);
          const double sc = (rt >= r_min) ? (1.0 + em) / rt : (cut ? exp(-kappa * rc) / rc : 1.0 / rc - lr);
          const double inv2 = 1.0 / (rc * rc);
          const double* pp = s_pair + a * NV * 3;
#pragma unroll
          for (int g = 0; g < NV; ++g) {
            const double s2 = pp[g * 3 + 1] * inv2;
            const double s6 = s2 * s2 * s2;
            acc[g] -= pp[g * 3 + 0] * sc + pp[g * 3 + 2] * (s6 * s6 - s6);
          }
        }
      }
    }
  }
  phi[idx] = ph;
#pragma unroll
  for (int g = 0; g < NV; ++g) w[(size_t)g * npts + idx] = acc[g];
}

int launch_potential(const Grid& g, const Buffers& b, const SolverParams& sp, int n_atoms, const double* d_atoms,
                     const double* d_pair, double rcut, cudaStream_t s) {
  const unsigned blocks = (unsigned)(g.npts / 128);
  const double rcut2 = rcut > 0.0 ? rcut * rcut : 0.0;
  const double4* at = reinterpret_cast<const double4*>(d_atoms);
#define POT(NV)                                                                                                   \
  potential_kernel<NV><<<blocks, 128, 0, s>>>(b.w, b.phi, at, d_pair, n_atoms, g.n, g.h, g.origin[0], g.origin[1], \
                                              g.origin[2], sp.kappa, sp.r_min, rcut2, g.npts)
  switch (g.nv) {
    case 1: POT(1); break;
    case 2: POT(2); break;
    case 4: POT(4); break;
    case 8: POT(8); break;
    default: return 0;
  }
#undef POT
  return 1;
}

// ------------------------------------------------------------------------------------------------
// phi~(k): separable phase tables E_axis[a][j] = exp(-i k_j (R_a,axis - r0,axis)), then
//   phik[jx][jy][p] = (4 pi beta C / dV) kappa^2 / (k^2 (k^2 + kappa^2)) sum_a q_a Ex[a][jx] Ey[a][jy] Ez[a][2p]
// d_phase: [3][n_atoms][n] complex (z table holds only the even j at index p, n/2 entries used)
// ------------------------------------------------------------------------------------------------
__global__ void phase_kernel(double2* __restrict__ phase, const double4* __restrict__ atoms, int n_atoms, int n,
                             double h, double ox, double oy, double oz) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t total = (size_t)3 * n_atoms * n;
  if (idx >= total) return;
  const int j = (int)(idx % n);
  const int a = (int)((idx / n) % n_atoms);
  const int axis = (int)(idx / ((size_t)n * n_atoms));
  const double4 at = atoms[a];
  const double d = axis == 0 ? at.x - ox : (axis == 1 ? at.y - oy : at.z - oz);
  int jj = j;
  if (axis == 2) { if (j >= n / 2) { phase[idx] = make_double2(0.0, 0.0); return; } jj = 2 * j; }
  const double f = (jj < n / 2) ? (jj + 0.5) : (jj + 0.5 - n);          // k = dk * f, dk = 2 pi / (n h)
  double sn, cs;
  sincospi(2.0 * f * (d / (n * h)), &sn, &cs);
  phase[idx] = make_double2(cs, -sn);
}

constexpr int PT_JY = 8;      // jy values per thread
constexpr int PT_AC = 32;     // atoms per shared-memory chunk

__global__ void __launch_bounds__(64)
    phi_tilde_kernel(double2* __restrict__ phik, const double2* __restrict__ phase, const double* __restrict__ qa,
                     int n_atoms, int n, double h, double kappa, double pref) {
  __shared__ double2 s_a[PT_AC][PT_JY];
  const int nz = n / 2;
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  const int jy0 = blockIdx.y * PT_JY;
  const int jx = blockIdx.z;
  const double2* Ex = phase;
  const double2* Ey = phase + (size_t)n_atoms * n;
  const double2* Ez = phase + (size_t)2 * n_atoms * n;
  double2 acc[PT_JY];
#pragma unroll
  for (int i = 0; i < PT_JY; ++i) acc[i] = make_double2(0.0, 0.0);
  for (int a0 = 0; a0 < n_atoms; a0 += PT_AC) {
    const int na = min(PT_AC, n_atoms - a0);
    __syncthreads();
    for (int i = threadIdx.x; i < na * PT_JY; i += blockDim.x) {
      const int a = a0 + i / PT_JY, jy = jy0 + i % PT_JY;
      const double2 ex = Ex[(size_t)a * n + jx], ey = Ey[(size_t)a * n + jy];
      const double q = qa[a];
      s_a[i / PT_JY][i % PT_JY] = make_double2(q * (ex.x * ey.x - ex.y * ey.y), q * (ex.x * ey.y + ex.y * ey.x));
    }
    __syncthreads();
    if (p < nz) {
      for (int a = 0; a < na; ++a) {
        const double2 ez = Ez[(size_t)(a0 + a) * n + p];
#pragma unroll
        for (int i = 0; i < PT_JY; ++i) {
          const double2 v = s_a[a][i];
          acc[i].x += v.x * ez.x - v.y * ez.y;
          acc[i].y += v.x * ez.y + v.y * ez.x;
        }
      }
    }
  }
  if (p >= nz) return;
  const double dk = 2.0 * 3.14159265358979323846 / (n * h);
  auto kof = [&](int j) { return dk * ((j < nz) ? (j + 0.5) : (j + 0.5 - n)); };
  const double kx = kof(jx), kz = kof(2 * p);
#pragma unroll
  for (int i = 0; i < PT_JY; ++i) {
    const double ky = kof(jy0 + i);
    const double k2 = kx * kx + ky * ky + kz * kz;
    const double f = pref * kappa * kappa / (k2 * (k2 + kappa * kappa));
    phik[((size_t)jx * n + (jy0 + i)) * nz + p] = make_double2(f * acc[i].x, f * acc[i].y);
  }
}

int launch_phi_tilde(const Grid& g, const Buffers& b, const SolverParams& sp, int n_atoms, const double* d_atoms,
                     double2* d_phase, cudaStream_t s) {
  const size_t total = (size_t)3 * n_atoms * g.n;
  const double4* at = reinterpret_cast<const double4*>(d_atoms);
  int launched = 1;
  if (total > 0) {                                       // an empty solute has no phase table (phi~ = 0)
    phase_kernel<<<(unsigned)((total + 255) / 256), 256, 0, s>>>(d_phase, at, n_atoms, g.n, g.h, g.origin[0],
                                                                g.origin[1], g.origin[2]);
    launched = 2;
  }
  // charges q_a live in a separate array right after the atom records (set up by the API layer)
  const double* qa = d_atoms + (size_t)4 * n_atoms;
  const int nz = g.n / 2;
  const int bx = nz < 64 ? nz : 64;
  dim3 grid((nz + bx - 1) / bx, g.n / PT_JY, g.n);
  const double pref = 4.0 * 3.14159265358979323846 * sp.beta * COULOMB / (g.h * g.h * g.h);
  phi_tilde_kernel<<<grid, bx, 0, s>>>(b.phik, d_phase, qa, n_atoms, g.n, g.h, sp.kappa, pref);
  return launched;
}

// ------------------------------------------------------------------------------------------------
// chi per |k| shell.  table: [n_k][nv][nv] (chi[m][g'][g]);  out: [nshell][g][g']
// ------------------------------------------------------------------------------------------------
__global__ void chi_shell_kernel(double* __restrict__ out, const double* __restrict__ table, int n_k, double k0,
                                 double dkt, int nv, double dk_grid, int nshell) {
  const int sidx = blockIdx.x * blockDim.x + threadIdx.x;
  if (sidx >= nshell) return;
  const double kmag = dk_grid * sqrt(2.0 * sidx + 0.75);
  const double xk = (kmag - k0) / dkt;
  int m = (int)floor(xk);
  int first = m - 1;
  if (first < 0) first = 0;
  if (first > n_k - 4) first = n_k - 4;
  const double u = xk - first;
  const double l0 = -(u - 1.0) * (u - 2.0) * (u - 3.0) / 6.0;
  const double l1 = u * (u - 2.0) * (u - 3.0) / 2.0;
  const double l2 = -u * (u - 1.0) * (u - 3.0) / 2.0;
  const double l3 = u * (u - 1.0) * (u - 2.0) / 6.0;
  const size_t st = (size_t)nv * nv;
  for (int gp = 0; gp < nv; ++gp)
    for (int g = 0; g < nv; ++g) {
      const double* t = table + (size_t)first * st + gp * nv + g;
      out[(size_t)sidx * st + g * nv + gp] = l0 * t[0] + l1 * t[st] + l2 * t[2 * st] + l3 * t[3 * st];
    }
}

int launch_chi_shell(const Grid& g, const Buffers& b, const double* d_table, int n_k, double k0, double dk,
                     cudaStream_t s) {
  const int hn = g.n / 2;
  const int nshell = 3 * (hn - 1) * hn / 2 + 1;
  const double dk_grid = 2.0 * 3.14159265358979323846 / (g.n * g.h);
  chi_shell_kernel<<<(nshell + 127) / 128, 128, 0, s>>>(b.chi_shell, d_table, n_k, k0, dk, g.nv, dk_grid, nshell);
  return 1;
}

// ------------------------------------------------------------------------------------------------
// Solvation free energy:  dmu_g = kT dV rho_g sum_n [ -c_sr - h c / 2 + h^2 / 2 - B ],  c = c_sr - q_g phi
//   B = h^2/2 Theta(h) (KH), Theta(d) d^(n+1)/(n+1)! (PSE-n), 0 (HNC)
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
    free_energy_kernel(double* __restrict__ part, const double* __restrict__ tau, const double* __restrict__ w,
                       const double* __restrict__ phi, const double* __restrict__ qv,
                       const DevState* __restrict__ st, int nv, size_t npts, size_t field, int closure, int order) {
  __shared__ double s_red[8][4];
  double inv_fact = 1.0;
  for (int i = 2; i <= order + 1; ++i) inv_fact /= (double)i;
  for (int g = 0; g < nv; ++g) {
    double hi = 0.0, lo = 0.0, chi_ = 0.0, clo = 0.0;    // integrand of Eq. 17/18; c_sr alone (for Eq. 19)
    const double q = qv[g];
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < npts; i += (size_t)gridDim.x * blockDim.x) {
      const double t = tau[(size_t)g * npts + i];
      const double d = w[(size_t)g * npts + i] + t;
      const double gg = closure_g(d, closure, order);
      const double hh = gg - 1.0;
      const double csr = gg - 1.0 - t;
      const double c = csr - q * phi[i];
      double B = 0.0;
      if (closure == RISM3D_KH) B = hh > 0.0 ? 0.5 * hh * hh : 0.0;
      else if (closure == RISM3D_PSE) B = d > 0.0 ? pow(d, order + 1) * inv_fact : 0.0;
      const double v = -csr - 0.5 * hh * c + 0.5 * hh * hh - B;
      dd_add(hi, lo, v, 0.0);
      dd_add(chi_, clo, csr, 0.0);
    }
    for (int o = 16; o > 0; o >>= 1) {
      const double h2 = __shfl_down_sync(0xffffffffu, hi, o), l2 = __shfl_down_sync(0xffffffffu, lo, o);
      dd_add(hi, lo, h2, l2);
      const double h3 = __shfl_down_sync(0xffffffffu, chi_, o), l3 = __shfl_down_sync(0xffffffffu, clo, o);
      dd_add(chi_, clo, h3, l3);
    }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) { s_red[wid][0] = hi; s_red[wid][1] = lo; s_red[wid][2] = chi_; s_red[wid][3] = clo; }
    __syncthreads();
    if (threadIdx.x == 0) {
      hi = 0.0; lo = 0.0; chi_ = 0.0; clo = 0.0;
      for (int k = 0; k < 8; ++k) { dd_add(hi, lo, s_red[k][0], s_red[k][1]); dd_add(chi_, clo, s_red[k][2], s_red[k][3]); }
      part[((size_t)blockIdx.x * MAX_NV + g) * 2 + 0] = hi;
      part[((size_t)blockIdx.x * MAX_NV + g) * 2 + 1] = lo;
      part[((size_t)(gridDim.x + blockIdx.x) * MAX_NV + g) * 2 + 0] = chi_;
      part[((size_t)(gridDim.x + blockIdx.x) * MAX_NV + g) * 2 + 1] = clo;
    }
  }
}

__global__ void free_energy_final_kernel(double* __restrict__ out, const double* __restrict__ part, int nblocks,
                                         const double* __restrict__ rhov, int nv, double scale, double dv) {
  const int g = threadIdx.x;
  if (g >= nv) return;
  double hi = 0.0, lo = 0.0;
  for (int b = 0; b < nblocks; ++b) dd_add(hi, lo, part[((size_t)b * MAX_NV + g) * 2], part[((size_t)b * MAX_NV + g) * 2 + 1]);
  out[g] = scale * rhov[g] * (hi + lo);
  // second set: dV sum_r c_sr,g(r)  (A^3), not density weighted
  hi = 0.0; lo = 0.0;
  for (int b = 0; b < nblocks; ++b)
    dd_add(hi, lo, part[((size_t)(nblocks + b) * MAX_NV + g) * 2], part[((size_t)(nblocks + b) * MAX_NV + g) * 2 + 1]);
  out[MAX_NV + g] = dv * (hi + lo);
}

int launch_free_energy(const Grid& g, const Buffers& b, const SolverParams& sp, double* d_out, cudaStream_t s) {
  const int blocks = FE_BLOCKS;
  free_energy_kernel<<<blocks, 256, 0, s>>>(b.fe_part, b.tau, b.w, b.phi, b.qv, b.state, g.nv, g.npts, g.field,
                                            sp.closure, sp.pse_order);
  free_energy_final_kernel<<<1, 32, 0, s>>>(d_out, b.fe_part, blocks, b.rhov, g.nv, sp.kT * g.h * g.h * g.h,
                                            g.h * g.h * g.h);
  return 2;
}

// ------------------------------------------------------------------------------------------------
__global__ void get_field_kernel(double* __restrict__ dst, const double* __restrict__ tau_all, const double* __restrict__ w,
                                 const double* __restrict__ phi, const double* __restrict__ qv,
                                 const DevState* __restrict__ st, int which, int site, size_t npts, size_t field,
                                 int closure, int order) {
  const double* tau = tau_all + (size_t)site * npts;
  const double* ws = w + (size_t)site * npts;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < npts; i += (size_t)gridDim.x * blockDim.x) {
    double v;
    if (which == RISM3D_FIELD_PHI) v = phi[i];
    else if (which == RISM3D_FIELD_W) v = ws[i];
    else if (which == RISM3D_FIELD_TAU) v = tau[i];
    else if (which == RISM3D_FIELD_T) v = tau[i] + qv[site] * phi[i];
    else {
      const double t = tau[i];
      const double gg = closure_g(ws[i] + t, closure, order);
      v = which == RISM3D_FIELD_G ? gg : (which == RISM3D_FIELD_H ? gg - 1.0 : gg - 1.0 - t);
    }
    dst[i] = v;
  }
}

int launch_get_field(const Grid& g, const Buffers& b, const SolverParams& sp, int which, int site, double* d_dst,
                     cudaStream_t s) {
  size_t blocks = (g.npts + 255) / 256;
  if (blocks > 148 * 16) blocks = 148 * 16;
  get_field_kernel<<<(unsigned)blocks, 256, 0, s>>>(d_dst, b.tau, b.w, b.phi, b.qv, b.state, which, site, g.npts,
                                                    g.field, sp.closure, sp.pse_order);
  return 1;
}

// ------------------------------------------------------------------------------------------------
// Solvent-induced gradient on the solute atoms (the equation after Eq. 23):
//   d(dmu)/dR_a = sum_g rho_g dV sum_r g_g(r) du_g(r)/dR_a,   u of Eq. 22, all pairs, distance clamp of Q11
//   du_g/dR_a = [C q_a q_g / r^3 + 4 eps_ag (12 s^12/r^14 - 6 s^6/r^8)] (r - R_a)
// Grid: (point chunks, chunks of GRAD_ATOMS atoms).  A thread walks its points, reads rho_g dV g_g(r) (formed once by
// gradient_weights_kernel) and accumulates the 3 components for the block's atoms in registers; the block sum (double-double, fixed
// order) goes to partial[chunk][atom][3]; gradient_final_kernel adds the chunks in order.  pair carries beta
// (beta C q_a q_g, sigma_ag^2, 4 beta eps_ag), so the final sum is multiplied by kT.
// ------------------------------------------------------------------------------------------------
constexpr int GRAD_ATOMS = 8;
constexpr int GRAD_THREADS = 256;

// gw_g(r) = rho_g dV g_g(r), g = closure(w + tau): formed once per call, read by every atom chunk
__global__ void gradient_weights_kernel(double* __restrict__ gw, const double* __restrict__ tau,
                                        const double* __restrict__ w, const double* __restrict__ rhov, size_t npts,
                                        int nv, double dv, int closure, int order) {
  for (int g = 0; g < nv; ++g) {
    const double f = rhov[g] * dv;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < npts; i += (size_t)gridDim.x * blockDim.x)
      gw[(size_t)g * npts + i] = f * closure_g(w[(size_t)g * npts + i] + tau[(size_t)g * npts + i], closure, order);
  }
}

template <int NV>
__global__ void __launch_bounds__(GRAD_THREADS)
    gradient_kernel(double* __restrict__ partial, const double* __restrict__ gwf, const double4* __restrict__ atoms,
                    const double* __restrict__ pair, int n_atoms, int n, double h, double ox, double oy, double oz,
                    double r_min, size_t npts, size_t pts_per_block) {
  __shared__ double4 s_atom[GRAD_ATOMS];
  __shared__ double s_pair[GRAD_ATOMS * NV * 3];
  __shared__ double s_red[GRAD_THREADS / 32][GRAD_ATOMS * 3][2];
  const int tid = threadIdx.x;
  const int a0 = blockIdx.y * GRAD_ATOMS;
  const int na = min(GRAD_ATOMS, n_atoms - a0);
  if (tid < na) s_atom[tid] = atoms[a0 + tid];
  for (int i = tid; i < na * NV * 3; i += GRAD_THREADS) s_pair[i] = pair[(size_t)a0 * NV * 3 + i];
  __syncthreads();
  double acc[GRAD_ATOMS][3];
#pragma unroll
  for (int a = 0; a < GRAD_ATOMS; ++a) acc[a][0] = acc[a][1] = acc[a][2] = 0.0;
  const double rmin2 = r_min * r_min;
  const size_t p0 = (size_t)blockIdx.x * pts_per_block;
  const size_t p1 = min(npts, p0 + pts_per_block);
  for (size_t idx = p0 + tid; idx < p1; idx += GRAD_THREADS) {
    const int iz = (int)(idx % n), iy = (int)((idx / n) % n), ix = (int)(idx / ((size_t)n * n));
    const double x = __dadd_rn(ox, __dmul_rn(h, (double)ix));
    const double y = __dadd_rn(oy, __dmul_rn(h, (double)iy));
    const double z = __dadd_rn(oz, __dmul_rn(h, (double)iz));
    double gw[NV];
#pragma unroll
    for (int g = 0; g < NV; ++g) gw[g] = gwf[(size_t)g * npts + idx];
    // (compiler barrier: re-read the atom tables from shared memory for every point instead of pinning all
    //  GRAD_ATOMS * (4 + 3 NV) of them in registers across the loop)
    asm volatile("" ::: "memory");
#pragma unroll
    for (int a = 0; a < GRAD_ATOMS; ++a) {
      if (a < na) {
        const double4 at = s_atom[a];
        const double dx = x - at.x, dy = y - at.y, dz = z - at.z;
        const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
        if (r2 >= rmin2) {                                  // inside the clamp the potential is flat
          double rinv = (double)rsqrtf((float)r2);
          rinv = rinv * fma(-0.5 * r2, rinv * rinv, 1.5);
          rinv = rinv * fma(-0.5 * r2, rinv * rinv, 1.5);
          const double inv2 = rinv * rinv, inv3 = inv2 * rinv;
          const double* pp = s_pair + a * NV * 3;
          double coef = 0.0;
#pragma unroll
          for (int g = 0; g < NV; ++g) {
            const double s2 = pp[g * 3 + 1] * inv2;
            const double s6 = s2 * s2 * s2;
            coef += gw[g] * (pp[g * 3 + 0] * inv3 + pp[g * 3 + 2] * (12.0 * s6 * s6 - 6.0 * s6) * inv2);
          }
          acc[a][0] = fma(coef, dx, acc[a][0]);
          acc[a][1] = fma(coef, dy, acc[a][1]);
          acc[a][2] = fma(coef, dz, acc[a][2]);
        }
      }
    }
  }
  // block sum in double-double, fixed order
  const int lane = tid & 31, wid = tid >> 5;
#pragma unroll
  for (int a = 0; a < GRAD_ATOMS; ++a)
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      double v = acc[a][k];                                // 32 per-thread sums: plain fp64 tree, then double-double
      for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
      if (lane == 0) { s_red[wid][a * 3 + k][0] = v; s_red[wid][a * 3 + k][1] = 0.0; }
    }
  __syncthreads();
  if (tid < na * 3) {
    double hi = 0.0, lo = 0.0;
    for (int wv = 0; wv < GRAD_THREADS / 32; ++wv) dd_add(hi, lo, s_red[wv][tid][0], s_red[wv][tid][1]);
    dd_norm(hi, lo);
    double* dst = partial + (((size_t)blockIdx.x * n_atoms + a0) * 3 + tid) * 2;
    dst[0] = hi;
    dst[1] = lo;
  }
}

__global__ void gradient_final_kernel(double* __restrict__ out, const double* __restrict__ partial, int nchunks,
                                      int n_atoms, double kT) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;    // atom * 3 + component
  if (e >= n_atoms * 3) return;
  double hi = 0.0, lo = 0.0;
  for (int c = 0; c < nchunks; ++c) {
    const double* p = partial + ((size_t)c * n_atoms * 3 + e) * 2;
    dd_add(hi, lo, p[0], p[1]);
  }
  out[e] = kT * (hi + lo);
}

// d_gw: one field-set of scratch; d_atoms: [n_atoms] double4 (x, y, z, unused); d_pair as in launch_potential;
// d_partial: nchunks*n_atoms*3*2 doubles; d_out: n_atoms*3 doubles.  Returns the number of kernels launched.
int launch_gradient(const Grid& g, const Buffers& b, const SolverParams& sp, int n_atoms, double* d_gw,
                    const double* d_atoms, const double* d_pair, double* d_partial, int nchunks, double* d_out,
                    cudaStream_t s) {
  if (n_atoms == 0) return 0;
  gradient_weights_kernel<<<148 * 8, 256, 0, s>>>(d_gw, b.tau, b.w, b.rhov, g.npts, g.nv, g.h * g.h * g.h, sp.closure,
                                                 sp.pse_order);
  const size_t per = (g.npts + nchunks - 1) / nchunks;
  dim3 grid((unsigned)nchunks, (unsigned)((n_atoms + GRAD_ATOMS - 1) / GRAD_ATOMS));
  const double4* at = reinterpret_cast<const double4*>(d_atoms);
#define GRD(NV)                                                                                                     \
  gradient_kernel<NV><<<grid, GRAD_THREADS, 0, s>>>(d_partial, d_gw, at, d_pair, n_atoms, g.n, g.h, g.origin[0],   \
                                                    g.origin[1], g.origin[2], sp.r_min, g.npts, per)
  switch (g.nv) {
    case 1: GRD(1); break;
    case 2: GRD(2); break;
    case 4: GRD(4); break;
    case 8: GRD(8); break;
    default: return 0;
  }
#undef GRD
  gradient_final_kernel<<<(n_atoms * 3 + 127) / 128, 128, 0, s>>>(d_out, d_partial, nchunks, n_atoms, sp.kT);
  return 3;
}

}  // namespace r3d
