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

// One atom - grid point pair: adds the pair's (1 - exp(-kappa r))/r term to ph (WITH_PHI; never cut off) and its
// short-range terms -beta [C q q exp(-kappa r)/r + LJ] to acc[g] (WITH_W; only when the pair is inside the cutoff).
// qa = beta C q_a; pp = (beta C q_a q_g, sigma_ag^2, 4 beta eps_ag) per site.
// 1/r: float rsqrt seed + two Newton steps in double (~2 ulp; r^2 is far inside the float range).  Beyond kappa r = 40,
// exp(-kappa r) < 5e-18 vanishes against 1 in double precision: (1 - exp(-kappa r))/r is 1/r to the last bit and the
// short-range Coulomb term is 0, so far pairs (most of them on the large grids) need no exp at all.
template <int NV, bool WITH_PHI, bool WITH_W>
__device__ __forceinline__ void pair_terms(double r2, double qa, const double* __restrict__ pp, double kappa,
                                           double r_min, double rmin2, double far2, bool cut, double rcut2,
                                           double& ph, double (&acc)[NV]) {
  const bool inside = WITH_W && (!cut || r2 < rcut2);
  if (r2 >= rmin2) {
    double rinv = (double)rsqrtf((float)r2);
    rinv = rinv * fma(-0.5 * r2, rinv * rinv, 1.5);
    rinv = rinv * fma(-0.5 * r2, rinv * rinv, 1.5);
    if (r2 > far2) {
      if (WITH_PHI) ph = fma(qa, rinv, ph);
      if (inside) {                                         // LJ reaches further than exp(-kappa r)
        const double inv2 = rinv * rinv;
#pragma unroll
        for (int g = 0; g < NV; ++g) {
          const double s2 = pp[g * 3 + 1] * inv2;
          const double s6 = s2 * s2 * s2;
          acc[g] -= pp[g * 3 + 2] * (s6 * s6 - s6);
        }
      }
    } else if (WITH_PHI || inside) {
      const double kr = kappa * (r2 * rinv);
      if (WITH_PHI && !WITH_W && kr > 26.0) {
        // phi alone, 26 < kappa r <= 40: exp(-kappa r) < 5.2e-12, so a single-precision exponential (relative error
        // < 3e-6 including the rounding of its argument) changes 1 - exp(-kappa r) by < 2e-17, a tenth of its last bit
        ph = fma(qa, (1.0 - (double)__expf(-(float)kr)) * rinv, ph);
        return;
      }
      // 1 - exp(-kappa r): expm1 where the subtraction would cancel, exp elsewhere
      const double ex = (kr < 0.5) ? 1.0 + expm1(-kr) : exp(-kr);
      if (WITH_PHI) {
        const double om = (kr < 0.5) ? -expm1(-kr) : 1.0 - ex;
        ph = fma(qa, om * rinv, ph);
      }
      if (inside) {
        const double sc = ex * rinv;                        // exp(-kappa r)/r = 1/r - (1 - exp(-kappa r))/r
        const double inv2 = rinv * rinv;
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
    const double lr = (kr < 1e-8) ? kappa : -em / rt;       // (1 - exp(-kappa r)) / r and its limit
    if (WITH_PHI) ph += qa * lr;
    if (inside) {
      const double rc = fmax(rt, r_min);
      const double sc = (rt >= r_min) ? (1.0 + em) / rt : (cut ? exp(-kappa * rc) / rc : 1.0 / rc - lr);
      const double inv2 = 1.0 / (rc * rc);
#pragma unroll
      for (int g = 0; g < NV; ++g) {
        const double s2 = pp[g * 3 + 1] * inv2;
        const double s6 = s2 * s2 * s2;
        acc[g] -= pp[g * 3 + 0] * sc + pp[g * 3 + 2] * (s6 * s6 - s6);
      }
    }
  }
}

template <int NV>
__global__ void __launch_bounds__(128)
    potential_kernel(double* __restrict__ w, double* __restrict__ phi, const double4* __restrict__ atoms,
                     const double* __restrict__ pair, int n_atoms, int ny, int nz, int ix0, double h, double ox,
                     double oy, double oz, double kappa, double r_min, double rcut2, size_t npts) {
  __shared__ double4 s_atom[ATOM_CHUNK];
  __shared__ double s_pair[ATOM_CHUNK * NV * 3];
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;   // npts is a multiple of blockDim
  const int iz = (int)(idx % nz), iy = (int)((idx / nz) % ny), ix = ix0 + (int)(idx / ((size_t)nz * ny));
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
      pair_terms<NV, true, true>(r2, at.w, s_pair + a * NV * 3, kappa, r_min, rmin2, far2, cut, rcut2, ph, acc);
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
  potential_kernel<NV><<<blocks, 128, 0, s>>>(b.w, b.phi, at, d_pair, n_atoms, g.ny, g.nz, g.ix0, g.h, g.origin[0], \
                                              g.origin[1], g.origin[2], sp.kappa, sp.r_min, rcut2, g.npts)
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
// Cell-list grid potential (rcut > 0; Q12): w alone, from the atoms within the cutoff of each grid point.
// The host bins the atoms into cubic cells of edge >= rcut / 2 and sorts them by cell, z fastest, so that the cells
// (cx, cy, cz0..cz1) of one column are ONE contiguous range of the sorted atom table.  A CTA owns a brick of 4 x 8 x 8
// grid points and walks the cell columns that can reach the brick (box-box distance test), staging each column's
// atoms through shared memory; a thread (one grid point) applies the sharp test r < rcut per atom -- the same pair set,
// the same rounded r^2 and the same pair arithmetic as the all-pairs kernel, accumulated in the sorted atom order.
// phi(r), which is never cut off, is left to phi_kernel (computed when first needed, see api.cu).
// ------------------------------------------------------------------------------------------------
struct CellGrid {
  int nc[3];             // cells per axis
  double lo[3];          // lower corner of cell (0, 0, 0)
  double edge;           // cell edge
};
constexpr int BRICK_X = 4, BRICK_Y = 8, BRICK_Z = 8, BRICK_THREADS = BRICK_X * BRICK_Y * BRICK_Z;
constexpr int CELL_CHUNK = 128;

template <int NV>
__global__ void __launch_bounds__(BRICK_THREADS)
    w_cells_kernel(double* __restrict__ w, const double4* __restrict__ atoms, const double* __restrict__ pair,
                   const int* __restrict__ cell_start, CellGrid cg, int ny, int nz, int ix0, double h, double ox,
                   double oy, double oz, double kappa, double r_min, double rcut, size_t npts) {
  __shared__ double4 s_atom[CELL_CHUNK];
  __shared__ double s_pair[CELL_CHUNK * NV * 3];
  const int tid = threadIdx.x;
  const int iz = blockIdx.x * BRICK_Z + tid % BRICK_Z;
  const int iy = blockIdx.y * BRICK_Y + (tid / BRICK_Z) % BRICK_Y;
  const int ixl = blockIdx.z * BRICK_X + tid / (BRICK_Z * BRICK_Y);   // plane of this context's slab
  const int ix = ix0 + ixl;
  const double x = __dadd_rn(ox, __dmul_rn(h, (double)ix));
  const double y = __dadd_rn(oy, __dmul_rn(h, (double)iy));
  const double z = __dadd_rn(oz, __dmul_rn(h, (double)iz));
  double acc[NV];
#pragma unroll
  for (int g = 0; g < NV; ++g) acc[g] = 0.0;
  double ph_unused = 0.0;
  const double rcut2 = rcut * rcut, rmin2 = r_min * r_min, far2 = 1600.0 / (kappa * kappa);
  // the brick's box (with a safety margin of a grid spacing against rounding in the cell arithmetic) and the cells it
  // can reach; everything below is uniform over the CTA
  const double bx0 = ox + h * (ix0 + blockIdx.z * BRICK_X) - h, bx1 = ox + h * (ix0 + blockIdx.z * BRICK_X + BRICK_X - 1) + h;
  const double by0 = oy + h * (blockIdx.y * BRICK_Y) - h, by1 = oy + h * (blockIdx.y * BRICK_Y + BRICK_Y - 1) + h;
  const double bz0 = oz + h * (blockIdx.x * BRICK_Z) - h, bz1 = oz + h * (blockIdx.x * BRICK_Z + BRICK_Z - 1) + h;
  auto cell_lo = [&](double v, int axis) { return max(0, (int)floor((v - rcut - cg.lo[axis]) / cg.edge)); };
  auto cell_hi = [&](double v, int axis) { return min(cg.nc[axis] - 1, (int)floor((v + rcut - cg.lo[axis]) / cg.edge)); };
  const int cx0 = cell_lo(bx0, 0), cx1 = cell_hi(bx1, 0);
  const int cy0 = cell_lo(by0, 1), cy1 = cell_hi(by1, 1);
  const int cz0 = cell_lo(bz0, 2), cz1 = cell_hi(bz1, 2);
  // distance from the interval [b0, b1] to cell c of an axis
  auto gap = [&](double b0, double b1, int c, int axis) {
    const double c0 = cg.lo[axis] + c * cg.edge, c1 = c0 + cg.edge;
    return fmax(0.0, fmax(c0 - b1, b0 - c1));
  };
  if (cz0 <= cz1) {
    for (int cx = cx0; cx <= cx1; ++cx) {
      const double gx = gap(bx0, bx1, cx, 0);
      for (int cy = cy0; cy <= cy1; ++cy) {
        const double gy = gap(by0, by1, cy, 1);
        if (gx * gx + gy * gy > rcut2) continue;
        const size_t col = ((size_t)cx * cg.nc[1] + cy) * cg.nc[2];
        const int a_begin = cell_start[col + cz0], a_end = cell_start[col + cz1 + 1];
        for (int a0 = a_begin; a0 < a_end; a0 += CELL_CHUNK) {
          const int na = min(CELL_CHUNK, a_end - a0);
          __syncthreads();
          for (int i = tid; i < na; i += BRICK_THREADS) s_atom[i] = atoms[a0 + i];
          for (int i = tid; i < na * NV * 3; i += BRICK_THREADS) s_pair[i] = pair[(size_t)a0 * NV * 3 + i];
          __syncthreads();
          for (int a = 0; a < na; ++a) {
            const double4 at = s_atom[a];
            const double dx = x - at.x, dy = y - at.y, dz = z - at.z;
            const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
            if (r2 < rcut2)
              pair_terms<NV, false, true>(r2, at.w, s_pair + a * NV * 3, kappa, r_min, rmin2, far2, true, rcut2, ph_unused, acc);
          }
        }
      }
    }
  }
  const size_t idx = ((size_t)ixl * ny + iy) * nz + iz;
#pragma unroll
  for (int g = 0; g < NV; ++g) w[(size_t)g * npts + idx] = acc[g];
}

// d_atoms / d_pair: the atom and pair tables SORTED by cell; d_cell_start: [ncells + 1] first atom of every cell
int launch_w_cells(const Grid& g, const Buffers& b, const SolverParams& sp, const double* d_atoms, const double* d_pair,
                   const int* d_cell_start, const int nc[3], const double lo[3], double edge, double rcut,
                   cudaStream_t s) {
  CellGrid cg;
  for (int i = 0; i < 3; ++i) { cg.nc[i] = nc[i]; cg.lo[i] = lo[i]; }
  cg.edge = edge;
  dim3 grid((unsigned)(g.nz / BRICK_Z), (unsigned)(g.ny / BRICK_Y), (unsigned)(g.nxl / BRICK_X));
  const double4* at = reinterpret_cast<const double4*>(d_atoms);
#define WCELL(NV)                                                                                                   \
  w_cells_kernel<NV><<<grid, BRICK_THREADS, 0, s>>>(b.w, at, d_pair, d_cell_start, cg, g.ny, g.nz, g.ix0, g.h,      \
                                                    g.origin[0], g.origin[1], g.origin[2], sp.kappa, sp.r_min, rcut, \
                                                    g.npts)
  switch (g.nv) {
    case 1: WCELL(1); break;
    case 2: WCELL(2); break;
    case 4: WCELL(4); break;
    case 8: WCELL(8); break;
    default: return 0;
  }
#undef WCELL
  return 1;
}

// phi(r) = beta C sum_a q_a (1 - exp(-kappa r_a)) / r_a over ALL atoms (Eq. 29; never cut off).  Two grid points per
// thread (z and z + n/2: two independent dependency chains), atoms staged through shared memory.
constexpr int PHI_CHUNK = 256;
__global__ void __launch_bounds__(128)
    phi_kernel(double* __restrict__ phi, const double4* __restrict__ atoms, int n_atoms, int ny, int nz, int ix0,
               double h, double ox, double oy, double oz, double kappa, double r_min) {
  __shared__ double4 s_atom[PHI_CHUNK];
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;      // npts / 2 threads
  const int hz = nz / 2;
  const int iz = (int)(t % hz), iy = (int)((t / hz) % ny), ixl = (int)(t / ((size_t)hz * ny));
  const double x = __dadd_rn(ox, __dmul_rn(h, (double)(ix0 + ixl)));
  const double y = __dadd_rn(oy, __dmul_rn(h, (double)iy));
  const double z0 = __dadd_rn(oz, __dmul_rn(h, (double)iz));
  const double z1 = __dadd_rn(oz, __dmul_rn(h, (double)(iz + hz)));
  const double rmin2 = r_min * r_min, far2 = 1600.0 / (kappa * kappa);
  double ph0 = 0.0, ph1 = 0.0;
  double none[1] = {0.0};
  for (int a0 = 0; a0 < n_atoms; a0 += PHI_CHUNK) {
    const int na = min(PHI_CHUNK, n_atoms - a0);
    __syncthreads();
    for (int i = threadIdx.x; i < na; i += blockDim.x) s_atom[i] = atoms[a0 + i];
    __syncthreads();
#pragma unroll 2
    for (int a = 0; a < na; ++a) {
      const double4 at = s_atom[a];
      const double dx = x - at.x, dy = y - at.y, dz0 = z0 - at.z, dz1 = z1 - at.z;
      const double rxy = __dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy));
      pair_terms<1, true, false>(__dadd_rn(rxy, __dmul_rn(dz0, dz0)), at.w, nullptr, kappa, r_min, rmin2, far2, false, 0.0, ph0, none);
      pair_terms<1, true, false>(__dadd_rn(rxy, __dmul_rn(dz1, dz1)), at.w, nullptr, kappa, r_min, rmin2, far2, false, 0.0, ph1, none);
    }
  }
  const size_t idx = ((size_t)ixl * ny + iy) * nz + iz;
  phi[idx] = ph0;
  phi[idx + hz] = ph1;
}

// d_atoms: [n_atoms] (x, y, z, beta C q_a), any order
int launch_phi(const Grid& g, const Buffers& b, const SolverParams& sp, int n_atoms, const double* d_atoms,
               cudaStream_t s) {
  const unsigned blocks = (unsigned)(g.npts / 2 / 128);
  phi_kernel<<<blocks, 128, 0, s>>>(b.phi, reinterpret_cast<const double4*>(d_atoms), n_atoms, g.ny, g.nz, g.ix0, g.h,
                                   g.origin[0], g.origin[1], g.origin[2], sp.kappa, sp.r_min);
  return 1;
}

// ------------------------------------------------------------------------------------------------
// phi~(k): separable phase tables E_axis[a][j] = exp(-i k_j (R_a,axis - r0,axis)), then
//   phik[jx][jy_l][p] = (4 pi beta C / dV) kappa^2 / (k^2 (k^2 + kappa^2)) sum_a q_a Ex[a][jx] Ey[a][jy0 + jy_l] Ez[a][2p]
// d_phase: [3][n_atoms][nmax] complex (axis a uses its first n_a entries; the z table holds only the even j at index p,
// nz/2 entries used)
// ------------------------------------------------------------------------------------------------
struct AxisLen { int n[3]; };

__global__ void phase_kernel(double2* __restrict__ phase, const double4* __restrict__ atoms, int n_atoms, AxisLen al,
                             int nmax, double h, double ox, double oy, double oz) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t total = (size_t)3 * n_atoms * nmax;
  if (idx >= total) return;
  const int j = (int)(idx % nmax);
  const int a = (int)((idx / nmax) % n_atoms);
  const int axis = (int)(idx / ((size_t)nmax * n_atoms));
  const int n = al.n[axis];
  const double4 at = atoms[a];
  const double d = axis == 0 ? at.x - ox : (axis == 1 ? at.y - oy : at.z - oz);
  int jj = j;
  if (axis == 2) jj = 2 * j;
  if (jj >= n) { phase[idx] = make_double2(0.0, 0.0); return; }
  const double f = (jj < n / 2) ? (jj + 0.5) : (jj + 0.5 - n);          // k = dk * f, dk = 2 pi / (n h)
  double sn, cs;
  sincospi(2.0 * f * (d / (n * h)), &sn, &cs);
  phase[idx] = make_double2(cs, -sn);
}

constexpr int PT_JY = 8;      // jy values per thread
constexpr int PT_AC = 32;     // atoms per shared-memory chunk

__global__ void __launch_bounds__(64)
    phi_tilde_kernel(double2* __restrict__ phik, const double2* __restrict__ phase, const double* __restrict__ qa,
                     int n_atoms, AxisLen al, int nmax, int nyl, int jy0g, double h, double kappa, double pref) {
  __shared__ double2 s_a[PT_AC][PT_JY];
  const int nzh = al.n[2] / 2;
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  const int jyl0 = blockIdx.y * PT_JY;                   // first row of this CTA inside the context's k-space slab
  const int jx = blockIdx.z;
  const double2* Ex = phase;
  const double2* Ey = phase + (size_t)n_atoms * nmax;
  const double2* Ez = phase + (size_t)2 * n_atoms * nmax;
  double2 acc[PT_JY];
#pragma unroll
  for (int i = 0; i < PT_JY; ++i) acc[i] = make_double2(0.0, 0.0);
  for (int a0 = 0; a0 < n_atoms; a0 += PT_AC) {
    const int na = min(PT_AC, n_atoms - a0);
    __syncthreads();
    for (int i = threadIdx.x; i < na * PT_JY; i += blockDim.x) {
      const int a = a0 + i / PT_JY, jy = jy0g + jyl0 + i % PT_JY;
      const double2 ex = Ex[(size_t)a * nmax + jx], ey = Ey[(size_t)a * nmax + jy];
      const double q = qa[a];
      s_a[i / PT_JY][i % PT_JY] = make_double2(q * (ex.x * ey.x - ex.y * ey.y), q * (ex.x * ey.y + ex.y * ey.x));
    }
    __syncthreads();
    if (p < nzh) {
      for (int a = 0; a < na; ++a) {
        const double2 ez = Ez[(size_t)(a0 + a) * nmax + p];
#pragma unroll
        for (int i = 0; i < PT_JY; ++i) {
          const double2 v = s_a[a][i];
          acc[i].x += v.x * ez.x - v.y * ez.y;
          acc[i].y += v.x * ez.y + v.y * ez.x;
        }
      }
    }
  }
  if (p >= nzh) return;
  auto kof = [&](int j, int axis) {
    const int n = al.n[axis];
    const double dk = 2.0 * 3.14159265358979323846 / (n * h);
    return dk * ((j < n / 2) ? (j + 0.5) : (j + 0.5 - n));
  };
  const double kx = kof(jx, 0), kz = kof(2 * p, 2);
#pragma unroll
  for (int i = 0; i < PT_JY; ++i) {
    const double ky = kof(jy0g + jyl0 + i, 1);
    const double k2 = kx * kx + ky * ky + kz * kz;
    const double f = pref * kappa * kappa / (k2 * (k2 + kappa * kappa));
    phik[((size_t)jx * nyl + (jyl0 + i)) * nzh + p] = make_double2(f * acc[i].x, f * acc[i].y);
  }
}

int launch_phi_tilde(const Grid& g, const Buffers& b, const SolverParams& sp, int n_atoms, const double* d_atoms,
                     double2* d_phase, cudaStream_t s) {
  const size_t total = (size_t)3 * n_atoms * g.nmax;
  const double4* at = reinterpret_cast<const double4*>(d_atoms);
  const AxisLen al{{g.nx, g.ny, g.nz}};
  int launched = 1;
  if (total > 0) {                                       // an empty solute has no phase table (phi~ = 0)
    phase_kernel<<<(unsigned)((total + 255) / 256), 256, 0, s>>>(d_phase, at, n_atoms, al, g.nmax, g.h, g.origin[0],
                                                                g.origin[1], g.origin[2]);
    launched = 2;
  }
  // charges q_a live in a separate array right after the atom records (set up by the API layer)
  const double* qa = d_atoms + (size_t)4 * n_atoms;
  const int nzh = g.nz / 2;
  const int bx = nzh < 64 ? nzh : 64;
  dim3 grid((nzh + bx - 1) / bx, g.nyl / PT_JY, g.nx);
  const double pref = 4.0 * 3.14159265358979323846 * sp.beta * COULOMB / (g.h * g.h * g.h);
  phi_tilde_kernel<<<grid, bx, 0, s>>>(b.phik, d_phase, qa, n_atoms, al, g.nmax, g.nyl, g.jy0, g.h, sp.kappa, pref);
  return launched;
}

// ------------------------------------------------------------------------------------------------
// chi per |k| shell.  table: [n_k][nv][nv] (chi[m][g'][g]);  out: [nshell][g][k] = chi_{(g xor k) g}: row g holds
// the column of Eq. 13 that site g needs, ordered for the butterfly exchange of kspace_point (kspace_kernel.cu)
// ------------------------------------------------------------------------------------------------
__global__ void chi_shell_kernel(double* __restrict__ out, const double* __restrict__ table, int n_k, double k0,
                                 double dkt, int nv, double dk_grid, double quarter_w, int nshell) {
  const int sidx = blockIdx.x * blockDim.x + threadIdx.x;
  if (sidx >= nshell) return;
  const double kmag = dk_grid * sqrt(2.0 * sidx + quarter_w);   // |k|^2 = dk0^2 (s + (wx + wy + wz) / 4), s = 2 sidx
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
      out[(size_t)sidx * st + g * nv + (gp ^ g)] = l0 * t[0] + l1 * t[st] + l2 * t[2 * st] + l3 * t[3 * st];
    }
}

int launch_chi_shell(const Grid& g, const Buffers& b, const double* d_table, int n_k, double k0, double dk,
                     cudaStream_t s) {
  const double dk_grid = 2.0 * 3.14159265358979323846 / (g.nmax * g.h);
  chi_shell_kernel<<<(g.nshell + 127) / 128, 128, 0, s>>>(b.chi_shell, d_table, n_k, k0, dk, g.nv, dk_grid,
                                                          0.25 * (g.wx + g.wy + g.wz), g.nshell);
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

// one warp per site type and sum: the per-CTA double-double partials are added in a fixed order (lane l takes l, l + 32,
// ..., then the shuffle tree).  blockDim = 32 * 2 * MAX_NV; warp = g (free-energy integrand) or MAX_NV + g (c_sr alone).
__global__ void __launch_bounds__(64 * MAX_NV)
    free_energy_final_kernel(double* __restrict__ out, const double* __restrict__ part, int nblocks,
                             const double* __restrict__ rhov, int nv, double scale, double dv) {
  const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int g = wid % MAX_NV, second = wid / MAX_NV;
  if (g >= nv) return;
  double hi, lo;
  warp_sum_partials(part + ((size_t)second * nblocks * MAX_NV + g) * 2, nblocks, lane, hi, lo, MAX_NV);
  if (lane == 0) out[second * MAX_NV + g] = second ? dv * (hi + lo) : scale * rhov[g] * (hi + lo);
}

int launch_free_energy(const Grid& g, const Buffers& b, const SolverParams& sp, double* d_out, cudaStream_t s) {
  const int blocks = FE_BLOCKS;
  free_energy_kernel<<<blocks, 256, 0, s>>>(b.fe_part, b.tau, b.w, b.phi, b.qv, b.state, g.nv, g.npts, g.field,
                                            sp.closure, sp.pse_order);
  free_energy_final_kernel<<<1, 64 * MAX_NV, 0, s>>>(d_out, b.fe_part, blocks, b.rhov, g.nv, sp.kT * g.h * g.h * g.h,
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
                    const double* __restrict__ pair, int n_atoms, int ny, int nz, int ix0, double h, double ox,
                    double oy, double oz, double r_min, size_t npts, size_t pts_per_block) {
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
    const int iz = (int)(idx % nz), iy = (int)((idx / nz) % ny), ix = ix0 + (int)(idx / ((size_t)nz * ny));
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

// one warp per (atom, component): the chunk partials are added in a fixed order (warp_sum_partials)
__global__ void __launch_bounds__(256)
    gradient_final_kernel(double* __restrict__ out, const double* __restrict__ partial, int nchunks, int n_atoms,
                          double kT) {
  const int e = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);    // atom * 3 + component
  if (e >= n_atoms * 3) return;
  double hi, lo;
  warp_sum_partials(partial + (size_t)e * 2, nchunks, threadIdx.x & 31, hi, lo, n_atoms * 3);
  if ((threadIdx.x & 31) == 0) out[e] = kT * (hi + lo);
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
  gradient_kernel<NV><<<grid, GRAD_THREADS, 0, s>>>(d_partial, d_gw, at, d_pair, n_atoms, g.ny, g.nz, g.ix0, g.h,   \
                                                    g.origin[0], g.origin[1], g.origin[2], sp.r_min, g.npts, per)
  switch (g.nv) {
    case 1: GRD(1); break;
    case 2: GRD(2); break;
    case 4: GRD(4); break;
    case 8: GRD(8); break;
    default: return 0;
  }
#undef GRD
  gradient_final_kernel<<<(n_atoms * 3 + 7) / 8, 256, 0, s>>>(d_out, d_partial, nchunks, n_atoms, sp.kT);
  return 3;
}

// ------------------------------------------------------------------------------------------------
// fp64 FMA peak of the device, measured: 16 independent DFMA chains per thread, 1024 resident threads per SM.  The
// denominator of the setup kernels' roofline (they are bound by plain fp64 arithmetic, not by HBM).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dfma_peak_kernel(double* __restrict__ out, int iters, double a, double b) {
  double v[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = (double)(threadIdx.x + i);
  for (int k = 0; k < iters; ++k) {
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = fma(v[i], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += v[i];
  if (s == 12345.678) out[0] = s;                        // never true: keeps the chains alive
}

// -> fp64 TFLOP/s (2 flops per DFMA) over ~reps launches; returns the best launch
double measure_dfma_peak(int num_sms, double* d_scratch, cudaStream_t s) {
  const int iters = 4096, blocks = num_sms * 4, threads = 256;
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return 0.0;
  double best = 0.0;
  for (int rep = 0; rep < 5; ++rep) {
    cudaEventRecord(e0, s);
    dfma_peak_kernel<<<blocks, threads, 0, s>>>(d_scratch, iters, 0.999999, 1e-9);
    cudaEventRecord(e1, s);
    if (cudaEventSynchronize(e1) != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double tf = 2.0 * 16.0 * iters * (double)blocks * threads / (ms * 1e-3) / 1e12;
    if (rep > 0 && tf > best) best = tf;                 // the first launch is a warm-up
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return best;
}

}  // namespace r3d
