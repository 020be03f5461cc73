// rism1d.cu -- the 1D solvent-solvent RISM solve on the GPU (include/rism1d.h; Eq. 4, 90-99 Eq. 5-7, 109,
// 158-172).  The problem is small (n_s^2 pair functions of M - 1 radial points: a few
// hundred thousand doubles), so every step is a short kernel over all pairs at once and the iteration is bound by
// launch latency, not by bandwidth; what matters is that the whole solve -- thousands of iterations over a charge ramp
// -- never leaves the device.  One iteration:
//   closure1d      g = closure(w + tau), c_sr = g - 1 - tau, odd extension of r c_sr(r) into the FFT buffer
//   fft1d_pass x3  batched complex FFT of length 2M (Stockham, radix 32): the type-I sine transform of every pair
//   kspace1d       per k: C = C_sr - F, H = (I - W C R)^-1 W C W (Gaussian elimination, partial pivoting), odd
//                  extension of k (H - C_sr)
//   fft1d_pass x3
//   residual1d     tau' symmetrised, R = tau' - tau, Z = tau + b R into the history, per-CTA Gram partials
//   gram_solve     the 3D path's kernel: sums the partial rows in order, rms test, restart rule, bordered solve
//   mdiis_update   the 3D path's kernel: tau = sum_i c_i Z_i
// The MDIIS state, its bookkeeping and its update are the 3D path's (DevState, mdiis_device.cuh, mdiis_kernels.cu).
// Pair arrays are [a][b][i], i = 0..M-1 with entry 0 unused (kept 0): even, 16-byte aligned slices.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <vector>

#include "../../include/rism1d.h"
#include "fft_core.cuh"
#include "rism3d_internal.h"

using namespace r3d;

namespace {

constexpr int MAX_S = 8;                   // full sites
constexpr int R1D_THREADS = 256;

struct Solvent1d {
  double q[MAX_S], sigma[MAX_S], eps[MAX_S], rho[MAX_S];
  int species[MAX_S];
  double bond[MAX_S][MAX_S];
};

// ---- batched complex FFT of length L through global memory (the data of all pairs fits the L2) -----------------
// One Stockham pass of radix R: thread j of a transform takes v[r] = in[j + r L/R], applies exp(-2 pi i r k/(Ns R)),
// k = j mod Ns, transforms, and writes out[(j - k) R + k + r Ns].  tab[a] = exp(-2 pi i a / L).
template <int R>
__global__ void __launch_bounds__(128)
    fft1d_pass_kernel(const cplx* __restrict__ in, cplx* __restrict__ out, const cplx* __restrict__ tab, int L, int Ns,
                      int n_batch, const DevState* __restrict__ st) {
  if (st->done) return;
  const int per = L / R;
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= per * n_batch) return;
  const int batch = idx / per, j = idx % per;
  const int k = j & (Ns - 1);
  const cplx* src = in + (size_t)batch * L;
  cplx* dst = out + (size_t)batch * L;
  const int tstep = L / (Ns * R);
  cplx v[R];
#pragma unroll
  for (int r = 0; r < R; ++r) {
    v[r] = src[j + r * per];
    if (r > 0 && k > 0) v[r] = cmul(v[r], __ldg(tab + ((r * k * tstep) & (L - 1))));
  }
  Dft<R, -1>::run(v);
  const int j0 = (j - k) * R + k;
#pragma unroll
  for (int r = 0; r < R; ++r) dst[j0 + r * Ns] = v[r];
}

// w_ab(r_i) = -beta [4 eps_ab ((s/r)^12 - (s/r)^6) + C lam^2 q_a q_b exp(-kappa r)/r]
__global__ void setup_w1d_kernel(double* __restrict__ w, Solvent1d sv, int ns, int M, double dr, double beta,
                                 double kappa, double lam) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= ns * ns * M) return;
  const int i = idx % M, ab = idx / M, a = ab / ns, b = ab % ns;
  if (i == 0) { w[idx] = 0.0; return; }
  const double r = i * dr;
  const double s = 0.5 * (sv.sigma[a] + sv.sigma[b]);
  const double e = sqrt(sv.eps[a] * sv.eps[b]);
  const double sr2 = (s / r) * (s / r);
  const double sr6 = sr2 * sr2 * sr2;
  const double lj = 4.0 * e * (sr6 * sr6 - sr6);
  const double qq = lam * lam * sv.q[a] * sv.q[b];
  w[idx] = -beta * (lj + COULOMB * qq * exp(-kappa * r) / r);
}

// closure + c_sr + odd extension of x_i = r_i c_sr(r_i):  z[i] = x_i, z[L - i] = -x_i, z[0] = z[M] = 0  (L = 2M)
__global__ void closure1d_kernel(cplx* __restrict__ z, const double* __restrict__ tau, const double* __restrict__ w,
                                 int npairs, int M, double dr, int closure, int order, const DevState* __restrict__ st) {
  if (st->done) return;
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= npairs * M) return;
  const int i = idx % M, ab = idx / M;
  cplx* zz = z + (size_t)ab * 2 * M;
  if (i == 0) {
    zz[0] = make_double2(0.0, 0.0);
    zz[M] = make_double2(0.0, 0.0);
    return;
  }
  const double t = tau[idx];
  const double x = (closure_g(w[idx] + t, closure, order) - 1.0 - t) * (i * dr);
  zz[i] = make_double2(x, 0.0);
  zz[2 * M - i] = make_double2(-x, 0.0);
}

// S_j = 2 sum_i x_i sin(pi i j / M) = -Im Z_j of the odd extension's transform
__device__ __forceinline__ double dst_value(const cplx* Z, int j) { return -Z[j].y; }

// per k_j: Eq. 4 solved for H, then the odd extension of k_j (H - C_sr)_ab for the way back.  chi_out != nullptr:
// also chi_ab(k_j) = W_ab + rho_a H_ab into chi_out[j - 1][a][b].
__global__ void __launch_bounds__(64)
    kspace1d_kernel(const cplx* __restrict__ Zin, cplx* __restrict__ zout, double* __restrict__ chi_out, Solvent1d sv,
                    int ns, int M, double dr, double beta, double kappa, double lam, const DevState* __restrict__ st) {
  if (chi_out == nullptr && st->done) return;
  const int j = blockIdx.x * blockDim.x + threadIdx.x + 1;
  if (j >= M) return;
  const int L = 2 * M;
  const double dk = 3.14159265358979323846 / (M * dr);
  const double k = j * dk;
  const double fwd = 2.0 * 3.14159265358979323846 * dr / k;          // F(k_j) = (2 pi dr / k_j) S_j
  double Csr[MAX_S][MAX_S], W[MAX_S][MAX_S], WC[MAX_S][MAX_S], A[MAX_S][MAX_S], B[MAX_S][MAX_S];
  for (int a = 0; a < ns; ++a)
    for (int b = 0; b < ns; ++b) {
      Csr[a][b] = fwd * dst_value(Zin + (size_t)(a * ns + b) * L, j);
      double wv = 0.0;
      if (a == b) wv = 1.0;
      else if (sv.species[a] == sv.species[b]) { const double x = k * sv.bond[a][b]; wv = sin(x) / x; }
      W[a][b] = wv;
    }
  const double flr = 4.0 * 3.14159265358979323846 * beta * COULOMB * kappa * kappa / (k * k * (k * k + kappa * kappa));
  for (int a = 0; a < ns; ++a)
    for (int b = 0; b < ns; ++b) {
      double acc = 0.0;
      for (int c = 0; c < ns; ++c) acc += W[a][c] * (Csr[c][b] - flr * lam * lam * sv.q[c] * sv.q[b]);   // W (C_sr - F)
      WC[a][b] = acc;
    }
  for (int a = 0; a < ns; ++a)
    for (int b = 0; b < ns; ++b) {
      A[a][b] = (a == b ? 1.0 : 0.0) - WC[a][b] * sv.rho[b];         // I - W C R
      double acc = 0.0;
      for (int c = 0; c < ns; ++c) acc += WC[a][c] * W[c][b];        // W C W
      B[a][b] = acc;
    }
  // A H = B: Gaussian elimination with partial pivoting, all right-hand sides at once
  for (int col = 0; col < ns; ++col) {
    int piv = col;
    for (int r = col + 1; r < ns; ++r)
      if (fabs(A[r][col]) > fabs(A[piv][col])) piv = r;
    if (piv != col)
      for (int c = 0; c < ns; ++c) {
        double t = A[col][c]; A[col][c] = A[piv][c]; A[piv][c] = t;
        t = B[col][c]; B[col][c] = B[piv][c]; B[piv][c] = t;
      }
    const double inv = 1.0 / A[col][col];
    for (int r = col + 1; r < ns; ++r) {
      const double f = A[r][col] * inv;
      for (int c = col; c < ns; ++c) A[r][c] -= f * A[col][c];
      for (int c = 0; c < ns; ++c) B[r][c] -= f * B[col][c];
    }
  }
  for (int r = ns - 1; r >= 0; --r)
    for (int c = 0; c < ns; ++c) {
      double acc = B[r][c];
      for (int m = r + 1; m < ns; ++m) acc -= A[r][m] * B[m][c];
      B[r][c] = acc / A[r][r];                                       // B now holds H
    }
  for (int a = 0; a < ns; ++a)
    for (int b = 0; b < ns; ++b) {
      if (chi_out) chi_out[((size_t)(j - 1) * ns + a) * ns + b] = W[a][b] + sv.rho[a] * B[a][b];
      if (zout) {
        const double y = (B[a][b] - Csr[a][b]) * k;
        cplx* zz = zout + (size_t)(a * ns + b) * L;
        zz[j] = make_double2(y, 0.0);
        zz[L - j] = make_double2(-y, 0.0);
        if (j == 1) { zz[0] = make_double2(0.0, 0.0); zz[M] = make_double2(0.0, 0.0); }
      }
    }
}

// tau'_ab(r_i) = (dk / (4 pi^2 r_i)) S_i, symmetrised; R = tau' - tau; Z = tau + b R; Gram partials of this CTA:
// rows[blockIdx][jj] (double-double), jj < nother: <R, R_other[jj]>, jj = nother: <R, R>
__global__ void __launch_bounds__(R1D_THREADS)
    residual1d_kernel(const cplx* __restrict__ Zin, const double* __restrict__ tau, double* __restrict__ Zh,
                      double* __restrict__ Rh, double* __restrict__ rows, int ns, int M, double dr, double bdamp, int Mhist,
                      const DevState* __restrict__ st) {
  if (st->done) return;
  __shared__ int s_other[MAX_M];
  __shared__ int s_nother;
  __shared__ double s_red[R1D_THREADS / 32][MAX_M + 1][2];
  if (threadIdx.x == 0) {
    const int m = st->m;
    const int skip = (m == Mhist) ? 1 : 0;
    s_nother = m - skip;
    for (int i = 0; i < m - skip; ++i) s_other[i] = st->list[i + skip];
  }
  __syncthreads();
  const int nother = s_nother;
  const size_t field = (size_t)ns * ns * M;
  const int cur = st->cur;
  const int L = 2 * M;
  const double dk = 3.14159265358979323846 / (M * dr);
  double acc[MAX_M + 1];
#pragma unroll
  for (int jj = 0; jj <= MAX_M; ++jj) acc[jj] = 0.0;
  for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < field; idx += (size_t)gridDim.x * blockDim.x) {
    const int i = (int)(idx % M), ab = (int)(idx / M), a = ab / ns, b = ab % ns;
    double r = 0.0, x = 0.0;
    if (i > 0) {
      const double fac = dk / (4.0 * 3.14159265358979323846 * 3.14159265358979323846 * (i * dr));
      const double t_ab = fac * dst_value(Zin + (size_t)ab * L, i);
      const double t_ba = fac * dst_value(Zin + (size_t)(b * ns + a) * L, i);
      x = tau[idx];
      r = 0.5 * (t_ab + t_ba) - x;
    }
    Rh[(size_t)cur * field + idx] = r;
    Zh[(size_t)cur * field + idx] = __dadd_rn(x, __dmul_rn(bdamp, r));
    acc[MAX_M] = fma(r, r, acc[MAX_M]);
#pragma unroll
    for (int jj = 0; jj < MAX_M; ++jj)
      if (jj < nother) acc[jj] = fma(r, Rh[(size_t)s_other[jj] * field + idx], acc[jj]);
  }
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int jj = 0; jj <= MAX_M; ++jj) {
    if (jj < nother || jj == MAX_M) {
      double hi = acc[jj], lo = 0.0;
      for (int o = 16; o > 0; o >>= 1) {
        const double h2 = __shfl_down_sync(0xffffffffu, hi, o), l2 = __shfl_down_sync(0xffffffffu, lo, o);
        dd_add(hi, lo, h2, l2);
      }
      if (lane == 0) { s_red[wid][jj][0] = hi; s_red[wid][jj][1] = lo; }
    }
  }
  __syncthreads();
  if (threadIdx.x <= MAX_M && (threadIdx.x < nother || threadIdx.x == MAX_M)) {
    const int jj = threadIdx.x;
    double hi = 0.0, lo = 0.0;
    for (int wv = 0; wv < R1D_THREADS / 32; ++wv) dd_add(hi, lo, s_red[wv][jj][0], s_red[wv][jj][1]);
    dd_norm(hi, lo);
    const int slot = (jj == MAX_M) ? nother : jj;                    // the row layout gram_solve_kernel reads
    *reinterpret_cast<double2*>(rows + ((size_t)blockIdx.x * GRAM_SLOT + slot) * 2) = make_double2(hi, lo);
  }
}

// pair functions of the current tau (which: 0 g, 1 tau, 2 c_sr) without the unused entry 0: dst [a][b][M - 1]
__global__ void get_pair1d_kernel(double* __restrict__ dst, const double* __restrict__ tau, const double* __restrict__ w,
                                  int npairs, int M, int which, int closure, int order) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= npairs * (M - 1)) return;
  const int i = idx % (M - 1) + 1, ab = idx / (M - 1);
  const double t = tau[(size_t)ab * M + i];
  const double g = closure_g(w[(size_t)ab * M + i] + t, closure, order);
  dst[idx] = which == 0 ? g : (which == 1 ? t : g - 1.0 - t);
}

// int c_sr,ab dr = 4 pi dr sum_i r_i^2 c_sr,ab(r_i): one CTA per pair, double-double, fixed order
__global__ void __launch_bounds__(256)
    c_integral1d_kernel(double* __restrict__ out, const double* __restrict__ tau, const double* __restrict__ w, int M,
                        double dr, int closure, int order) {
  __shared__ double s_red[8][2];
  const int ab = blockIdx.x;
  double hi = 0.0, lo = 0.0;
  for (int i = 1 + threadIdx.x; i < M; i += blockDim.x) {
    const double t = tau[(size_t)ab * M + i];
    const double c = closure_g(w[(size_t)ab * M + i] + t, closure, order) - 1.0 - t;
    const double r = i * dr;
    dd_add(hi, lo, c * r * r, 0.0);
  }
  for (int o = 16; o > 0; o >>= 1) {
    const double h2 = __shfl_down_sync(0xffffffffu, hi, o), l2 = __shfl_down_sync(0xffffffffu, lo, o);
    dd_add(hi, lo, h2, l2);
  }
  if ((threadIdx.x & 31) == 0) { s_red[threadIdx.x >> 5][0] = hi; s_red[threadIdx.x >> 5][1] = lo; }
  __syncthreads();
  if (threadIdx.x == 0) {
    hi = 0.0; lo = 0.0;
    for (int k = 0; k < 8; ++k) dd_add(hi, lo, s_red[k][0], s_red[k][1]);
    out[ab] = 4.0 * 3.14159265358979323846 * dr * (hi + lo);
  }
}

__global__ void begin1d_kernel(DevState* st, double tol) {
  st->tol = tol;
  st->done = 0;
  st->status = 0;
  st->n_done = 0;
}

size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

}  // namespace

struct rism1d_ctx {
  rism1d_params p;
  cudaStream_t stream;
  int ns, M, L, npairs, n_rows;
  size_t field;
  double beta, lam;
  bool lam_set;              // a solve has fixed the charge scale (until then the getters build w with lam = 1)
  Solvent1d sv;
  bool have_solvent, w_valid;
  DevState* state;
  double *Z, *R, *tau, *w, *rows, *chi, *c0;
  cplx *bufA, *bufB, *tab;
  StateHeader* h_hdr;
  SolverParams sp;
  long long launches;
  char err[256];
};

static int fail1(rism1d_ctx* ctx, int code, const char* fmt, ...) {
  if (ctx) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
    va_end(ap);
  }
  return code;
}
#define CU1(call)                                                                                        \
  do {                                                                                                   \
    cudaError_t e_ = (call);                                                                             \
    if (e_ != cudaSuccess) return fail1(ctx, RISM3D_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
  } while (0)

struct DeviceGuard1 {
  int prev = -1;
  bool switched = false;
  bool ok = true;            // false: the context's device could not be made current
  explicit DeviceGuard1(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
    if (prev != dev) {
      switched = (cudaSetDevice(dev) == cudaSuccess);
      ok = switched;
    }
  }
  ~DeviceGuard1() {
    if (switched) cudaSetDevice(prev);
  }
};

static bool valid1(const rism1d_params* p) {
  if (!p) return false;
  if (p->n_sites < 1 || p->n_sites > MAX_S) return false;
  if (p->n_points < 512 || p->n_points > 16384 || (p->n_points & (p->n_points - 1))) return false;
  if (!(p->dr > 0.0) || !(p->temperature > 0.0) || !(p->kappa > 0.0)) return false;
  if (p->closure != RISM3D_KH && p->closure != RISM3D_PSE && p->closure != RISM3D_HNC) return false;
  if (p->closure == RISM3D_PSE && p->pse_order < 1) return false;
  if (p->mdiis_nvec < 1 || p->mdiis_nvec > MAX_M || !(p->mdiis_b > 0.0)) return false;
  return true;
}

static int rows_of(const rism1d_params* p) {
  const size_t field = (size_t)p->n_sites * p->n_sites * p->n_points;
  size_t blocks = (field + R1D_THREADS * 4 - 1) / (R1D_THREADS * 4);
  return (int)(blocks > 256 ? 256 : blocks);
}

static size_t carve1(const rism1d_params* p, char* base, rism1d_ctx* c) {
  const size_t ns = p->n_sites, M = p->n_points, L = 2 * M, np_ = ns * ns, field = np_ * M, Mh = p->mdiis_nvec;
  size_t off = 0;
  auto take = [&](size_t bytes) { char* ptr = base ? base + off : nullptr; off += align256(bytes); return ptr; };
  char* st = take(sizeof(DevState));
  char* Z = take(Mh * field * 8);
  char* R = take(Mh * field * 8);
  char* tau = take(field * 8);
  char* w = take(field * 8);
  char* A = take(np_ * L * 16);
  char* B = take(np_ * L * 16);
  char* tab = take(L * 16);
  char* rows = take((size_t)rows_of(p) * GRAM_SLOT * 16);
  char* chi = take(np_ * M * 8);
  char* c0 = take(np_ * 8);
  if (c) {
    c->state = (DevState*)st; c->Z = (double*)Z; c->R = (double*)R; c->tau = (double*)tau; c->w = (double*)w;
    c->bufA = (cplx*)A; c->bufB = (cplx*)B; c->tab = (cplx*)tab; c->rows = (double*)rows; c->chi = (double*)chi;
    c->c0 = (double*)c0;
  }
  return off;
}

extern "C" size_t rism1d_workspace_bytes(const rism1d_params* p) { return valid1(p) ? carve1(p, nullptr, nullptr) : 0; }

extern "C" const char* rism1d_last_error(const rism1d_ctx* ctx) { return ctx ? ctx->err : "null context"; }
extern "C" long long rism1d_launch_count(const rism1d_ctx* ctx) { return ctx ? ctx->launches : 0; }

extern "C" int rism1d_init(rism1d_ctx** out, const rism1d_params* p, void* d_ws, size_t bytes, void* stream) {
  if (!out || !p || !d_ws) return RISM3D_ERR_ARG;
  *out = nullptr;
  if (!valid1(p)) return RISM3D_ERR_SIZE;
  if (bytes < carve1(p, nullptr, nullptr)) return RISM3D_ERR_WORKSPACE;
  if (((uintptr_t)d_ws) & 255) return RISM3D_ERR_ARG;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || p->device < 0 || ndev <= p->device) return RISM3D_ERR_CUDA;
  DeviceGuard1 guard(p->device);
  if (!guard.ok) return RISM3D_ERR_CUDA;
  rism1d_ctx* ctx = new rism1d_ctx();
  memset(ctx, 0, sizeof(*ctx));
  ctx->p = *p;
  ctx->stream = (cudaStream_t)stream;
  ctx->ns = p->n_sites; ctx->M = p->n_points; ctx->L = 2 * p->n_points; ctx->npairs = p->n_sites * p->n_sites;
  ctx->field = (size_t)ctx->npairs * ctx->M;
  ctx->n_rows = rows_of(p);
  ctx->beta = 1.0 / (K_BOLTZMANN * p->temperature);
  ctx->lam = 1.0;
  ctx->lam_set = false;
  carve1(p, (char*)d_ws, ctx);
  SolverParams& sp = ctx->sp;
  memset(&sp, 0, sizeof(sp));
  sp.closure = p->closure; sp.pse_order = p->closure == RISM3D_PSE ? p->pse_order : 1;
  sp.M = p->mdiis_nvec; sp.b = p->mdiis_b; sp.restart = p->mdiis_restart; sp.accel = RISM3D_ACCEL_MDIIS; sp.dyn_b = false;
  std::vector<double> tab(2 * (size_t)ctx->L);
  for (int a = 0; a < ctx->L; ++a) {
    const long double ang = 2.0L * 3.14159265358979323846264338327950288L * (long double)a / (long double)ctx->L;
    tab[2 * a] = (double)cosl(ang);
    tab[2 * a + 1] = (double)(-sinl(ang));
  }
  cudaError_t e = cudaMallocHost((void**)&ctx->h_hdr, sizeof(StateHeader));
  if (e == cudaSuccess) e = cudaMemcpyAsync(ctx->tab, tab.data(), tab.size() * 8, cudaMemcpyHostToDevice, ctx->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(ctx->state, 0, sizeof(DevState), ctx->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(ctx->tau, 0, ctx->field * 8, ctx->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
  if (e != cudaSuccess) {
    if (ctx->h_hdr) cudaFreeHost(ctx->h_hdr);
    delete ctx;
    return RISM3D_ERR_CUDA;
  }
  *out = ctx;
  return RISM3D_OK;
}

extern "C" void rism1d_destroy(rism1d_ctx* ctx) {
  if (!ctx) return;
  DeviceGuard1 guard(ctx->p.device);
  cudaStreamSynchronize(ctx->stream);
  if (ctx->h_hdr) cudaFreeHost(ctx->h_hdr);
  delete ctx;
}

extern "C" int rism1d_set_solvent(rism1d_ctx* ctx, const double* q, const double* sigma, const double* eps,
                                  const double* rho, const int* species, const double* bond) {
  if (!ctx) return RISM3D_ERR_ARG;
  if (!q || !sigma || !eps || !rho || !species || !bond) return fail1(ctx, RISM3D_ERR_ARG, "bad argument");
  const int ns = ctx->ns;
  // everything is checked on a local copy: a refused call leaves the context's solvent (and its flags) as they were
  Solvent1d sv;
  memset(&sv, 0, sizeof(sv));
  double neutral = 0.0;
  for (int a = 0; a < ns; ++a) {
    if (!isfinite(q[a]) || !isfinite(eps[a]) || !(eps[a] >= 0.0))
      return fail1(ctx, RISM3D_ERR_ARG, "site %d: q and eps must be finite, eps >= 0 (q = %g, eps = %g)", a, q[a], eps[a]);
    if (!isfinite(sigma[a]) || !(sigma[a] > 0.0) || !isfinite(rho[a]) || !(rho[a] > 0.0))
      return fail1(ctx, RISM3D_ERR_ARG, "site %d: sigma and rho must be positive (sigma = %g, rho = %g)", a, sigma[a], rho[a]);
    if (species[a] < 0 || species[a] >= ns) return fail1(ctx, RISM3D_ERR_ARG, "site %d: species %d outside 0..%d", a, species[a], ns - 1);
    neutral += rho[a] * q[a];
  }
  if (fabs(neutral) > 1e-12) return fail1(ctx, RISM3D_ERR_NEUTRAL, "sum rho_a q_a = %.3e", neutral);
  for (int a = 0; a < ns; ++a) {
    sv.q[a] = q[a]; sv.sigma[a] = sigma[a]; sv.eps[a] = eps[a]; sv.rho[a] = rho[a];
    sv.species[a] = species[a];
    for (int b = 0; b < ns; ++b) {
      sv.bond[a][b] = bond[a * ns + b];
      if (a != b && species[a] == species[b] && !(bond[a * ns + b] > 0.0 && isfinite(bond[a * ns + b])))
        return fail1(ctx, RISM3D_ERR_ARG, "sites %d and %d share a species but have no bond length", a, b);
    }
  }
  ctx->sv = sv;
  ctx->have_solvent = true;
  ctx->w_valid = false;
  return RISM3D_OK;
}

// batched FFT of bufA (all pairs); returns the buffer that holds the result
static cplx* fft_all(rism1d_ctx* ctx) {
  cplx *in = ctx->bufA, *out = ctx->bufB;
  const int L = ctx->L, nb = ctx->npairs;
  int Ns = 1;
  while (Ns < L) {
    int R = L / Ns >= 32 ? 32 : L / Ns;
    const int threads = (L / R) * nb;
    const unsigned blocks = (unsigned)((threads + 127) / 128);
    switch (R) {
      case 32: fft1d_pass_kernel<32><<<blocks, 128, 0, ctx->stream>>>(in, out, ctx->tab, L, Ns, nb, ctx->state); break;
      case 16: fft1d_pass_kernel<16><<<blocks, 128, 0, ctx->stream>>>(in, out, ctx->tab, L, Ns, nb, ctx->state); break;
      case 8: fft1d_pass_kernel<8><<<blocks, 128, 0, ctx->stream>>>(in, out, ctx->tab, L, Ns, nb, ctx->state); break;
      case 4: fft1d_pass_kernel<4><<<blocks, 128, 0, ctx->stream>>>(in, out, ctx->tab, L, Ns, nb, ctx->state); break;
      default: fft1d_pass_kernel<2><<<blocks, 128, 0, ctx->stream>>>(in, out, ctx->tab, L, Ns, nb, ctx->state); break;
    }
    ctx->launches += 1;
    Ns *= R;
    cplx* t = in; in = out; out = t;
  }
  return in;
}

static int ensure_w(rism1d_ctx* ctx, double lam) {
  if (ctx->w_valid && lam == ctx->lam) return RISM3D_OK;
  const int n = ctx->npairs * ctx->M;
  setup_w1d_kernel<<<(n + 255) / 256, 256, 0, ctx->stream>>>(ctx->w, ctx->sv, ctx->ns, ctx->M, ctx->p.dr, ctx->beta,
                                                              ctx->p.kappa, lam);
  ctx->launches += 1;
  CU1(cudaGetLastError());
  ctx->lam = lam;
  ctx->lam_set = true;
  ctx->w_valid = true;
  return RISM3D_OK;
}

// closure -> transform -> Eq. 4; zout == nullptr: only chi is wanted
static int forward_half(rism1d_ctx* ctx, bool for_chi) {
  const int n = ctx->npairs * ctx->M;
  closure1d_kernel<<<(n + 255) / 256, 256, 0, ctx->stream>>>(ctx->bufA, ctx->tau, ctx->w, ctx->npairs, ctx->M, ctx->p.dr,
                                                              ctx->sp.closure, ctx->sp.pse_order, ctx->state);
  ctx->launches += 1;
  cplx* spec = fft_all(ctx);
  // the k-space kernel writes the input of the way back into bufA; the spectrum must then not live there
  if (spec == ctx->bufA && !for_chi) {
    CU1(cudaMemcpyAsync(ctx->bufB, ctx->bufA, (size_t)ctx->npairs * ctx->L * 16, cudaMemcpyDeviceToDevice, ctx->stream));
    spec = ctx->bufB;
  }
  kspace1d_kernel<<<(ctx->M - 1 + 63) / 64, 64, 0, ctx->stream>>>(spec, for_chi ? nullptr : ctx->bufA, for_chi ? ctx->chi : nullptr,
                                                                  ctx->sv, ctx->ns, ctx->M, ctx->p.dr, ctx->beta,
                                                                  ctx->p.kappa, ctx->lam, ctx->state);
  ctx->launches += 1;
  CU1(cudaGetLastError());
  return RISM3D_OK;
}

static int read_header1(rism1d_ctx* ctx) {
  CU1(cudaMemcpyAsync(ctx->h_hdr, ctx->state, sizeof(StateHeader), cudaMemcpyDeviceToHost, ctx->stream));
  CU1(cudaStreamSynchronize(ctx->stream));
  return RISM3D_OK;
}

extern "C" int rism1d_solve(rism1d_ctx* ctx, double charge_scale, int max_iter, double tol, int* n_done, double* rms) {
  if (!ctx) return RISM3D_ERR_ARG;
  DeviceGuard1 guard(ctx->p.device);
  if (!guard.ok) return fail1(ctx, RISM3D_ERR_CUDA, "device %d could not be made current", ctx->p.device);
  if (max_iter < 0) return fail1(ctx, RISM3D_ERR_ARG, "max_iter < 0");
  if (!isfinite(charge_scale) || charge_scale < 0.0) return fail1(ctx, RISM3D_ERR_ARG, "charge_scale = %g (must be finite and >= 0)", charge_scale);
  if (!ctx->have_solvent) return fail1(ctx, RISM3D_ERR_ORDER, "set_solvent must come before solve");
  int rc = ensure_w(ctx, charge_scale);
  if (rc) return rc;
  CU1(cudaMemsetAsync(ctx->state, 0, sizeof(DevState), ctx->stream));       // a fresh MDIIS history per call
  begin1d_kernel<<<1, 1, 0, ctx->stream>>>(ctx->state, tol);
  ctx->launches += 1;
  Grid g{};
  g.field = ctx->field;
  Buffers b{};
  b.state = ctx->state; b.Z = ctx->Z; b.R = ctx->R; b.tau = ctx->tau;
  const double n_values = (double)ctx->npairs * (ctx->M - 1);
  for (int it = 0; it < max_iter; ++it) {
    rc = forward_half(ctx, false);
    if (rc) return rc;
    cplx* back = fft_all(ctx);
    residual1d_kernel<<<ctx->n_rows, R1D_THREADS, 0, ctx->stream>>>(back, ctx->tau, ctx->Z, ctx->R, ctx->rows, ctx->ns, ctx->M,
                                                                   ctx->p.dr, ctx->sp.b, ctx->sp.M, ctx->state);
    ctx->launches += 1;
    ctx->launches += launch_gram_solve_rows(ctx->state, ctx->rows, ctx->n_rows, ctx->sp, n_values, ctx->stream);
    ctx->launches += launch_mdiis_update(g, b, ctx->sp, ctx->stream);
    CU1(cudaGetLastError());
    if ((it + 1) % 16 == 0) {
      rc = read_header1(ctx);
      if (rc) return rc;
      if (ctx->h_hdr->done) break;
    }
  }
  rc = read_header1(ctx);
  if (rc) return rc;
  if (n_done) *n_done = ctx->h_hdr->n_done;
  if (rms) *rms = ctx->h_hdr->rms_last;
  if (ctx->h_hdr->status == RISM3D_ERR_DIVERGED)
    return fail1(ctx, RISM3D_ERR_DIVERGED, "non-finite residual after %d iterations", ctx->h_hdr->n_done);
  return RISM3D_OK;
}

extern "C" int rism1d_get_pair(rism1d_ctx* ctx, int which, double* dst) {
  if (!ctx) return RISM3D_ERR_ARG;
  DeviceGuard1 guard(ctx->p.device);
  if (!guard.ok) return fail1(ctx, RISM3D_ERR_CUDA, "device %d could not be made current", ctx->p.device);
  if (!dst || which < 0 || which > 2) return fail1(ctx, RISM3D_ERR_ARG, "bad argument");
  if (!ctx->have_solvent) return fail1(ctx, RISM3D_ERR_ORDER, "set_solvent must come first");
  int rc = ensure_w(ctx, ctx->lam_set ? ctx->lam : 1.0);
  if (rc) return rc;
  const int n = ctx->npairs * (ctx->M - 1);
  double* d = (double*)ctx->bufA;                                          // scratch between iterations
  get_pair1d_kernel<<<(n + 255) / 256, 256, 0, ctx->stream>>>(d, ctx->tau, ctx->w, ctx->npairs, ctx->M, which,
                                                               ctx->sp.closure, ctx->sp.pse_order);
  ctx->launches += 1;
  CU1(cudaGetLastError());
  CU1(cudaMemcpyAsync(dst, d, (size_t)n * 8, cudaMemcpyDeviceToHost, ctx->stream));
  CU1(cudaStreamSynchronize(ctx->stream));
  return RISM3D_OK;
}

extern "C" int rism1d_get_chi(rism1d_ctx* ctx, double* dst) {
  if (!ctx) return RISM3D_ERR_ARG;
  DeviceGuard1 guard(ctx->p.device);
  if (!guard.ok) return fail1(ctx, RISM3D_ERR_CUDA, "device %d could not be made current", ctx->p.device);
  if (!dst) return fail1(ctx, RISM3D_ERR_ARG, "dst is NULL");
  if (!ctx->have_solvent) return fail1(ctx, RISM3D_ERR_ORDER, "set_solvent must come first");
  int rc = ensure_w(ctx, ctx->lam_set ? ctx->lam : 1.0);
  if (rc) return rc;
  CU1(cudaMemsetAsync(&ctx->state->done, 0, sizeof(int), ctx->stream));     // the transform kernels skip a finished solve
  rc = forward_half(ctx, true);
  if (rc) return rc;
  CU1(cudaMemcpyAsync(dst, ctx->chi, (size_t)(ctx->M - 1) * ctx->npairs * 8, cudaMemcpyDeviceToHost, ctx->stream));
  CU1(cudaStreamSynchronize(ctx->stream));
  return RISM3D_OK;
}

extern "C" int rism1d_get_chi_types(rism1d_ctx* ctx, int n_types, const int* site_type, double* dst) {
  if (!ctx) return RISM3D_ERR_ARG;
  if (!site_type || !dst || n_types < 1 || n_types > ctx->ns) return fail1(ctx, RISM3D_ERR_ARG, "bad argument");
  const int ns = ctx->ns, nk = ctx->M - 1;
  int first[MAX_S];
  for (int g = 0; g < n_types; ++g) first[g] = -1;
  for (int a = 0; a < ns; ++a) {
    if (site_type[a] < 0 || site_type[a] >= n_types) return fail1(ctx, RISM3D_ERR_ARG, "site_type[%d] out of range", a);
    if (first[site_type[a]] < 0) first[site_type[a]] = a;
  }
  for (int g = 0; g < n_types; ++g)
    if (first[g] < 0) return fail1(ctx, RISM3D_ERR_ARG, "type %d has no site", g);
  std::vector<double> full((size_t)nk * ns * ns);
  const int rc = rism1d_get_chi(ctx, full.data());
  if (rc) return rc;
  for (int j = 0; j < nk; ++j)
    for (int gp = 0; gp < n_types; ++gp)
      for (int gm = 0; gm < n_types; ++gm) {
        double acc = 0.0;
        for (int a = 0; a < ns; ++a)
          if (site_type[a] == gp) acc += full[((size_t)j * ns + a) * ns + first[gm]];
        dst[((size_t)j * n_types + gp) * n_types + gm] = acc;
      }
  return RISM3D_OK;
}

extern "C" int rism1d_thermo(rism1d_ctx* ctx, double* chi_t, double* pressure, double* c0) {
  if (!ctx) return RISM3D_ERR_ARG;
  DeviceGuard1 guard(ctx->p.device);
  if (!guard.ok) return fail1(ctx, RISM3D_ERR_CUDA, "device %d could not be made current", ctx->p.device);
  if (!ctx->have_solvent) return fail1(ctx, RISM3D_ERR_ORDER, "set_solvent must come first");
  int rc = ensure_w(ctx, ctx->lam_set ? ctx->lam : 1.0);
  if (rc) return rc;
  c_integral1d_kernel<<<ctx->npairs, 256, 0, ctx->stream>>>(ctx->c0, ctx->tau, ctx->w, ctx->M, ctx->p.dr, ctx->sp.closure,
                                                           ctx->sp.pse_order);
  ctx->launches += 1;
  CU1(cudaGetLastError());
  double host[MAX_S * MAX_S];
  CU1(cudaMemcpyAsync(host, ctx->c0, (size_t)ctx->npairs * 8, cudaMemcpyDeviceToHost, ctx->stream));
  CU1(cudaStreamSynchronize(ctx->stream));
  const int ns = ctx->ns;
  double rrc = 0.0;                                     // sum_ab rho_a rho_b int c_ab dr
  for (int a = 0; a < ns; ++a)
    for (int b = 0; b < ns; ++b) rrc += ctx->sv.rho[a] * host[a * ns + b] * ctx->sv.rho[b];
  // species densities and site counts from the per-site arrays
  double rho_sum = 0.0, ideal = 0.0;
  for (int a = 0; a < ns; ++a) {
    bool first = true;
    int count = 0;
    for (int b = 0; b < ns; ++b) {
      if (ctx->sv.species[b] == ctx->sv.species[a]) { ++count; if (b < a) first = false; }
    }
    if (first) { rho_sum += ctx->sv.rho[a]; ideal += ctx->sv.rho[a] * (count + 1); }
  }
  const double kT = 1.0 / ctx->beta;
  if (chi_t) *chi_t = 1.0 / (kT * (rho_sum - rrc));
  if (pressure) *pressure = kT * (0.5 * ideal - 0.5 * rrc);
  if (c0) for (int i = 0; i < ns * ns; ++i) c0[i] = host[i];
  return RISM3D_OK;
}
