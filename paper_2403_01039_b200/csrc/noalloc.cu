// noalloc.cu -- rism3d_noalloc_free_energy (include/rism3d_noalloc.h): the solvation-free-energy sum of Eq. 17-18
// for callers that cannot hand the library a workspace -- a host program whose own pool holds the
// whole GPU, code that must not stall the device with cudaMalloc / cudaFree, an analysis step that was only given the
// fields.  Same integrand, block shape and summation order as free_energy_kernel / free_energy_final_kernel of
// setup_kernels.cu (which stay as they are); the difference is where the per-block partial sums live: in the fixed
// array below instead of the caller's workspace, and the site constants travel in the launch parameters instead of
// device arrays.  This file calls no allocating routine.
#include <stdarg.h>
#include <stdio.h>

#include <mutex>

#include "../../include/rism3d_noalloc.h"
#include "rism3d_internal.h"

using namespace r3d;

namespace {

constexpr int NA_BLOCKS = FE_BLOCKS;                       // as the workspace path: 4 CTAs of 256 threads per SM of a B200
constexpr int NA_THREADS = 256;
constexpr size_t NA_SCRATCH_DOUBLES = (size_t)2 * NA_BLOCKS * RISM3D_NOALLOC_MAX_SITES * 2;   // [sum][block][site][hi, lo]
static_assert(NA_SCRATCH_DOUBLES * sizeof(double) == RISM3D_NOALLOC_SCRATCH_BYTES, "header and array disagree");
static_assert(RISM3D_NOALLOC_MAX_SITES == MAX_NV, "slot layout follows MAX_NV");

// The scratch.  One copy per GPU that loads this library, resident until the process exits.  In HOST code this name is
// only a handle for cudaGetSymbolAddress -- it is not a device address and must never be passed to a kernel as one; the
// kernels below get the pointer that scratch_of() looked up.
static __device__ __align__(256) double g_noalloc_scratch[NA_SCRATCH_DOUBLES];

constexpr int NA_MAX_DEVICES = 64;
std::mutex g_setup_mutex;
double* g_scratch_ptr[NA_MAX_DEVICES];                     // device address of g_noalloc_scratch on each GPU, once known

struct SiteConstants {                                     // by value in the launch parameters: no device table needed
  double q[RISM3D_NOALLOC_MAX_SITES];
  double rho[RISM3D_NOALLOC_MAX_SITES];
};

int na_fail(char* err, size_t cap, int code, const char* fmt, ...) {
  if (err && cap) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(err, cap, fmt, ap);
    va_end(ap);
  }
  return code;
}

// Device address of the scratch array on `device`, which must be the current device.  The first call per device asks the
// runtime (this may load the module's device code: do it at start-up, outside stream capture); later calls read the cache.
cudaError_t scratch_of(int device, double** out) {
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  if (g_scratch_ptr[device] == nullptr) {
    double* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    if (p == nullptr) return cudaErrorInvalidSymbol;
    g_scratch_ptr[device] = p;
  }
  *out = g_scratch_ptr[device];
  return cudaSuccess;
}

struct CurrentDevice {                                     // make `dev` current, put the caller's device back on exit
  int prev = -1;
  cudaError_t status = cudaSuccess;
  explicit CurrentDevice(int dev) {
    status = cudaGetDevice(&prev);
    if (status == cudaSuccess && prev != dev) status = cudaSetDevice(dev);
  }
  ~CurrentDevice() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};

// Per-block partial sums of the integrand of Eq. 17/18 and of c_sr alone, every site type in turn.  Block b writes
// part[(b * MAX + g) * 2 .. +1] (integrand) and part[((nblocks + b) * MAX + g) * 2 .. +1] (c_sr) for every g < nv: all
// the slots the final kernel reads are rewritten by every call, so the array's old contents never matter.
__global__ void __launch_bounds__(NA_THREADS)
    noalloc_free_energy_kernel(double* __restrict__ part, const double* __restrict__ tau, const double* __restrict__ w,
                               const double* __restrict__ phi, SiteConstants sc, int nv, size_t npts, int closure,
                               int order) {
  __shared__ double s_red[NA_THREADS / 32][4];
  double inv_fact = 1.0;
  for (int i = 2; i <= order + 1; ++i) inv_fact /= (double)i;
  for (int g = 0; g < nv; ++g) {
    double hi = 0.0, lo = 0.0, chi_ = 0.0, clo = 0.0;
    const double q = sc.q[g];
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
      for (int k = 0; k < NA_THREADS / 32; ++k) {
        dd_add(hi, lo, s_red[k][0], s_red[k][1]);
        dd_add(chi_, clo, s_red[k][2], s_red[k][3]);
      }
      part[((size_t)blockIdx.x * RISM3D_NOALLOC_MAX_SITES + g) * 2 + 0] = hi;
      part[((size_t)blockIdx.x * RISM3D_NOALLOC_MAX_SITES + g) * 2 + 1] = lo;
      part[((size_t)(gridDim.x + blockIdx.x) * RISM3D_NOALLOC_MAX_SITES + g) * 2 + 0] = chi_;
      part[((size_t)(gridDim.x + blockIdx.x) * RISM3D_NOALLOC_MAX_SITES + g) * 2 + 1] = clo;
    }
  }
}

// One warp per (sum, site type): the block partials in a fixed order.  out[g] = kT dV rho_g * integrand sum,
// out[nv + g] = dV * c_sr sum.
__global__ void __launch_bounds__(64 * RISM3D_NOALLOC_MAX_SITES)
    noalloc_free_energy_final_kernel(double* __restrict__ out, const double* __restrict__ part, int nblocks,
                                     SiteConstants sc, int nv, double scale, double dv) {
  const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int g = wid % RISM3D_NOALLOC_MAX_SITES, second = wid / RISM3D_NOALLOC_MAX_SITES;
  if (g >= nv) return;
  double hi, lo;
  warp_sum_partials(part + ((size_t)second * nblocks * RISM3D_NOALLOC_MAX_SITES + g) * 2, nblocks, lane, hi, lo,
                    RISM3D_NOALLOC_MAX_SITES);
  if (lane == 0) out[second * nv + g] = second ? dv * (hi + lo) : scale * sc.rho[g] * (hi + lo);
}

}  // namespace

extern "C" int rism3d_noalloc_free_energy(int device, void* cuda_stream, size_t n_points, double spacing, int n_sites,
                                          int closure, int pse_order, double temperature, const double* q,
                                          const double* rho, const double* d_tau, const double* d_w,
                                          const double* d_phi, double* d_out, char* err, size_t err_cap) {
  if (err && err_cap) err[0] = '\0';
  if (!q || !rho || !d_tau || !d_w || !d_phi || !d_out)
    return na_fail(err, err_cap, RISM3D_ERR_ARG, "rism3d_noalloc_free_energy: NULL pointer among q, rho, d_tau, d_w, d_phi, d_out");
  if (closure != RISM3D_KH && closure != RISM3D_PSE && closure != RISM3D_HNC)
    return na_fail(err, err_cap, RISM3D_ERR_ARG, "rism3d_noalloc_free_energy: unknown closure %d", closure);
  if (n_sites < 1 || n_sites > RISM3D_NOALLOC_MAX_SITES)
    return na_fail(err, err_cap, RISM3D_ERR_SIZE,
                   "rism3d_noalloc_free_energy: n_sites = %d, but the fixed scratch array has slots for 1..%d site types "
                   "(use rism3d_free_energy with a workspace for more)", n_sites, RISM3D_NOALLOC_MAX_SITES);
  if (n_points < 1 || n_points > (size_t)RISM3D_NOALLOC_MAX_POINTS)
    return na_fail(err, err_cap, RISM3D_ERR_SIZE,
                   "rism3d_noalloc_free_energy: n_points = %zu is outside 1..%d (512^3, the largest grid of the library)",
                   n_points, RISM3D_NOALLOC_MAX_POINTS);
  if (!(spacing > 0.0) || !(temperature > 0.0) || (closure == RISM3D_PSE && pse_order < 1))
    return na_fail(err, err_cap, RISM3D_ERR_SIZE,
                   "rism3d_noalloc_free_energy: spacing, temperature and pse_order must be positive");
  int n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev < 1)
    return na_fail(err, err_cap, RISM3D_ERR_CUDA, "rism3d_noalloc_free_energy: no CUDA device (there is no CPU fallback)");
  if (device < 0 || device >= n_dev || device >= NA_MAX_DEVICES)
    return na_fail(err, err_cap, RISM3D_ERR_ARG, "rism3d_noalloc_free_energy: device %d does not exist (%d devices)", device, n_dev);

  CurrentDevice on(device);
  if (on.status != cudaSuccess)
    return na_fail(err, err_cap, RISM3D_ERR_CUDA, "rism3d_noalloc_free_energy: cudaSetDevice(%d): %s", device,
                   cudaGetErrorString(on.status));
  double* d_scratch = nullptr;
  cudaError_t e = scratch_of(device, &d_scratch);
  if (e != cudaSuccess)
    return na_fail(err, err_cap, RISM3D_ERR_CUDA, "rism3d_noalloc_free_energy: cudaGetSymbolAddress(scratch) on device %d: %s",
                   device, cudaGetErrorString(e));

  SiteConstants sc;
  for (int g = 0; g < RISM3D_NOALLOC_MAX_SITES; ++g) {
    sc.q[g] = g < n_sites ? q[g] : 0.0;
    sc.rho[g] = g < n_sites ? rho[g] : 0.0;
  }
  const int order = closure == RISM3D_PSE ? pse_order : 1;
  const double dv = spacing * spacing * spacing;
  const double kT = K_BOLTZMANN * temperature;               // the products below in the order rism3d_free_energy forms them
  cudaStream_t s = (cudaStream_t)cuda_stream;
  noalloc_free_energy_kernel<<<NA_BLOCKS, NA_THREADS, 0, s>>>(d_scratch, d_tau, d_w, d_phi, sc, n_sites, n_points,
                                                              closure, order);
  noalloc_free_energy_final_kernel<<<1, 64 * RISM3D_NOALLOC_MAX_SITES, 0, s>>>(d_out, d_scratch, NA_BLOCKS, sc, n_sites,
                                                                               kT * spacing * spacing * spacing, dv);
  e = cudaGetLastError();
  if (e != cudaSuccess)
    return na_fail(err, err_cap, RISM3D_ERR_CUDA, "rism3d_noalloc_free_energy: launch: %s", cudaGetErrorString(e));
  return RISM3D_OK;
}
