// mdiis_kernels.cu -- step 6 of the loop (Q7, Q8): MDIIS with M stored
// (input, residual) pairs.  R_i = Y_i - X_i; c = argmin |sum c_i R_i|^2 with sum c_i = 1 (Lagrange multiplier);
// X_new = sum_i c_i (X_i + b R_i).
//
// The history stores Z_i = X_i + b R_i (written by zinv_residual next to R_i) instead of X_i: Eq. 40 needs X_i
// in no other form, and the update then reads M fields instead of 2M.  The current input lives in its own field.
//
// The Gram row, the rms / convergence test, the history bookkeeping and the bordered solve ride on zinv_residual
// (fft_kernels.cu + mdiis_device.cuh); the update rides on the next closure_zfwd.  What is left here:
//   mdiis_update_kernel : streaming linear combination tau = sum_i c_i Z_i over the stored slots, launched once at
//                         the end of rism3d_iterate, when no closure pass follows.
#include "rism3d_internal.h"

namespace r3d {

// tau = sum_i c_i Z_i over the stored entries, Z_i = X_i + b R_i (Eq. 40 as read in Q7); products and sums are
// rounded one by one, in the order of the oracle's loop.
template <bool DYN>
__global__ void __launch_bounds__(256)
    mdiis_update_kernel(const DevState* __restrict__ st, const double* __restrict__ Z, const double* __restrict__ Rh,
                        double* __restrict__ tau, size_t field) {
  if (st->done) return;
  __shared__ int s_list[MAX_M];
  __shared__ double s_c[MAX_M];
  __shared__ int s_m;
  if (threadIdx.x == 0) {
    s_m = st->upd_m;
    for (int i = 0; i < st->upd_m; ++i) { s_list[i] = st->upd_list[i]; s_c[i] = st->upd_coef[i]; }
  }
  __syncthreads();
  const int m = s_m;
  if (m == 0) return;
  const double bdyn = st->b_dyn;
  double2* dst = reinterpret_cast<double2*>(tau);
  const size_t n2 = field / 2;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n2; i += (size_t)gridDim.x * blockDim.x) {
    double2 acc = make_double2(0.0, 0.0);
#pragma unroll 4
    for (int k = 0; k < m; ++k) {
      double2 zv = __ldcs(reinterpret_cast<const double2*>(Z + (size_t)s_list[k] * field) + i);
      if constexpr (DYN) {                             // X_i + b R_i with the current b (dynamic damping)
        const double2 rv = __ldcs(reinterpret_cast<const double2*>(Rh + (size_t)s_list[k] * field) + i);
        zv = make_double2(__dadd_rn(zv.x, __dmul_rn(bdyn, rv.x)), __dadd_rn(zv.y, __dmul_rn(bdyn, rv.y)));
      }
      const double ck = s_c[k];
      acc.x = __dadd_rn(acc.x, __dmul_rn(ck, zv.x));
      acc.y = __dadd_rn(acc.y, __dmul_rn(ck, zv.y));
    }
    dst[i] = acc;
  }
}

__global__ void clear_pending_update_kernel(DevState* st) { st->upd_m = 0; }

int launch_mdiis_update(const Grid& g, const Buffers& b, const SolverParams& sp, cudaStream_t s) {
  const size_t n2 = g.field / 2;
  size_t blocks = (n2 + 255) / 256;
  const size_t cap = 148 * 8 * 4;
  if (blocks > cap) blocks = cap;
  if (sp.dyn_b) mdiis_update_kernel<true><<<(unsigned)blocks, 256, 0, s>>>(b.state, b.Z, b.R, b.tau, g.field);
  else mdiis_update_kernel<false><<<(unsigned)blocks, 256, 0, s>>>(b.state, b.Z, b.R, b.tau, g.field);
  clear_pending_update_kernel<<<1, 1, 0, s>>>(b.state);
  return 2;
}

}  // namespace r3d
