// mdiis_kernels.cu -- step 6 of the loop (Q7, Q8): MDIIS with M stored
// (input, residual) pairs.  R_i = Y_i - X_i; c = argmin |sum c_i R_i|^2 with sum c_i = 1 (Lagrange multiplier);
// X_new = sum_i c_i (X_i + b R_i).
//
// The history stores Z_i = X_i + b R_i (written by zinv_residual next to R_i) instead of X_i: Eq. 40 needs X_i
// in no other form, and the update then reads M fields instead of 2M.  The current input lives in its own field.
//
//   gram_row_kernel     : streaming pass over the new residual and the stored ones: per-CTA double-double partial
//                         sums of <R_new, R_new> and <R_new, R_i>.  The CTA that finishes last (ticket counter)
//                         adds the partials in a fixed order, then does rms and the convergence test (Eq. 41 as
//                         read in Q9), the history bookkeeping (circular overwrite, restart rule), the bordered
//                         (m+1)x(m+1) solve by Gaussian elimination with partial pivoting, and picks the slot the
//                         next pair goes to.
//   mdiis_update_kernel : streaming linear combination tau = sum_i c_i Z_i over the stored slots.
#include "rism3d_internal.h"

namespace r3d {

// History bookkeeping and the small solve, run by ONE thread (the last gram_row CTA) once the Gram row s_row
// (entries 0..nother-1: <R_new, R_other[j]>, entry nother: <R_new, R_new>) is complete.
__device__ void mdiis_bookkeeping_and_solve(DevState* __restrict__ st, const double* s_row, int m_old, int nother,
                                            int M, double restart, double npts_total) {
  const int skip = (m_old == M) ? 1 : 0;
  const double self = s_row[nother];
  const double rms = sqrt(self / npts_total);          // Eq. 41 (Q9)
  st->rms_last = rms;
  st->n_done += 1;
  st->rms_hist[st->hist_n % RMS_HIST_CAP] = rms;
  st->hist_n += 1;
  st->upd_m = 0;
  if (!isfinite(rms)) { st->done = 1; st->status = RISM3D_ERR_DIVERGED; return; }
  if (st->tol > 0.0 && rms < st->tol) { st->done = 1; return; }   // converged: tau stays as it is

  // append (cur, R_new) to the history, dropping the oldest entry of a full history
  int m = m_old;
  if (skip) {
    for (int i = 0; i + 1 < m; ++i) {
      st->list[i] = st->list[i + 1];
      st->rms[i] = st->rms[i + 1];
      for (int j = 0; j + 1 < m; ++j) st->S[i][j] = st->S[i + 1][j + 1];
    }
    m -= 1;
  }
  const int cur = st->cur;
  st->list[m] = cur;
  st->rms[m] = rms;
  for (int i = 0; i < m; ++i) st->S[m][i] = st->S[i][m] = s_row[i];
  st->S[m][m] = self;
  m += 1;

  // restart rule (Q8): keep only the entry with the smallest rms (first minimum)
  if (restart > 0.0) {
    double rmin = st->rms[0];
    int best = 0;
    for (int i = 1; i < m; ++i)
      if (st->rms[i] < rmin) { rmin = st->rms[i]; best = i; }
    if (rms > restart * rmin) {
      st->list[0] = st->list[best];
      st->rms[0] = st->rms[best];
      st->S[0][0] = st->S[best][best];
      m = 1;
    }
  }
  st->m = m;

  // bordered system [[S/smax, 1], [1^T, 0]] [c; lambda] = [0; 1]; every product and difference is rounded
  // separately (no FMA contraction) so the elimination takes the same steps as the oracle's
  double c[MAX_M];
  for (int i = 0; i < m; ++i) c[i] = (i == m - 1) ? 1.0 : 0.0;     // fallback: unit vector on the newest entry
  double smax = st->S[0][0];
  for (int i = 1; i < m; ++i) smax = fmax(smax, st->S[i][i]);
  if (smax > 0.0) {
    const int n = m + 1;
    double A[MAX_M + 1][MAX_M + 2];
    for (int i = 0; i < n; ++i)
      for (int j = 0; j <= n; ++j) A[i][j] = 0.0;
    for (int i = 0; i < m; ++i) {
      for (int j = 0; j < m; ++j) A[i][j] = st->S[i][j] / smax;
      A[i][m] = 1.0;
      A[m][i] = 1.0;
    }
    A[m][n] = 1.0;
    bool ok = true;
    for (int colx = 0; colx < n && ok; ++colx) {
      int piv = colx;
      for (int r = colx + 1; r < n; ++r)
        if (fabs(A[r][colx]) > fabs(A[piv][colx])) piv = r;
      if (A[piv][colx] == 0.0) { ok = false; break; }
      if (piv != colx)
        for (int j = 0; j <= n; ++j) { const double tmp = A[colx][j]; A[colx][j] = A[piv][j]; A[piv][j] = tmp; }
      for (int r = colx + 1; r < n; ++r) {
        const double fac = A[r][colx] / A[colx][colx];
        for (int j = colx; j <= n; ++j) A[r][j] = __dsub_rn(A[r][j], __dmul_rn(fac, A[colx][j]));
      }
    }
    if (ok) {
      double xs[MAX_M + 1];
      for (int r = n - 1; r >= 0; --r) {
        double acc = A[r][n];
        for (int j = r + 1; j < n; ++j) acc = __dsub_rn(acc, __dmul_rn(A[r][j], xs[j]));
        xs[r] = acc / A[r][r];
      }
      for (int i = 0; i < m; ++i) c[i] = xs[i];
    }
  }

  // slot of the NEXT (Z, R) pair: a full history reuses the slot of its oldest entry (dropped next iteration,
  // and not read by the Gram row of that iteration), otherwise the first unused slot
  int nxt;
  if (m == M) {
    nxt = st->list[0];
  } else {
    unsigned used = 0;
    for (int i = 0; i < m; ++i) used |= 1u << st->list[i];
    nxt = 0;
    while (used & (1u << nxt)) ++nxt;
  }
  st->upd_m = m;
  for (int i = 0; i < m; ++i) { st->upd_list[i] = st->list[i]; st->upd_coef[i] = c[i]; }
  st->cur = nxt;
}

// Gram row.  One CTA = GRAM_THREADS * GRAM_EPT consecutive double2 of every field; each thread accumulates its
// 2 * GRAM_EPT elements per entry in plain fp64 FMAs, the per-thread sums are then combined in double-double (warp
// shuffles, fixed order) into one partial per CTA and entry; mdiis_solve adds the partials of all CTAs in
// double-double, again in a fixed order.  Entry j < nother: <R_new, R_other[j]>;
// entry MAX_M: <R_new, R_new>.  MAXO = M - 1 bounds nother at compile time.
constexpr int GRAM_THREADS = 256;
constexpr int GRAM_EPT = 16;

template <int MAXO>
__global__ void __launch_bounds__(GRAM_THREADS)
    gram_row_kernel(DevState* __restrict__ st, const double* __restrict__ R, double* __restrict__ gram_part,
                    size_t field, int M, double restart) {
  if (st->done) return;
  __shared__ int s_other[MAX_M];
  __shared__ int s_nother, s_cur, s_m;
  __shared__ bool s_last;
  __shared__ double s_row[MAX_M + 1];
  __shared__ double s_part[(MAX_M + 1) * (GRAM_THREADS / 32) * 2];
  const int tid = threadIdx.x;
  if (tid == 0) {
    const int m = st->m;
    const int skip = (m == M) ? 1 : 0;                 // a full history drops its oldest entry this iteration
    s_nother = m - skip;
    s_m = m;
    s_cur = st->cur;
    for (int i = 0; i < m - skip; ++i) s_other[i] = st->list[i + skip];
  }
  __syncthreads();
  const int nother = s_nother;
  const size_t n2 = field / 2;
  const double2* Rn = reinterpret_cast<const double2*>(R + (size_t)s_cur * field);
  const double2* Ro[MAXO > 0 ? MAXO : 1];
#pragma unroll
  for (int j = 0; j < MAXO; ++j)
    Ro[j] = reinterpret_cast<const double2*>(R + (size_t)s_other[j < nother ? j : 0] * field);
  double acc[MAXO + 1];
#pragma unroll
  for (int j = 0; j <= MAXO; ++j) acc[j] = 0.0;
  const size_t base = (size_t)blockIdx.x * (GRAM_THREADS * GRAM_EPT) + tid;
#pragma unroll 2
  for (int it = 0; it < GRAM_EPT; ++it) {
    const size_t i = base + (size_t)it * GRAM_THREADS;
    if (i < n2) {
      const double2 r = __ldcs(Rn + i);
      acc[MAXO] = fma(r.x, r.x, fma(r.y, r.y, acc[MAXO]));
#pragma unroll
      for (int j = 0; j < MAXO; ++j)
        if (j < nother) {
          const double2 q = __ldcs(Ro[j] + i);
          acc[j] = fma(r.x, q.x, fma(r.y, q.y, acc[j]));
        }
    }
  }
  // warp level: double-double butterfly-free tree in a fixed order, then one thread per entry adds the warps
  const int lane = tid & 31, wid = tid >> 5;
#pragma unroll
  for (int j = 0; j <= MAXO; ++j) {
    if (j < nother || j == MAXO) {
      double hi = acc[j], lo = 0.0;
      for (int o = 16; o > 0; o >>= 1) {
        const double h2 = __shfl_down_sync(0xffffffffu, hi, o), l2 = __shfl_down_sync(0xffffffffu, lo, o);
        dd_add(hi, lo, h2, l2);
      }
      if (lane == 0) {
        s_part[(j * (GRAM_THREADS / 32) + wid) * 2] = hi;
        s_part[(j * (GRAM_THREADS / 32) + wid) * 2 + 1] = lo;
      }
    }
  }
  __syncthreads();
  if (tid <= MAXO && (tid < nother || tid == MAXO)) {
    double hi = 0.0, lo = 0.0;
    for (int w = 0; w < GRAM_THREADS / 32; ++w)
      dd_add(hi, lo, s_part[(tid * (GRAM_THREADS / 32) + w) * 2], s_part[(tid * (GRAM_THREADS / 32) + w) * 2 + 1]);
    dd_norm(hi, lo);
    const int j = (tid == MAXO) ? MAX_M : tid;
    *reinterpret_cast<double2*>(gram_part + ((size_t)j * gridDim.x + blockIdx.x) * 2) = make_double2(hi, lo);
    __threadfence();                                   // the partial is visible before this CTA takes its ticket
  }
  __syncthreads();
  if (tid == 0) {
    const unsigned t = atomicAdd(&st->ticket, 1u);
    s_last = (t == gridDim.x - 1);
  }
  __syncthreads();
  if (!s_last) return;

  // The CTA that finishes last adds the partials of all CTAs, entry by entry, in double-double and in a fixed order
  // (thread i takes partials i, i + 256, ...; then the warp tree and the 8 warps in order), then one thread does the
  // bookkeeping and the small solve.  Which CTA is last does not affect any value.
  __threadfence();
  const int nblk = (int)gridDim.x;
  for (int jj = 0; jj <= nother; ++jj) {
    const int j = (jj == nother) ? MAX_M : jj;
    double hi = 0.0, lo = 0.0;
    const double2* part = reinterpret_cast<const double2*>(gram_part) + (size_t)j * nblk;
    for (int blk = tid; blk < nblk; blk += GRAM_THREADS) {
      const double2 p = __ldcg(part + blk);
      dd_add(hi, lo, p.x, p.y);
    }
    for (int o = 16; o > 0; o >>= 1) {
      const double h2 = __shfl_down_sync(0xffffffffu, hi, o), l2 = __shfl_down_sync(0xffffffffu, lo, o);
      dd_add(hi, lo, h2, l2);
    }
    if (lane == 0) {
      s_part[(jj * (GRAM_THREADS / 32) + wid) * 2] = hi;
      s_part[(jj * (GRAM_THREADS / 32) + wid) * 2 + 1] = lo;
    }
  }
  __syncthreads();
  if (tid <= nother) {
    double hi = 0.0, lo = 0.0;
    for (int w = 0; w < GRAM_THREADS / 32; ++w)
      dd_add(hi, lo, s_part[(tid * (GRAM_THREADS / 32) + w) * 2], s_part[(tid * (GRAM_THREADS / 32) + w) * 2 + 1]);
    s_row[tid] = hi + lo;
  }
  __syncthreads();
  if (tid != 0) return;
  st->ticket = 0;
  mdiis_bookkeeping_and_solve(st, s_row, s_m, nother, M, restart, (double)field);
}

int gram_blocks(const Grid& g) {
  const size_t per = (size_t)GRAM_THREADS * GRAM_EPT;
  return (int)((g.field / 2 + per - 1) / per);
}
int gram_blocks_for(int n, int nv) {
  Grid g{};
  g.n = n;
  g.nv = nv;
  g.field = (size_t)n * n * n * nv;
  return gram_blocks(g);
}

int launch_gram_row(const Grid& g, const Buffers& b, const SolverParams& sp, cudaStream_t s) {
  const unsigned blocks = (unsigned)gram_blocks(g);
#define R3D_GRAM(MO) case MO + 1: gram_row_kernel<MO><<<blocks, GRAM_THREADS, 0, s>>>(b.state, b.R, b.gram_part, g.field, sp.M, sp.restart); break
  switch (sp.M) {
    R3D_GRAM(0); R3D_GRAM(1); R3D_GRAM(2); R3D_GRAM(3); R3D_GRAM(4); R3D_GRAM(5); R3D_GRAM(6); R3D_GRAM(7);
    R3D_GRAM(8); R3D_GRAM(9); R3D_GRAM(10); R3D_GRAM(11); R3D_GRAM(12); R3D_GRAM(13); R3D_GRAM(14); R3D_GRAM(15);
    default: return 0;
  }
#undef R3D_GRAM
  return 1;
}

// tau = sum_i c_i Z_i over the stored entries, Z_i = X_i + b R_i (Eq. 40 as read in Q7); products and sums are
// rounded one by one, in the order of the oracle's loop.
__global__ void __launch_bounds__(256)
    mdiis_update_kernel(const DevState* __restrict__ st, const double* __restrict__ Z, double* __restrict__ tau,
                        size_t field) {
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
  double2* dst = reinterpret_cast<double2*>(tau);
  const size_t n2 = field / 2;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n2; i += (size_t)gridDim.x * blockDim.x) {
    double2 acc = make_double2(0.0, 0.0);
#pragma unroll 4
    for (int k = 0; k < m; ++k) {
      const double2 zv = __ldcs(reinterpret_cast<const double2*>(Z + (size_t)s_list[k] * field) + i);
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
  mdiis_update_kernel<<<(unsigned)blocks, 256, 0, s>>>(b.state, b.Z, b.tau, g.field);
  clear_pending_update_kernel<<<1, 1, 0, s>>>(b.state);
  return 2;
}

}  // namespace r3d
