// mdiis_device.cuh -- device-side pieces of the MDIIS step shared by the kernels that finish a Gram row
// (Q7, Q8): the block-level double-double reduction of per-thread partial sums, the
// two-level, fixed-order reduction of the per-CTA partials by "last arriver" CTAs (ticket counters), and the
// history bookkeeping + bordered solve run by one thread at the very end.
#pragma once
#include "rism3d_internal.h"

namespace r3d {

constexpr int GRAM_GROUP = 64;       // CTAs per first-level group of the partial-sum reduction

// History bookkeeping and the small solve, run by ONE thread (the last gram_row CTA) once the Gram row s_row
// (entries 0..nother-1: <R_new, R_other[j]>, entry nother: <R_new, R_new>) is complete.
// accelerator settings handed to the kernels that finish a Gram row
struct AccelArgs {
  int M;                 // stored pairs (modified Anderson: 3 = the newest + two histories)
  double restart;        // MDIIS restart factor (<= 0: never)
  int accel;             // rism3d_accelerator
  double s1, s2;         // tuning parameters of Eq. 34-35
};

static __device__ __noinline__ void mdiis_bookkeeping_and_solve(DevState* __restrict__ st, const double* s_row, int m_old,
                                                                int nother, AccelArgs aa, double self_unweighted,
                                                                double npts_total) {
  const int M = aa.M;
  const double restart = aa.restart;
  const int skip = (m_old == M) ? 1 : 0;
  const double self = s_row[nother];
  const double rms = sqrt(self_unweighted / npts_total);   // Eq. 41 (Q9): always the unweighted sum
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
  if (aa.accel == RISM3D_ACCEL_ANDERSON) {
    // Modified Anderson, two histories (Eq. 34-39).  Entries: newest = m-1 (R0), m-2 (R1), m-3 (R2).  theta from the
    // normal equations of min |R0 - sum_j theta_j dR_j|^2, dR_j = R0 - Rj (Eq. 36); with a_i = theta_i + s_i,
    //   X_new = u + b (v - u) = (1 - a1 - a2)(X0 + b R0) + a1 (X1 + b R1) + a2 (X2 + b R2) = sum_k c_k Z_k.
    // Picard steps (unit vector on the newest Z) until two histories exist.
    if (m == 3) {
      const double s00 = st->S[2][2], s01 = st->S[2][1], s02 = st->S[2][0], s11 = st->S[1][1], s12 = st->S[1][0],
                   s22 = st->S[0][0];
      double a11 = s00 - s01 - s01 + s11, a12 = s00 - s01 - s02 + s12, a22 = s00 - s02 - s02 + s22;
      double r1 = s00 - s01, r2 = s00 - s02;
      const double amax = fmax(a11, a22);
      double th1 = 0.0, th2 = 0.0;
      if (amax > 0.0) {
        a11 /= amax; a12 /= amax; a22 /= amax; r1 /= amax; r2 /= amax;
        // Cramer's rule, products and differences rounded separately (as the oracle's Python expression)
        const double det = __dsub_rn(__dmul_rn(a11, a22), __dmul_rn(a12, a12));
        if (det != 0.0) {
          th1 = __dsub_rn(__dmul_rn(r1, a22), __dmul_rn(a12, r2)) / det;
          th2 = __dsub_rn(__dmul_rn(a11, r2), __dmul_rn(r1, a12)) / det;
        }
      }
      const double a1 = th1 + aa.s1, a2 = th2 + aa.s2;
      c[2] = 1.0 - a1 - a2;
      c[1] = a1;
      c[0] = a2;
    }
  } else if (smax > 0.0) {
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

// Sum of `count` double-double partials part[0..count) by ONE warp, in a fixed order: lane l adds l, l + 32, ...,
// then the shuffle tree.  Result (hi, lo) in lane 0.
static __device__ __forceinline__ void warp_sum_partials(const double* part, int count, int lane, double& hi, double& lo) {
  hi = 0.0;
  lo = 0.0;
  for (int i = lane; i < count; i += 32) {
    const double2 p = __ldcg(reinterpret_cast<const double2*>(part) + i);
    dd_add(hi, lo, p.x, p.y);
  }
  for (int o = 16; o > 0; o >>= 1) {
    const double h2 = __shfl_down_sync(0xffffffffu, hi, o), l2 = __shfl_down_sync(0xffffffffu, lo, o);
    dd_add(hi, lo, h2, l2);
  }
}

// Called by ALL threads of every CTA of a kernel that has just written its per-CTA partials
//   part1[(j * nblk + blockIdx.x)]  (double-double, j = 0..nother-1 and j = MAX_M for <R_new, R_new>)
// with a __threadfence() after the writes.  Level 1: the last CTA of each group of GRAM_GROUP consecutive CTAs adds
// the group's partials into part2[(j * ngroups + group)].  Level 2: the last such group adder adds the group sums,
// then one thread runs the bookkeeping and the small solve.  Every sum runs in a fixed order, so the result does not
// depend on which CTA arrives last.  tickets: [ngroups] counters, zero on entry, zero again on exit.
template <int NT>
static __device__ __forceinline__ void gram_finish(DevState* __restrict__ st, double* __restrict__ part1,
                                                   double* __restrict__ part2, unsigned* __restrict__ tickets,
                                                   int m_old, int nother, AccelArgs aa, bool weighted,
                                                   double npts_total, double* s_row /* shared, MAX_M + 2 */,
                                                   int* s_flag /* shared */) {
  // entries: jj < nother: <R_new, R_other[jj]> (slot jj); jj = nother: <R_new, R_new> (slot MAX_M); and, when the
  // inner product is weighted, jj = nother + 1: the unweighted <R_new, R_new> for the rms (slot MAX_M - 1, free
  // because a weighted run stores at most 3 pairs)
  const int nent = nother + (weighted ? 2 : 1);
  auto slot = [&](int jj) { return jj < nother ? jj : (jj == nother ? MAX_M : MAX_M - 1); };
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  constexpr int NW = NT / 32;
  const int nblk = (int)gridDim.x, ngroups = (nblk + GRAM_GROUP - 1) / GRAM_GROUP;
  const int grp = (int)blockIdx.x / GRAM_GROUP;
  const int gsize = min(GRAM_GROUP, nblk - grp * GRAM_GROUP);
  __syncthreads();                                     // all partial writes (and their fences) of this CTA are done
  if (tid == 0) *s_flag = (atomicAdd(&tickets[grp], 1u) == (unsigned)(gsize - 1));
  __syncthreads();
  if (!*s_flag) return;
  __threadfence();
  for (int jj = wid; jj < nent; jj += NW) {            // level 1: this group's partials, one warp per entry
    const int j = slot(jj);
    double hi, lo;
    warp_sum_partials(part1 + ((size_t)j * nblk + (size_t)grp * GRAM_GROUP) * 2, gsize, lane, hi, lo);
    if (lane == 0) {
      dd_norm(hi, lo);
      *reinterpret_cast<double2*>(part2 + ((size_t)j * ngroups + grp) * 2) = make_double2(hi, lo);
      __threadfence();
    }
  }
  __syncthreads();
  if (tid == 0) {
    tickets[grp] = 0;
    *s_flag = (atomicAdd(&st->ticket, 1u) == (unsigned)(ngroups - 1));
  }
  __syncthreads();
  if (!*s_flag) return;
  __threadfence();
  for (int jj = wid; jj < nent; jj += NW) {            // level 2: the group sums
    const int j = slot(jj);
    double hi, lo;
    warp_sum_partials(part2 + (size_t)j * ngroups * 2, ngroups, lane, hi, lo);
    if (lane == 0) s_row[jj] = hi + lo;
  }
  __syncthreads();
  if (tid != 0) return;
  st->ticket = 0;
  mdiis_bookkeeping_and_solve(st, s_row, m_old, nother, aa, weighted ? s_row[nother + 1] : s_row[nother], npts_total);
}

}  // namespace r3d
