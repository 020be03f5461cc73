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
  double b_min, b_max;   // b_max > 0: dynamic damping b = clamp(-0.2 log10 rms, b_min, b_max) (Q18)
};

// shared-memory scratch of the final step (one per CTA; only the last-arriving CTA uses it)
struct SolveScratch {
  double S[MAX_M][MAX_M];
  double A[MAX_M + 1][MAX_M + 2];
  double rms[MAX_M];
  double c[MAX_M];
  int list[MAX_M];
  int m, go, cur_next;
};

// Run by WARP 0 of the last-arriving CTA once the Gram row s_row (entries 0..nother-1: <R_new, R_other[j]>, entry
// nother: <R_new, R_new>) is complete.  Lane 0 does the bookkeeping on a shared-memory copy of the history state;
// the elimination of the bordered system runs across the lanes (one column each), every element taking exactly the
// operations of the oracle's serial loop, so the result is the same to the last bit.
static __device__ __noinline__ void mdiis_bookkeeping_and_solve(DevState* __restrict__ st, SolveScratch& ss,
                                                                const double* s_row, int m_old, int nother,
                                                                AccelArgs aa, double self_unweighted,
                                                                double npts_total) {
  const int lane = threadIdx.x & 31;
  const int M = aa.M;
  const double restart = aa.restart;
  const int skip = (m_old == M) ? 1 : 0;
  // stage the history state (coalesced)
  for (int e = lane; e < MAX_M * MAX_M; e += 32) ss.S[e / MAX_M][e % MAX_M] = st->S[e / MAX_M][e % MAX_M];
  if (lane < MAX_M) { ss.list[lane] = st->list[lane]; ss.rms[lane] = st->rms[lane]; }
  __syncwarp();
  const double self = s_row[nother];
  const double rms = sqrt(self_unweighted / npts_total);   // Eq. 41 (Q9): always the unweighted sum
  if (lane == 0) {
    ss.go = 1;
    st->rms_last = rms;
    st->n_done += 1;
    st->rms_hist[st->hist_n % RMS_HIST_CAP] = rms;
    st->hist_n += 1;
    st->upd_m = 0;
    if (aa.b_max > 0.0) st->b_dyn = fmin(aa.b_max, fmax(aa.b_min, -0.2 * log10(rms)));
    if (!isfinite(rms)) { st->done = 1; st->status = RISM3D_ERR_DIVERGED; ss.go = 0; }
    else if (st->tol > 0.0 && rms < st->tol) { st->done = 1; ss.go = 0; }   // converged: tau stays as it is
    if (ss.go) {
      // append (cur, R_new) to the history, dropping the oldest entry of a full history
      int m = m_old;
      if (skip) {
        for (int i = 0; i + 1 < m; ++i) {
          ss.list[i] = ss.list[i + 1];
          ss.rms[i] = ss.rms[i + 1];
          for (int j = 0; j + 1 < m; ++j) ss.S[i][j] = ss.S[i + 1][j + 1];
        }
        m -= 1;
      }
      ss.list[m] = st->cur;
      ss.rms[m] = rms;
      for (int i = 0; i < m; ++i) ss.S[m][i] = ss.S[i][m] = s_row[i];
      ss.S[m][m] = self;
      m += 1;
      // restart rule (Q8): keep only the entry with the smallest rms (first minimum)
      if (restart > 0.0) {
        double rmin = ss.rms[0];
        int best = 0;
        for (int i = 1; i < m; ++i)
          if (ss.rms[i] < rmin) { rmin = ss.rms[i]; best = i; }
        if (rms > restart * rmin) {
          ss.list[0] = ss.list[best];
          ss.rms[0] = ss.rms[best];
          ss.S[0][0] = ss.S[best][best];
          m = 1;
        }
      }
      ss.m = m;
      for (int i = 0; i < m; ++i) ss.c[i] = (i == m - 1) ? 1.0 : 0.0;   // fallback: unit vector on the newest entry
    }
  }
  __syncwarp();
  if (!ss.go) return;
  const int m = ss.m;
  double smax = ss.S[0][0];
  for (int i = 1; i < m; ++i) smax = fmax(smax, ss.S[i][i]);
  if (aa.accel == RISM3D_ACCEL_ANDERSON) {
    // Modified Anderson, two histories (Eq. 34-39).  Entries: newest = m-1 (R0), m-2 (R1), m-3 (R2).  theta from the
    // normal equations of min |R0 - sum_j theta_j dR_j|^2, dR_j = R0 - Rj (Eq. 36); with a_i = theta_i + s_i,
    //   X_new = u + b (v - u) = (1 - a1 - a2)(X0 + b R0) + a1 (X1 + b R1) + a2 (X2 + b R2) = sum_k c_k Z_k.
    // Picard steps (unit vector on the newest Z) until two histories exist.
    if (m == 3 && lane == 0) {
      const double s00 = ss.S[2][2], s01 = ss.S[2][1], s02 = ss.S[2][0], s11 = ss.S[1][1], s12 = ss.S[1][0],
                   s22 = ss.S[0][0];
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
      ss.c[2] = 1.0 - a1 - a2;
      ss.c[1] = a1;
      ss.c[0] = a2;
    }
  } else if (smax > 0.0) {
    // bordered system [[S/smax, 1], [1^T, 0]] [c; lambda] = [0; 1], Gaussian elimination with partial pivoting; every
    // product and difference is rounded separately (no FMA contraction), as in the oracle.  Lane j owns column j.
    const int n = m + 1;
    for (int e = lane; e < n * (n + 1); e += 32) {
      const int i = e / (n + 1), j = e % (n + 1);
      double v = 0.0;
      if (i < m && j < m) v = ss.S[i][j] / smax;
      else if ((i < m && j == m) || (i == m && j < m) || (i == m && j == n)) v = 1.0;
      ss.A[i][j] = v;
    }
    __syncwarp();
    bool ok = true;
    for (int colx = 0; colx < n; ++colx) {
      int piv = colx;                                   // every lane finds the same pivot
      for (int r = colx + 1; r < n; ++r)
        if (fabs(ss.A[r][colx]) > fabs(ss.A[piv][colx])) piv = r;
      if (ss.A[piv][colx] == 0.0) { ok = false; break; }
      __syncwarp();
      if (piv != colx && lane <= n) { const double tmp = ss.A[colx][lane]; ss.A[colx][lane] = ss.A[piv][lane]; ss.A[piv][lane] = tmp; }
      __syncwarp();
      const double pivot = ss.A[colx][colx];
      for (int r = colx + 1; r < n; ++r) {
        const double fac = ss.A[r][colx] / pivot;
        __syncwarp();                                   // everyone has read A[r][colx] before lane colx overwrites it
        if (lane >= colx && lane <= n) ss.A[r][lane] = __dsub_rn(ss.A[r][lane], __dmul_rn(fac, ss.A[colx][lane]));
      }
      __syncwarp();
    }
    if (ok && lane == 0) {
      double xs[MAX_M + 1];
      for (int r = n - 1; r >= 0; --r) {
        double acc = ss.A[r][n];
        for (int j = r + 1; j < n; ++j) acc = __dsub_rn(acc, __dmul_rn(ss.A[r][j], xs[j]));
        xs[r] = acc / ss.A[r][r];
      }
      for (int i = 0; i < m; ++i) ss.c[i] = xs[i];
    }
  }
  __syncwarp();

  // slot of the NEXT (Z, R) pair: a full history reuses the slot of its oldest entry (dropped next iteration,
  // and not read by the Gram row of that iteration), otherwise the first unused slot
  if (lane == 0) {
    int nxt;
    if (m == M) {
      nxt = ss.list[0];
    } else {
      unsigned used = 0;
      for (int i = 0; i < m; ++i) used |= 1u << ss.list[i];
      nxt = 0;
      while (used & (1u << nxt)) ++nxt;
    }
    st->m = m;
    st->upd_m = m;
    st->cur = nxt;
  }
  // write the history state back (coalesced)
  for (int e = lane; e < MAX_M * MAX_M; e += 32) st->S[e / MAX_M][e % MAX_M] = ss.S[e / MAX_M][e % MAX_M];
  if (lane < MAX_M) {
    st->list[lane] = ss.list[lane];
    st->rms[lane] = ss.rms[lane];
    if (lane < m) { st->upd_list[lane] = ss.list[lane]; st->upd_coef[lane] = ss.c[lane]; }
  }
}

// Called by ALL threads of every CTA of a kernel that has just written its per-CTA partials
//   part1[(j * nblk + blockIdx.x)]  (double-double, j = 0..nother-1 and j = MAX_M for <R_new, R_new>)
// with a __threadfence() after the writes.  Level 1: the last CTA of each group of GRAM_GROUP consecutive CTAs adds
// the group's partials into part2[(j * ngroups + group)].  Level 2: the last such group adder adds the group sums,
// then one thread runs the bookkeeping and the small solve.  Every sum runs in a fixed order, so the result does not
// depend on which CTA arrives last.  tickets: [ngroups] counters, zero on entry, zero again on exit.
// Slab-decomposed runs (xr.n_dst > 0): this rank's sums cover its own planes only.  The last arriver then writes its
// row of double-double totals into slot `rank` of every destination's exchange array and stops; gram_solve_kernel,
// launched once all ranks' rows are there, adds them in rank order and runs the bookkeeping and the solve -- on every
// rank, from identical numbers, so all ranks take identical decisions.
struct GramExchange {
  double* dst[MAX_RANKS];   // [n_ranks][GRAM_SLOT][2] arrays: this rank's own, and its peers' when they are mapped
  int n_dst;                // 0: single rank, solve right away
  int rank;
};

template <int NT>
static __device__ __forceinline__ void gram_finish(DevState* __restrict__ st, double* __restrict__ part1,
                                                   double* __restrict__ part2, unsigned* __restrict__ tickets,
                                                   int m_old, int nother, AccelArgs aa, bool weighted,
                                                   double npts_total, double* s_row /* shared, MAX_M + 2 */,
                                                   int* s_flag /* shared */, SolveScratch& ss /* shared */,
                                                   const GramExchange& xr) {
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
    if (lane == 0) {
      if (xr.n_dst > 0) {
        dd_norm(hi, lo);
        for (int d = 0; d < xr.n_dst; ++d)
          *reinterpret_cast<double2*>(xr.dst[d] + ((size_t)xr.rank * GRAM_SLOT + jj) * 2) = make_double2(hi, lo);
      } else {
        s_row[jj] = hi + lo;
      }
    }
  }
  __syncthreads();
  if (wid != 0) return;
  if (lane == 0) st->ticket = 0;
  if (xr.n_dst > 0) {
    __threadfence_system();                            // peers read the row after the in-stream barrier
    return;
  }
  mdiis_bookkeeping_and_solve(st, ss, s_row, m_old, nother, aa, weighted ? s_row[nother + 1] : s_row[nother], npts_total);
}

}  // namespace r3d
