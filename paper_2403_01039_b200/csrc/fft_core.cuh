// fft_core.cuh -- fp64 complex FFT building blocks for sm_100a: in-register radix-2/4/8/16/32 DFTs and
// the multi-pass Stockham-free (in-place, digit-indexed) line transforms that the 3D passes share.
//
// The transform is the SHIFTED DFT of the paper's half-integer k grid:
//     forward   F_j = sum_m f_m exp(-2 pi i (j + 1/2) m / N)
//     inverse   f_m = (1/N) sum_j F_j exp(+2 pi i (j + 1/2) m / N)
// (HALF = true) or the plain DFT (HALF = false, used for the z axis where the half shift is folded
// into the real<->half-spectrum packing).  Forward lines run decimation-in-frequency, inverse lines
// the mirrored decimation-in-time, so that both read and write NATURAL order in global memory and
// exchange data through one shared-memory tile in place:
//     N = R1*R2(*R3),  m = m1*S1 + r  (S1 = N/R1),  j = k1 + R1*k2 (+ R1*R2*k3)
//     forward pass A : DFT_R1 over m1 (odd-frequency when HALF), twiddle exp(-2 pi i (k1+1/2) r / N)
//     forward pass B : DFT_R2 over m2 inside block k1 (, twiddle, pass C: DFT_R3)
//     inverse        : the conjugate transpose of the above, stage by stage.
// Nothing here is shared with the CPU oracle (oracle/ is numpy).
#pragma once
#include <cuda_runtime.h>

namespace r3d {

typedef double2 cplx;

__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cmul(cplx a, cplx b) {
  return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ cplx cmulc(cplx a, cplx b) {   // a * conj(b)
  return make_double2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}
__device__ __forceinline__ cplx cscale(cplx a, double s) { return make_double2(a.x * s, a.y * s); }

// multiply by exp(DIR * 2 pi i * idx / 16), idx a compile-time-foldable integer in [0, 8)
template <int DIR>
__device__ __forceinline__ cplx mul_w16(cplx v, int idx) {
  const double C1 = 0.92387953251128673848;   // cos(pi/8)
  const double S1 = 0.38268343236508978178;   // sin(pi/8)
  const double H = 0.70710678118654752440;    // sqrt(1/2)
  const double d = (double)DIR;
  switch (idx) {
    case 0: return v;
    case 4: return make_double2(-d * v.y, d * v.x);                                  // * (DIR i)
    case 2: return make_double2(H * (v.x - d * v.y), H * (v.y + d * v.x));           // * (1 + DIR i)/sqrt2
    case 6: return make_double2(-H * (v.x + d * v.y), H * (d * v.x - v.y));          // * (-1 + DIR i)/sqrt2
    case 1: return make_double2(C1 * v.x - d * S1 * v.y, C1 * v.y + d * S1 * v.x);
    case 3: return make_double2(S1 * v.x - d * C1 * v.y, S1 * v.y + d * C1 * v.x);
    case 5: return make_double2(-S1 * v.x - d * C1 * v.y, -S1 * v.y + d * C1 * v.x);
    default: return make_double2(-C1 * v.x - d * S1 * v.y, -C1 * v.y + d * S1 * v.x);  // 7
  }
}

// cos(pi k / 16), k = 0..16 (compile-time: folds to immediates in fully unrolled code)
__host__ __device__ constexpr double cos_pi16(int k) {
  switch (k) {
    case 0: return 1.0;
    case 1: return 0.98078528040323044913;
    case 2: return 0.92387953251128673848;
    case 3: return 0.83146961230254523708;
    case 4: return 0.70710678118654752440;
    case 5: return 0.55557023301960222474;
    case 6: return 0.38268343236508978178;
    case 7: return 0.19509032201612826785;
    case 8: return 0.0;
    default: return -cos_pi16(16 - k);
  }
}
__host__ __device__ constexpr double sin_pi16(int k) { return k <= 8 ? cos_pi16(8 - k) : cos_pi16(k - 8); }   // k = 0..16
// v * exp(DIR i pi IDX / 16), IDX in [0, 16)
template <int IDX, int DIR>
__device__ __forceinline__ cplx mul_w32c(cplx v) {
  if constexpr (IDX == 0) return v;
  else if constexpr (IDX == 8) return make_double2(-(double)DIR * v.y, (double)DIR * v.x);
  else {
    constexpr double c = cos_pi16(IDX), s = (double)DIR * sin_pi16(IDX);
    return make_double2(v.x * c - v.y * s, v.x * s + v.y * c);
  }
}
// cos(pi k / 32), k = 0..32
__host__ __device__ constexpr double cos_pi32(int k) {
  switch (k) {
    case 1: return 0.99518472667219688624;
    case 3: return 0.95694033573220886494;
    case 5: return 0.88192126434835502971;
    case 7: return 0.77301045336273696081;
    case 9: return 0.63439328416364549822;
    case 11: return 0.47139673682599764856;
    case 13: return 0.29028467725446236764;
    case 15: return 0.09801714032956060199;
    default: return (k & 1) ? -cos_pi32(32 - k) : cos_pi16(k / 2);
  }
}
__host__ __device__ constexpr double sin_pi32(int k) { return k <= 16 ? cos_pi32(16 - k) : cos_pi32(k - 16); }   // k = 0..32
// v * exp(DIR i pi IDX / 32), IDX in [0, 32)
template <int IDX, int DIR>
__device__ __forceinline__ cplx mul_w64c(cplx v) {
  if constexpr (IDX % 2 == 0) return mul_w32c<IDX / 2, DIR>(v);
  else {
    constexpr double c = cos_pi32(IDX), s = (double)DIR * sin_pi32(IDX);
    return make_double2(v.x * c - v.y * s, v.x * s + v.y * c);
  }
}
template <int R, int DIR, int M1 = 1>
struct HalfShiftAll {       // x[m1] *= exp(DIR i pi m1 / R) for m1 = 1..R-1, R in {2, 4, 8, 16, 32}
  static __device__ __forceinline__ void run(cplx (&x)[R]) {
    if constexpr (M1 < R) {
      x[M1] = mul_w64c<M1 * (32 / R), DIR>(x[M1]);
      HalfShiftAll<R, DIR, M1 + 1>::run(x);
    }
  }
};

// In-register DFT, natural order in and out:  X[k] = sum_m x[m] exp(DIR 2 pi i m k / R),  R in {1,2,4,8,16}
template <int R, int DIR>
struct Dft {
  static __device__ __forceinline__ void run(cplx (&x)[R]) {
    cplx e[R / 2], o[R / 2];
#pragma unroll
    for (int k = 0; k < R / 2; ++k) { e[k] = x[2 * k]; o[k] = x[2 * k + 1]; }
    Dft<R / 2, DIR>::run(e);
    Dft<R / 2, DIR>::run(o);
#pragma unroll
    for (int k = 0; k < R / 2; ++k) {
      cplx t = mul_w16<DIR>(o[k], k * (16 / R));
      x[k] = cadd(e[k], t);
      x[k + R / 2] = csub(e[k], t);
    }
  }
};
template <int DIR>
struct Dft<1, DIR> {
  static __device__ __forceinline__ void run(cplx (&)[1]) {}
};
// radix 32 (the 512-point k-space lines): two radix-16 halves and the 16 twiddles exp(DIR i pi k / 16) as immediates
template <int DIR, int K = 0>
struct Dft32Combine {
  static __device__ __forceinline__ void run(cplx (&x)[32], const cplx (&e)[16], const cplx (&o)[16]) {
    if constexpr (K < 16) {
      const cplx t = mul_w32c<K, DIR>(o[K]);
      x[K] = cadd(e[K], t);
      x[K + 16] = csub(e[K], t);
      Dft32Combine<DIR, K + 1>::run(x, e, o);
    }
  }
};
template <int DIR>
struct Dft<32, DIR> {
  static __device__ __forceinline__ void run(cplx (&x)[32]) {
    cplx e[16], o[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) { e[k] = x[2 * k]; o[k] = x[2 * k + 1]; }
    Dft<16, DIR>::run(e);
    Dft<16, DIR>::run(o);
    Dft32Combine<DIR>::run(x, e, o);
  }
};

// Twiddle table of one grid axis: tab[j] = exp(-i pi j / n), j = 0 .. 2n-1 (device memory, built by the host
// in long double).  For a line transform of length N = n / mul:  exp(-2 pi i a / (2N)) = tab[(a * mul) mod 2n].
struct Twiddle {
  const cplx* tab;
  int mul;
  int mask;   // 2n - 1
  __device__ __forceinline__ cplx operator()(int a) const { return __ldg(tab + ((a * mul) & mask)); }
};

// ---------------------------------------------------------------------------------------------
// Forward (DIR = -1) decimation-in-frequency passes.  Ld(idx) -> cplx, St(idx, cplx).
// t = index of this thread within its column, T = threads per column.
// ---------------------------------------------------------------------------------------------
template <int N, int R1, bool HALF, class Ld, class St>
__device__ __forceinline__ void fwd_pass_a(int t, int T, const Twiddle& tw, Ld ld, St st) {
  constexpr int S1 = N / R1;
  for (int r = t; r < S1; r += T) {
    cplx x[R1];
#pragma unroll
    for (int m1 = 0; m1 < R1; ++m1) x[m1] = ld(m1 * S1 + r);
    if (HALF) {
#pragma unroll
      for (int m1 = 1; m1 < R1; ++m1) x[m1] = cmul(x[m1], tw(m1 * S1));   // exp(-i pi m1 / R1)
    }
    Dft<R1, -1>::run(x);
#pragma unroll
    for (int k1 = 0; k1 < R1; ++k1) {
      const int a = HALF ? (2 * k1 + 1) * r : 2 * k1 * r;                 // exp(-2 pi i (k1 [+1/2]) r / N)
      st(k1 * S1 + r, (a == 0) ? x[k1] : cmul(x[k1], tw(a)));
    }
  }
}

// middle pass of a 3-pass transform: DFT_R2 inside block k1 over m2 (stride S2), twiddle exp(-2 pi i k2 r2 / S1)
template <int N, int R1, int R2, class Ld, class St>
__device__ __forceinline__ void fwd_pass_mid(int t, int T, const Twiddle& tw, Ld ld, St st) {
  constexpr int S1 = N / R1, S2 = S1 / R2;
  for (int b = t; b < N / R2; b += T) {
    const int k1 = b / S2, r2 = b % S2;
    cplx x[R2];
#pragma unroll
    for (int m2 = 0; m2 < R2; ++m2) x[m2] = ld(k1 * S1 + m2 * S2 + r2);
    Dft<R2, -1>::run(x);
#pragma unroll
    for (int k2 = 0; k2 < R2; ++k2) {
      const int a = 2 * R1 * k2 * r2;
      st(k1 * S1 + k2 * S2 + r2, (a == 0) ? x[k2] : cmul(x[k2], tw(a)));
    }
  }
}

// last pass: DFT_RL over the unit-stride digit of block `blk` (blk = k1 for 2 passes, k1*R2+k2 for 3).
// Out(j, value) receives NATURAL frequency index j.  JMUL = product of the earlier radices.
template <int N, int RL, int R1, class Ld, class Out>
__device__ __forceinline__ void fwd_pass_last(int t, int T, Ld ld, Out out) {
  constexpr int NB = N / RL;          // number of blocks
  constexpr int RMID = NB / R1;       // R2 of a 3-pass transform, 1 otherwise
  for (int blk = t; blk < NB; blk += T) {
    cplx x[RL];
#pragma unroll
    for (int m = 0; m < RL; ++m) x[m] = ld(blk * RL + m);
    Dft<RL, -1>::run(x);
    const int k1 = blk / RMID, k2 = blk % RMID;
    const int j0 = k1 + R1 * k2;
#pragma unroll
    for (int k = 0; k < RL; ++k) out(j0 + NB * k, x[k]);
  }
}

// ---------------------------------------------------------------------------------------------
// Inverse (DIR = +1) decimation-in-time stages: the mirror image of the passes above.
// ---------------------------------------------------------------------------------------------
// first stage: In(j, pos) reads NATURAL frequency index j (pos = the in-place slot blk*RL + k of that value, for
// sources staged in digit-reversed order, see inv_first_slot); DFT_RL over the last digit; twiddle (3-pass only); St(idx)
template <int N, int RL, int R1, class In, class St>
__device__ __forceinline__ void inv_stage_first(int t, int T, const Twiddle& tw, bool half2, In in, St st) {
  constexpr int NB = N / RL;
  constexpr int RMID = NB / R1;
  for (int blk = t; blk < NB; blk += T) {
    const int k1 = blk / RMID, k2 = blk % RMID;
    const int j0 = k1 + R1 * k2;
    cplx x[RL];
#pragma unroll
    for (int k = 0; k < RL; ++k) x[k] = in(j0 + NB * k, blk * RL + k);
    Dft<RL, +1>::run(x);
#pragma unroll
    for (int r = 0; r < RL; ++r) {
      // 2-pass: this stage's output index r is the r of pass A: twiddle exp(+2 pi i (k1 [+1/2]) r / N)
      // 3-pass: mirror of the middle pass: exp(+2 pi i k2 r / S1)
      int a;
      if (RMID == 1) a = half2 ? (2 * k1 + 1) * r : 2 * k1 * r;
      else a = 2 * R1 * k2 * r;
      st(blk * RL + r, (a == 0) ? x[r] : cmulc(x[r], tw(a)));
    }
  }
}

// slot of natural frequency index j in the layout inv_stage_first works on in place: j = k1 + R1*k2 + NB*k
// -> (k1*RMID + k2)*RL + k
template <int N, int RL, int R1>
__device__ __forceinline__ int inv_first_slot(int j) {
  constexpr int NB = N / RL, RMID = NB / R1;
  const int k = j / NB, rem = j % NB;
  return ((rem % R1) * RMID + rem / R1) * RL + k;
}

// middle stage of a 3-pass inverse: DFT_R2 over k2 (stride S2) inside block k1, twiddle exp(+2 pi i (k1[+1/2]) r / N)
template <int N, int R1, int R2, bool HALF, class Ld, class St>
__device__ __forceinline__ void inv_stage_mid(int t, int T, const Twiddle& tw, Ld ld, St st) {
  constexpr int S1 = N / R1, S2 = S1 / R2;
  for (int b = t; b < N / R2; b += T) {
    const int k1 = b / S2, r2 = b % S2;
    cplx x[R2];
#pragma unroll
    for (int k2 = 0; k2 < R2; ++k2) x[k2] = ld(k1 * S1 + k2 * S2 + r2);
    Dft<R2, +1>::run(x);
#pragma unroll
    for (int m2 = 0; m2 < R2; ++m2) {
      const int r = m2 * S2 + r2;
      const int a = HALF ? (2 * k1 + 1) * r : 2 * k1 * r;
      st(k1 * S1 + r, (a == 0) ? x[m2] : cmulc(x[m2], tw(a)));
    }
  }
}

// last stage: DFT_R1 over k1 (stride S1); when HALF the outputs get exp(+i pi m1 / R1); Out(m, value), m natural.
template <int N, int R1, bool HALF, class Ld, class Out>
__device__ __forceinline__ void inv_stage_last(int t, int T, const Twiddle& tw, Ld ld, Out out) {
  constexpr int S1 = N / R1;
  for (int r = t; r < S1; r += T) {
    cplx x[R1];
#pragma unroll
    for (int k1 = 0; k1 < R1; ++k1) x[k1] = ld(k1 * S1 + r);
    Dft<R1, +1>::run(x);
#pragma unroll
    for (int m1 = 0; m1 < R1; ++m1) {
      cplx v = x[m1];
      if (HALF && m1 > 0) v = cmulc(v, tw(m1 * S1));
      out(m1 * S1 + r, v);
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Register-cached twiddles for the persistent strided passes.  A thread of a persistent CTA keeps its position
// (t, column) for every tile, so the twiddles it needs are loop invariants: they are loaded once and stay in
// registers.  To make forward and inverse share ONE set, the inverse applies its twiddles where a stage LOADS
// (thread-fixed r, varying k) instead of where the previous stage stores:
//   a[i][k1] = exp(-2 pi i (k1 + 1/2) r / N),  r = t + i T        forward pass A out  / inverse last stage in
//   m[i][k2] = exp(-2 pi i k2 r2 / S1),  b = t + i T, r2 = b % S2  forward middle out  / inverse middle stage in
// The pre/post factors exp(-+ i pi m1 / R1) of the half-integer grid are compile-time constants for R1 <= 8.
// ---------------------------------------------------------------------------------------------
// MREG = false keeps m in a small shared-memory table [S2][R2] (one per CTA, filled by fill_mid_table) instead of
// registers, for kernels that are short of registers.
template <int N, int R1, int R2, int R3, int T, bool MREG = true>
struct LineTw {
  static constexpr int S1 = N / R1, IA = S1 / T;
  static constexpr bool THREE = (R3 != 1);
  static constexpr int S2 = S1 / R2, IM = THREE ? (N / R2) / T : 1;
  static constexpr int MID_TABLE = THREE ? S2 * R2 : 0;             // complex entries of the shared table
  cplx a[IA][R1];
  cplx m[(THREE && MREG) ? IM : 1][(THREE && MREG) ? R2 : 1];
  const cplx* mt;
  __device__ __forceinline__ void init(int t, const Twiddle& tw, const cplx* mid_table = nullptr) {
#pragma unroll
    for (int i = 0; i < IA; ++i)
#pragma unroll
      for (int k1 = 0; k1 < R1; ++k1) a[i][k1] = tw((2 * k1 + 1) * (t + i * T));
    mt = mid_table;
    if constexpr (THREE && MREG) {
#pragma unroll
      for (int i = 0; i < IM; ++i)
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) m[i][k2] = tw(2 * R1 * k2 * ((t + i * T) % S2));
    }
  }
  __device__ __forceinline__ cplx mid(int i, int r2, int k2) const {
    if constexpr (MREG) return m[i][k2];
    else return mt[r2 * R2 + k2];
  }
  // all threads of the CTA: table[r2 * R2 + k2] = exp(-2 pi i k2 r2 / S1); the caller synchronises afterwards
  static __device__ __forceinline__ void fill_mid_table(cplx* table, const Twiddle& tw, int tid, int nthreads) {
    for (int e = tid; e < MID_TABLE; e += nthreads) table[e] = tw(2 * R1 * (e % R2) * (e / R2));
  }
};

// v * exp(DIR i pi m1 / R1)
template <int R1, int DIR>
__device__ __forceinline__ cplx half_shift(cplx v, int m1, const Twiddle& tw, int S1) {
  if constexpr (R1 <= 8) {
    return mul_w16<DIR>(v, m1 * (8 / R1));
  } else {
    return DIR < 0 ? cmul(v, tw(m1 * S1)) : cmulc(v, tw(m1 * S1));
  }
}

template <int N, int R1, int R2, int R3, int T, bool MR, class Ld, class St>
__device__ __forceinline__ void fwd_a_c(int t, const LineTw<N, R1, R2, R3, T, MR>& w, const Twiddle& tw, Ld ld, St st) {
  constexpr int S1 = N / R1, IA = S1 / T;
#pragma unroll
  for (int i = 0; i < IA; ++i) {
    const int r = t + i * T;
    cplx x[R1];
#pragma unroll
    for (int m1 = 0; m1 < R1; ++m1) x[m1] = ld(m1 * S1 + r);
#pragma unroll
    for (int m1 = 1; m1 < R1; ++m1) x[m1] = half_shift<R1, -1>(x[m1], m1, tw, S1);
    Dft<R1, -1>::run(x);
#pragma unroll
    for (int k1 = 0; k1 < R1; ++k1) st(k1 * S1 + r, cmul(x[k1], w.a[i][k1]));
  }
}

template <int N, int R1, int R2, int R3, int T, bool MR, class Ld, class St>
__device__ __forceinline__ void fwd_mid_c(int t, const LineTw<N, R1, R2, R3, T, MR>& w, Ld ld, St st) {
  constexpr int S1 = N / R1, S2 = S1 / R2, IM = (N / R2) / T;
#pragma unroll
  for (int i = 0; i < IM; ++i) {
    const int b = t + i * T, k1 = b / S2, r2 = b % S2;
    cplx x[R2];
#pragma unroll
    for (int m2 = 0; m2 < R2; ++m2) x[m2] = ld(k1 * S1 + m2 * S2 + r2);
    Dft<R2, -1>::run(x);
    st(k1 * S1 + r2, x[0]);
#pragma unroll
    for (int k2 = 1; k2 < R2; ++k2) st(k1 * S1 + k2 * S2 + r2, cmul(x[k2], w.mid(i, r2, k2)));
  }
}

// inverse first stage on slots staged by inv_first_slot: DFT_RL over the last digit, in place, no twiddle
template <int N, int RL, int T, class Ld, class St>
__device__ __forceinline__ void inv_first_c(int t, Ld ld, St st) {
  constexpr int NB = N / RL;
  for (int blk = t; blk < NB; blk += T) {
    cplx x[RL];
#pragma unroll
    for (int k = 0; k < RL; ++k) x[k] = ld(blk * RL + k);
    Dft<RL, +1>::run(x);
#pragma unroll
    for (int r = 0; r < RL; ++r) st(blk * RL + r, x[r]);
  }
}

template <int N, int R1, int R2, int R3, int T, bool MR, class Ld, class St>
__device__ __forceinline__ void inv_mid_c(int t, const LineTw<N, R1, R2, R3, T, MR>& w, Ld ld, St st) {
  constexpr int S1 = N / R1, S2 = S1 / R2, IM = (N / R2) / T;
#pragma unroll
  for (int i = 0; i < IM; ++i) {
    const int b = t + i * T, k1 = b / S2, r2 = b % S2;
    cplx x[R2];
    x[0] = ld(k1 * S1 + r2);
#pragma unroll
    for (int k2 = 1; k2 < R2; ++k2) x[k2] = cmulc(ld(k1 * S1 + k2 * S2 + r2), w.mid(i, r2, k2));
    Dft<R2, +1>::run(x);
#pragma unroll
    for (int m2 = 0; m2 < R2; ++m2) st(k1 * S1 + m2 * S2 + r2, x[m2]);
  }
}

template <int N, int R1, int R2, int R3, int T, bool MR, class Ld, class Out>
__device__ __forceinline__ void inv_last_c(int t, const LineTw<N, R1, R2, R3, T, MR>& w, const Twiddle& tw, Ld ld, Out out) {
  constexpr int S1 = N / R1, IA = S1 / T;
#pragma unroll
  for (int i = 0; i < IA; ++i) {
    const int r = t + i * T;
    cplx x[R1];
#pragma unroll
    for (int k1 = 0; k1 < R1; ++k1) x[k1] = cmulc(ld(k1 * S1 + r), w.a[i][k1]);
    Dft<R1, +1>::run(x);
    out(r, x[0]);
#pragma unroll
    for (int m1 = 1; m1 < R1; ++m1) out(m1 * S1 + r, half_shift<R1, +1>(x[m1], m1, tw, S1));
  }
}

// a[k] = a0 * s^k, k < R (R a power of two): s^2, s^4, ... by squaring, then a[k + h] = a[k] * s^h -- log2(R) dependent
// products instead of a chain of R - 1
template <int R>
__device__ __forceinline__ void twiddle_powers(cplx (&a)[R], cplx a0, cplx s) {
  a[0] = a0;
  cplx sh = s;
#pragma unroll
  for (int h = 1; h < R; h *= 2) {
#pragma unroll
    for (int k = 0; k < h; ++k) a[k + h] = cmul(a[k], sh);
    if (2 * h < R) sh = cmul(sh, sh);
  }
}
// The pass-A twiddles of one thread, a0 * s^k1 for k1 < R1.  Up to R1 = 16 all of them live in registers; for R1 = 32
// (beside 32 complex data values) only s^0..s^7 and the four chunk bases a0 s^(8c) do, and get() forms the product.
template <int R1>
struct PassATw {
  static constexpr int CH = (R1 > 16) ? 8 : R1, NCH = R1 / CH;
  cplx p[CH];      // NCH == 1: a0 s^k ;  else s^k, k < CH
  cplx base[NCH];  // a0 s^(CH c) (unused when NCH == 1)
  __device__ __forceinline__ PassATw(cplx a0, cplx s) {
    if constexpr (NCH == 1) {
      twiddle_powers<CH>(p, a0, s);
      base[0] = a0;
    } else {
      twiddle_powers<CH>(p, make_double2(1.0, 0.0), s);
      const cplx sc = cmul(p[CH - 1], s);                    // s^CH
      twiddle_powers<NCH>(base, a0, sc);
    }
  }
  __device__ __forceinline__ cplx get(int k1) const {        // k1 folds at compile time in unrolled loops
    if constexpr (NCH == 1) return p[k1];
    else return (k1 % CH == 0) ? base[k1 / CH] : cmul(base[k1 / CH], p[k1 % CH]);
  }
};

// chi row of one k point for this lane's site (kspace_point consumes it)
// Radix plan per line length.  T = threads per column, G = column groups (tiles) per CTA.
template <int N> struct FftCfg;
template <> struct FftCfg<4>   { enum { R1 = 2,  R2 = 2,  R3 = 1, T = 2,  G = 8 }; };
template <> struct FftCfg<8>   { enum { R1 = 4,  R2 = 2,  R3 = 1, T = 2,  G = 8 }; };
template <> struct FftCfg<16>  { enum { R1 = 4,  R2 = 4,  R3 = 1, T = 4,  G = 8 }; };
template <> struct FftCfg<32>  { enum { R1 = 8,  R2 = 4,  R3 = 1, T = 4,  G = 8 }; };
template <> struct FftCfg<64>  { enum { R1 = 8,  R2 = 8,  R3 = 1, T = 8,  G = 4 }; };
template <> struct FftCfg<128> { enum { R1 = 16, R2 = 8,  R3 = 1, T = 8,  G = 2 }; };
// 256: three passes of small radices (4 x 8 x 8, 32 threads per column) beat 16 x 16 in the strided passes, whose
// register-cached twiddles would not fit beside 16 complex values per thread
template <> struct FftCfg<256> { enum { R1 = 4, R2 = 8, R3 = 8, T = 32, G = 1 }; };
template <> struct FftCfg<512> { enum { R1 = 8,  R2 = 8,  R3 = 8, T = 64, G = 1 }; };

}  // namespace r3d
