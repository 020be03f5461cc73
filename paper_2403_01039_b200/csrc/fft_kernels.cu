// fft_kernels.cu -- the r-space <-> k-space passes of one 3D-RISM iteration (steps 2-5):
//
//   closure_zfwd   : g = closure(w + tau), c_sr = g - 1 - tau (Eq. 15-16, 31) fused with the forward
//                    transform along z of the real field into its half spectrum (even j_z only)
//   strided fwd/inv: forward / inverse shifted FFT along y or x (lines with a stride), in place
//   zinv_residual  : inverse transform along z back to the real tau', fused with the MDIIS residual
//                    R = tau' - tau (Eq. 33) and the Gram row <R, R_i>
//
// k-space layout of the work array: complex [jx][jy][p][site], p = 0..n/2-1 standing for j_z = 2p.  A real line
// f_m, m = 0..n-1, has F_{n-1-j} = conj F_j on the half-integer grid, so the even-j half is complete and
//   F_{2p} = sum_{m<n/2} u_m exp(-2 pi i p m/(n/2)),   u_m = (f_m - i f_{m+n/2}) exp(-i pi m / n)
// is a plain n/2-point complex FFT: no DC/Nyquist plane, same bytes as the real field.
#include "fft_core.cuh"
#include "rism3d_internal.h"

namespace r3d {

extern __shared__ double2 smem_dyn[];

constexpr int COLS = 8;   // complex columns per tile row = 128-byte runs in global memory

struct LineGeom {
  size_t outer_stride;     // complex elements between consecutive "outer" blocks of chunks
  size_t es;               // complex elements between consecutive points of one line
  unsigned chunks_per_outer;
};

// ------------------------------------------------------------------------------------------------
// Strided line FFT (y or x axis), in place.  One tile = N points x COLS adjacent columns.
// ------------------------------------------------------------------------------------------------
template <int N, bool INV>
__global__ void __launch_bounds__(FftCfg<N>::T* FftCfg<N>::G* COLS)
    fft_strided_kernel(cplx* __restrict__ data, LineGeom g, Twiddle tw, const DevState* __restrict__ st) {
  if (st != nullptr && st->done) return;
  using Cfg = FftCfg<N>;
  constexpr int T = Cfg::T, R1 = Cfg::R1, R2 = Cfg::R2, R3 = Cfg::R3, C = COLS;
  const int tid = threadIdx.x;
  const int col = tid % C, t = (tid / C) % T, grp = tid / (C * T);
  const size_t chunk = (size_t)blockIdx.x * Cfg::G + grp;
  cplx* sm = smem_dyn + grp * (N * C) + col;
  cplx* base = data + (chunk / g.chunks_per_outer) * g.outer_stride + (chunk % g.chunks_per_outer) * C + col;
  const size_t es = g.es;
  auto ld_sm = [&](int i) { return sm[i * C]; };
  auto st_sm = [&](int i, cplx v) { sm[i * C] = v; };
  if (!INV) {
    fwd_pass_a<N, R1, true>(t, T, tw, [&](int m) { return base[m * es]; }, st_sm);
    __syncthreads();
    auto out = [&](int j, cplx v) { base[j * es] = v; };
    if constexpr (R3 == 1) {
      fwd_pass_last<N, R2, R1>(t, T, ld_sm, out);
    } else {
      fwd_pass_mid<N, R1, R2>(t, T, tw, ld_sm, st_sm);
      __syncthreads();
      fwd_pass_last<N, (R3 == 1 ? R2 : R3), R1>(t, T, ld_sm, out);
    }
  } else {
    const double scale = 1.0 / (double)N;
    auto in = [&](int j) { return base[j * es]; };
    auto out = [&](int m, cplx v) { base[m * es] = cscale(v, scale); };
    if constexpr (R3 == 1) {
      inv_stage_first<N, R2, R1>(t, T, tw, true, in, st_sm);
      __syncthreads();
    } else {
      inv_stage_first<N, (R3 == 1 ? R2 : R3), R1>(t, T, tw, true, in, st_sm);
      __syncthreads();
      inv_stage_mid<N, R1, R2, true>(t, T, tw, ld_sm, st_sm);
      __syncthreads();
    }
    inv_stage_last<N, R1, true>(t, T, tw, ld_sm, out);
  }
}

template <int N, bool INV>
static int launch_strided_n(const Grid& gr, const Buffers& b, bool x_axis, bool use_state, cudaStream_t s) {
  using Cfg = FftCfg<N>;
  const size_t Q = (size_t)(gr.n / 2) * gr.nv;
  LineGeom g;
  size_t nchunks;
  if (x_axis) {
    g.outer_stride = 0;
    g.es = (size_t)gr.n * Q;
    g.chunks_per_outer = (unsigned)((size_t)gr.n * Q / COLS);
    nchunks = g.chunks_per_outer;
  } else {
    g.outer_stride = (size_t)gr.n * Q;
    g.es = Q;
    g.chunks_per_outer = (unsigned)(Q / COLS);
    nchunks = (size_t)gr.n * g.chunks_per_outer;
  }
  const int threads = Cfg::T * Cfg::G * COLS;
  const size_t shm = (size_t)Cfg::G * N * COLS * sizeof(cplx);
  auto kern = fft_strided_kernel<N, INV>;
  cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shm);
  Twiddle tw{b.tw, 1, 2 * gr.n - 1};
  kern<<<(unsigned)(nchunks / Cfg::G), threads, shm, s>>>(b.work, g, tw, use_state ? b.state : nullptr);
  return 1;
}

#define R3D_DISPATCH_N(n, CALL)                    \
  switch (n) {                                     \
    case 8: CALL(8); break;                        \
    case 16: CALL(16); break;                      \
    case 32: CALL(32); break;                      \
    case 64: CALL(64); break;                      \
    case 128: CALL(128); break;                    \
    case 256: CALL(256); break;                    \
    case 512: CALL(512); break;                    \
    default: break;                                \
  }

int launch_y_fwd(const Grid& g, const Buffers& b, bool use_state, cudaStream_t s) {
  int k = 0;
#define CALL(N) k = launch_strided_n<N, false>(g, b, false, use_state, s)
  R3D_DISPATCH_N(g.n, CALL)
#undef CALL
  return k;
}
int launch_y_inv(const Grid& g, const Buffers& b, bool use_state, cudaStream_t s) {
  int k = 0;
#define CALL(N) k = launch_strided_n<N, true>(g, b, false, use_state, s)
  R3D_DISPATCH_N(g.n, CALL)
#undef CALL
  return k;
}
int launch_x_fwd(const Grid& g, const Buffers& b, cudaStream_t s) {
  int k = 0;
#define CALL(N) k = launch_strided_n<N, false>(g, b, true, false, s)
  R3D_DISPATCH_N(g.n, CALL)
#undef CALL
  return k;
}
int launch_x_inv(const Grid& g, const Buffers& b, cudaStream_t s) {
  int k = 0;
#define CALL(N) k = launch_strided_n<N, true>(g, b, true, false, s)
  R3D_DISPATCH_N(g.n, CALL)
#undef CALL
  return k;
}

// ------------------------------------------------------------------------------------------------
// z passes.  A tile = LP = COLS/nv adjacent (ix,iy) lines x nv sites = COLS columns of NZ = n/2 complex points;
// column index = (line in tile) * nv + site, so the k-space rows [p][site] of one line are contiguous.
// Complex tile pitch COLS+1 (conflict-free transposing stores), real tile pitch n+2.
// ------------------------------------------------------------------------------------------------
constexpr int ZP = COLS + 1;

template <int NZ>
__global__ void __launch_bounds__(FftCfg<NZ>::T* FftCfg<NZ>::G* COLS)
    closure_zfwd_kernel(const double* __restrict__ X, const double* __restrict__ w, const double* __restrict__ raw,
                        cplx* __restrict__ work, Twiddle tw_shift, Twiddle tw, const DevState* __restrict__ st,
                        int nv, size_t npts, size_t field, int closure, int order) {
  if (raw == nullptr && st->done) return;
  using Cfg = FftCfg<NZ>;
  constexpr int T = Cfg::T, G = Cfg::G, R1 = Cfg::R1, R2 = Cfg::R2, R3 = Cfg::R3, C = COLS, n = 2 * NZ;
  const int tid = threadIdx.x;
  const int LP = C / nv, GL = G * LP;                 // lines per tile, lines per CTA
  const size_t line0 = (size_t)blockIdx.x * GL;
  const double* tau = raw ? nullptr : X + (size_t)st->cur * field;

  // stage in: closure, pack u_m = (c_m - i c_{m+n/2}) exp(-i pi m / n)
  for (int e = tid; e < GL * nv * NZ; e += blockDim.x) {
    const int m = e % NZ, lc = e / NZ;
    const int site = lc / GL, l = lc % GL;
    const size_t off = (size_t)site * npts + (line0 + l) * n + m;
    double c0, c1;
    if (raw) {
      c0 = raw[off];
      c1 = raw[off + NZ];
    } else {
      const double t0 = tau[off], t1 = tau[off + NZ];
      c0 = closure_g(w[off] + t0, closure, order) - 1.0 - t0;
      c1 = closure_g(w[off + NZ] + t1, closure, order) - 1.0 - t1;
    }
    const cplx u = cmul(make_double2(c0, -c1), tw_shift(m));
    smem_dyn[(l / LP) * (NZ * ZP) + m * ZP + (l % LP) * nv + site] = u;
  }
  __syncthreads();

  const int col = tid % C, t = (tid / C) % T, grp = tid / (C * T);
  cplx* sm = smem_dyn + grp * (NZ * ZP) + col;
  auto ld_sm = [&](int i) { return sm[i * ZP]; };
  auto st_sm = [&](int i, cplx v) { sm[i * ZP] = v; };
  fwd_pass_a<NZ, R1, false>(t, T, tw, ld_sm, st_sm);
  __syncthreads();
  const size_t line = line0 + (size_t)grp * LP + col / nv;
  cplx* dst = work + line * NZ * nv + (col % nv);
  auto out = [&](int p, cplx v) { dst[(size_t)p * nv] = v; };
  if constexpr (R3 == 1) {
    fwd_pass_last<NZ, R2, R1>(t, T, ld_sm, out);
  } else {
    fwd_pass_mid<NZ, R1, R2>(t, T, tw, ld_sm, st_sm);
    __syncthreads();
    fwd_pass_last<NZ, (R3 == 1 ? R2 : R3), R1>(t, T, ld_sm, out);
  }
}

template <int NZ>
static int launch_closure_zfwd_n(const Grid& gr, const Buffers& b, const SolverParams& sp, const double* raw,
                                 cudaStream_t s) {
  using Cfg = FftCfg<NZ>;
  const int LP = COLS / gr.nv, GL = Cfg::G * LP;
  const size_t nlines = (size_t)gr.n * gr.n;
  const int threads = Cfg::T * Cfg::G * COLS;
  const size_t shm = (size_t)Cfg::G * NZ * ZP * sizeof(cplx);
  auto kern = closure_zfwd_kernel<NZ>;
  cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shm);
  Twiddle tws{b.tw, 1, 2 * gr.n - 1}, tw{b.tw, 2, 2 * gr.n - 1};
  kern<<<(unsigned)(nlines / GL), threads, shm, s>>>(b.X, b.w, raw, b.work, tws, tw, b.state, gr.nv, gr.npts,
                                                       gr.field, sp.closure, sp.pse_order);
  return 1;
}

int launch_closure_zfwd(const Grid& g, const Buffers& b, const SolverParams& sp, const double* raw, cudaStream_t s) {
  int k = 0;
  switch (g.n / 2) {
    case 4: k = launch_closure_zfwd_n<4>(g, b, sp, raw, s); break;
    case 8: k = launch_closure_zfwd_n<8>(g, b, sp, raw, s); break;
    case 16: k = launch_closure_zfwd_n<16>(g, b, sp, raw, s); break;
    case 32: k = launch_closure_zfwd_n<32>(g, b, sp, raw, s); break;
    case 64: k = launch_closure_zfwd_n<64>(g, b, sp, raw, s); break;
    case 128: k = launch_closure_zfwd_n<128>(g, b, sp, raw, s); break;
    case 256: k = launch_closure_zfwd_n<256>(g, b, sp, raw, s); break;
    default: break;
  }
  return k;
}

// inverse z + residual + Gram row.  Persistent over tiles so that the Gram accumulators stay in registers.
template <int NZ>
__global__ void __launch_bounds__(FftCfg<NZ>::T* FftCfg<NZ>::G* COLS)
    zinv_residual_kernel(const cplx* __restrict__ work, const double* __restrict__ X, double* __restrict__ R,
                         double* __restrict__ raw_out, double* __restrict__ gram_part, Twiddle tw_shift,
                         Twiddle tw, const DevState* __restrict__ st, int nv, size_t npts, size_t field, int M,
                         unsigned ntiles) {
  if (raw_out == nullptr && st->done) return;
  using Cfg = FftCfg<NZ>;
  constexpr int T = Cfg::T, G = Cfg::G, R1 = Cfg::R1, R2 = Cfg::R2, R3 = Cfg::R3, C = COLS, n = 2 * NZ;
  constexpr int RP = n + 2;                            // real tile pitch (doubles)
  const int tid = threadIdx.x;
  const int LP = C / nv, GL = G * LP;
  cplx* smc = smem_dyn;                                // [G][NZ][ZP] complex
  double* smr = reinterpret_cast<double*>(smem_dyn + G * NZ * ZP);   // [G][C][RP] real

  // MDIIS bookkeeping: the entries the new residual is dotted with
  __shared__ int s_other[MAX_M];
  __shared__ int s_nother, s_cur;
  if (raw_out == nullptr && tid == 0) {
    const int m = st->m;
    const int skip = (m == M) ? 1 : 0;                 // a full history drops its oldest entry this iteration
    s_nother = m - skip;
    s_cur = st->cur;
    for (int i = 0; i < m - skip; ++i) s_other[i] = st->list[i + skip];
  }
  __syncthreads();
  const int nother = raw_out ? 0 : s_nother;
  const double* Xc = raw_out ? nullptr : X + (size_t)s_cur * field;
  double* Rc = raw_out ? nullptr : R + (size_t)s_cur * field;

  double acc_hi[MAX_M + 1], acc_lo[MAX_M + 1];
#pragma unroll
  for (int j = 0; j <= MAX_M; ++j) acc_hi[j] = acc_lo[j] = 0.0;

  const int col = tid % C, t = (tid / C) % T, grp = tid / (C * T);
  cplx* sm = smc + grp * (NZ * ZP) + col;
  double* sr = smr + (grp * C + col) * RP;
  auto ld_sm = [&](int i) { return sm[i * ZP]; };
  auto st_sm = [&](int i, cplx v) { sm[i * ZP] = v; };
  const double scale = 1.0 / (double)NZ;

  for (unsigned tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const size_t line0 = (size_t)tile * GL;
    const size_t line = line0 + (size_t)grp * LP + col / nv;
    const cplx* src = work + line * NZ * nv + (col % nv);
    auto in = [&](int p) { return src[(size_t)p * nv]; };
    if constexpr (R3 == 1) {
      inv_stage_first<NZ, R2, R1>(t, T, tw, false, in, st_sm);
      __syncthreads();
    } else {
      inv_stage_first<NZ, (R3 == 1 ? R2 : R3), R1>(t, T, tw, false, in, st_sm);
      __syncthreads();
      inv_stage_mid<NZ, R1, R2, false>(t, T, tw, ld_sm, st_sm);
      __syncthreads();
    }
    // u_m exp(+i pi m/n) / NZ = f_m - i f_{m+n/2}
    auto out = [&](int m, cplx v) {
      const cplx f = cscale(cmulc(v, tw_shift(m)), scale);
      sr[m] = f.x;
      sr[m + NZ] = -f.y;
    };
    inv_stage_last<NZ, R1, false>(t, T, tw, ld_sm, out);
    __syncthreads();

    // streaming phase: coalesced over z, sites outermost
    for (int e = tid; e < GL * nv * n; e += blockDim.x) {
      const int m = e % n, lc = e / n;
      const int site = lc / GL, l = lc % GL;
      const size_t off = (size_t)site * npts + (line0 + l) * n + m;
      const double tnew = smr[((l / LP) * C + (l % LP) * nv + site) * RP + m];
      if (raw_out) {
        raw_out[off] = tnew;
      } else {
        const double r = tnew - Xc[off];               // R = tau' - tau  (Eq. 33)
        Rc[off] = r;
        dd_add_prod(acc_hi[MAX_M], acc_lo[MAX_M], r, r);
#pragma unroll
        for (int j = 0; j < MAX_M; ++j)
          if (j < nother) dd_add_prod(acc_hi[j], acc_lo[j], r, R[(size_t)s_other[j] * field + off]);
      }
    }
    __syncthreads();
  }
  if (raw_out) return;

  // block reduction of the double-double partial sums: warp shuffles, then one warp over the warp results
  __shared__ double s_red[32][2];
  const int lane = tid & 31, wid = tid >> 5, nw = blockDim.x >> 5;
#pragma unroll
  for (int j = 0; j <= MAX_M; ++j) {
    if (j < nother || j == MAX_M) {
      double hi = acc_hi[j], lo = acc_lo[j];
      for (int o = 16; o > 0; o >>= 1) {
        const double h2 = __shfl_down_sync(0xffffffffu, hi, o), l2 = __shfl_down_sync(0xffffffffu, lo, o);
        dd_add(hi, lo, h2, l2);
      }
      if (lane == 0) { s_red[wid][0] = hi; s_red[wid][1] = lo; }
      __syncthreads();
      if (wid == 0) {
        hi = lane < nw ? s_red[lane][0] : 0.0;
        lo = lane < nw ? s_red[lane][1] : 0.0;
        for (int o = 16; o > 0; o >>= 1) {
          const double h2 = __shfl_down_sync(0xffffffffu, hi, o), l2 = __shfl_down_sync(0xffffffffu, lo, o);
          dd_add(hi, lo, h2, l2);
        }
        if (lane == 0) {
          dd_norm(hi, lo);
          gram_part[((size_t)blockIdx.x * (MAX_M + 1) + j) * 2 + 0] = hi;
          gram_part[((size_t)blockIdx.x * (MAX_M + 1) + j) * 2 + 1] = lo;
        }
      }
      __syncthreads();
    }
  }
}

template <int NZ>
static unsigned zinv_tiles(const Grid& gr) {
  const int LP = COLS / gr.nv, GL = FftCfg<NZ>::G * LP;
  return (unsigned)((size_t)gr.n * gr.n / GL);
}

static unsigned zinv_tiles_rt(const Grid& g) {
  switch (g.n / 2) {
    case 4: return zinv_tiles<4>(g);
    case 8: return zinv_tiles<8>(g);
    case 16: return zinv_tiles<16>(g);
    case 32: return zinv_tiles<32>(g);
    case 64: return zinv_tiles<64>(g);
    case 128: return zinv_tiles<128>(g);
    case 256: return zinv_tiles<256>(g);
    default: return 0;
  }
}

int gram_blocks(const Grid& g) {
  const unsigned tiles = zinv_tiles_rt(g);
  const unsigned cap = 148 * 4;
  return (int)(tiles < cap ? tiles : cap);
}

template <int NZ>
static int launch_zinv_n(const Grid& gr, const Buffers& b, const SolverParams& sp, double* raw_out, cudaStream_t s) {
  using Cfg = FftCfg<NZ>;
  const int threads = Cfg::T * Cfg::G * COLS;
  const size_t shm = (size_t)Cfg::G * NZ * ZP * sizeof(cplx) + (size_t)Cfg::G * COLS * (2 * NZ + 2) * sizeof(double);
  auto kern = zinv_residual_kernel<NZ>;
  cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shm);
  Twiddle tws{b.tw, 1, 2 * gr.n - 1}, tw{b.tw, 2, 2 * gr.n - 1};
  const unsigned tiles = zinv_tiles<NZ>(gr);
  kern<<<gram_blocks(gr), threads, shm, s>>>(b.work, b.X, b.R, raw_out, b.gram_part, tws, tw, b.state, gr.nv,
                                             gr.npts, gr.field, sp.M, tiles);
  return 1;
}

int launch_zinv_residual(const Grid& g, const Buffers& b, const SolverParams& sp, double* raw_out, cudaStream_t s) {
  int k = 0;
  switch (g.n / 2) {
    case 4: k = launch_zinv_n<4>(g, b, sp, raw_out, s); break;
    case 8: k = launch_zinv_n<8>(g, b, sp, raw_out, s); break;
    case 16: k = launch_zinv_n<16>(g, b, sp, raw_out, s); break;
    case 32: k = launch_zinv_n<32>(g, b, sp, raw_out, s); break;
    case 64: k = launch_zinv_n<64>(g, b, sp, raw_out, s); break;
    case 128: k = launch_zinv_n<128>(g, b, sp, raw_out, s); break;
    case 256: k = launch_zinv_n<256>(g, b, sp, raw_out, s); break;
    default: break;
  }
  return k;
}

}  // namespace r3d
