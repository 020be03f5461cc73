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
#include "async_copy.cuh"
#include "fft_core.cuh"
#include "mdiis_device.cuh"
#include "rism3d_internal.h"
#include "tma.cuh"

namespace r3d {

extern __shared__ __align__(128) double2 smem_dyn[];

constexpr int COLS = 8;   // complex columns per tile row = 128-byte runs in global memory

struct LineGeom {
  size_t outer_stride;     // complex elements between consecutive "outer" blocks of chunks
  size_t es;               // complex elements between consecutive points of one line
  unsigned chunks_per_outer;
};

// ------------------------------------------------------------------------------------------------
// Strided line FFT (y or x axis), in place.  One tile = N points x COLS adjacent columns (128-byte rows); a CTA owns
// G tiles at a time.  Persistent CTAs: work item i + gridDim.x streams into one shared-memory buffer (cp.async)
// while the line FFTs of item i run in place on the other; the last radix pass stores straight to global memory.
// ------------------------------------------------------------------------------------------------
template <int N>
struct StridedCfg {
  enum { NT = FftCfg<N>::T * FftCfg<N>::G * COLS,                  // threads per CTA
         ITEM = FftCfg<N>::G * N * COLS,                             // complex elements per work item
         SHM = 2 * ITEM * (int)sizeof(cplx),
         MINB = (SHM > 110 * 1024) ? 1 : 2 };      // <= 128 registers per thread: room for the cached twiddles
};

// Slab-decomposed runs (Grid::n_ranks > 1): the y lines of one x plane are complete in r space, but the rows j_y of the
// spectrum belong to the rank that transforms them along x.  Row j of plane ix_l lives at
//   base[j >> shift] + (ix_l * nyl + (j & mask)) * es          (+ the column offset inside the row)
// -- the forward pass WRITES its rows there (the transpose of PAPER.md:318-322 happens in its stores: a staging block
// per destination rank, or the destination's own array over NVLink), the inverse pass READS them from there.
struct RowMap {
  cplx* base[MAX_RANKS];
  int shift, mask, nyl;
};

// stage work item `item` (G tiles) into `buf` [G][N][COLS]
// (INV: row j goes to the slot the first inverse stage reads it from in place; SLAB: rows come through the row map)
template <int N, bool INV, bool SLAB>
__device__ __forceinline__ void stage_strided(cplx* buf, const cplx* data, const LineGeom& g, const RowMap& rm,
                                              size_t item, int tid) {
  using Cfg = FftCfg<N>;
  constexpr int NT = StridedCfg<N>::NT, C = COLS;
#pragma unroll
  for (int k = 0; k < StridedCfg<N>::ITEM / NT; ++k) {
    const int idx = tid + k * NT;
    const int grp = idx / (N * C), rem = idx % (N * C), row = rem / C, col = rem % C;
    const size_t chunk = item * Cfg::G + grp;
    const cplx* src;
    if constexpr (SLAB && INV)
      src = rm.base[row >> rm.shift] + ((chunk / g.chunks_per_outer) * rm.nyl + (size_t)(row & rm.mask)) * g.es +
            (chunk % g.chunks_per_outer) * C + col;
    else
      src = data + (chunk / g.chunks_per_outer) * g.outer_stride + (chunk % g.chunks_per_outer) * C +
            (size_t)row * g.es + col;
    constexpr int RL = (Cfg::R3 == 1) ? Cfg::R2 : Cfg::R3;
    const int slot = INV ? inv_first_slot<N, RL, Cfg::R1>(row) : row;
    cp_async16(buf + (grp * N + slot) * C + col, src);
  }
}

template <int N, bool INV, bool SLAB>
__global__ void __launch_bounds__(StridedCfg<N>::NT, StridedCfg<N>::MINB)
    fft_strided_kernel(cplx* __restrict__ data, LineGeom g, RowMap rm, Twiddle tw, const DevState* __restrict__ st,
                       unsigned nitems) {
  if (st != nullptr && st->done) return;
  using Cfg = FftCfg<N>;
  constexpr int T = Cfg::T, R1 = Cfg::R1, R2 = Cfg::R2, R3 = Cfg::R3, C = COLS;
  constexpr int ITEM = StridedCfg<N>::ITEM;
  const int tid = threadIdx.x;
  const int col = tid % C, t = (tid / C) % T, grp = tid / (C * T);
  const size_t es = g.es;
  constexpr int RL = (R3 == 1) ? R2 : R3;
  LineTw<N, R1, R2, R3, T> w;                          // this thread's twiddles: the same for every tile
  w.init(t, tw);
  int b = 0;
  size_t item = blockIdx.x;
  if (item < nitems) stage_strided<N, INV, SLAB>(smem_dyn, data, g, rm, item, tid);
  cp_async_commit();
  for (; item < nitems; item += gridDim.x) {
    const size_t next = item + gridDim.x;
    if (next < nitems) stage_strided<N, INV, SLAB>(smem_dyn + (b ^ 1) * ITEM, data, g, rm, next, tid);
    cp_async_commit();
    cp_async_wait<1>();
    __syncthreads();
    cplx* sm = smem_dyn + b * ITEM + grp * (N * C) + col;
    const size_t chunk = item * Cfg::G + grp;
    const size_t plane = chunk / g.chunks_per_outer, inrow = (chunk % g.chunks_per_outer) * C + col;
    cplx* base = data + plane * g.outer_stride + inrow;
    auto ld_sm = [&](int i) { return sm[i * C]; };
    auto st_sm = [&](int i, cplx v) { sm[i * C] = v; };
    if (!INV) {
      fwd_a_c(t, w, tw, ld_sm, st_sm);
      __syncthreads();
      auto out = [&](int j, cplx v) {
        if constexpr (SLAB) rm.base[j >> rm.shift][(plane * rm.nyl + (size_t)(j & rm.mask)) * es + inrow] = v;
        else base[j * es] = v;
      };
      if constexpr (R3 != 1) {
        fwd_mid_c(t, w, ld_sm, st_sm);
        __syncthreads();
      }
      fwd_pass_last<N, RL, R1>(t, T, ld_sm, out);
    } else {
      const double scale = 1.0 / (double)N;
      auto out = [&](int m, cplx v) { base[m * es] = cscale(v, scale); };
      inv_first_c<N, RL, T>(t, ld_sm, st_sm);
      __syncthreads();
      if constexpr (R3 != 1) {
        inv_mid_c(t, w, ld_sm, st_sm);
        __syncthreads();
      }
      inv_last_c(t, w, tw, ld_sm, out);
    }
    __syncthreads();                                   // buffer b is free again
    b ^= 1;
  }
}

template <int N, bool INV>
static int launch_strided_n(const Grid& gr, const Buffers& b, bool x_axis, bool use_state, cudaStream_t s) {
  using Cfg = FftCfg<N>;
  const size_t Q = gr.q();
  LineGeom g;
  size_t nchunks;
  if (x_axis) {                                          // lines along x of [nx][nyl][Q] (N = nx)
    g.outer_stride = 0;
    g.es = (size_t)gr.nyl * Q;
    g.chunks_per_outer = (unsigned)((size_t)gr.nyl * Q / COLS);
    nchunks = g.chunks_per_outer;
  } else {                                               // lines along y of [nxl][ny][Q] (N = ny)
    g.outer_stride = (size_t)gr.ny * Q;
    g.es = Q;
    g.chunks_per_outer = (unsigned)(Q / COLS);
    nchunks = (size_t)gr.nxl * g.chunks_per_outer;
  }
  const unsigned nitems = (unsigned)(nchunks / Cfg::G);
  const size_t shm = StridedCfg<N>::SHM;
  const bool slab = gr.n_ranks > 1 && !x_axis;
  RowMap rm{};
  if (slab) {
    rm.nyl = gr.nyl;
    rm.mask = gr.nyl - 1;
    rm.shift = 0;
    while ((1 << rm.shift) < gr.nyl) ++rm.shift;
    for (int r = 0; r < gr.n_ranks; ++r) rm.base[r] = INV ? const_cast<cplx*>(b.bwd_src[r]) : b.fwd_dst[r];
  }
  auto kern = slab ? fft_strided_kernel<N, INV, true> : fft_strided_kernel<N, INV, false>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shm) != cudaSuccess) return 0;
  Twiddle tw{b.tw, gr.nmax / N, 2 * gr.nmax - 1};
  unsigned grid = (unsigned)(gr.num_sms * StridedCfg<N>::MINB);
  if (grid > nitems) grid = nitems;
  kern<<<grid, StridedCfg<N>::NT, shm, s>>>(b.work, g, rm, tw, use_state ? b.state : nullptr, nitems);
  return 1;
}

// ------------------------------------------------------------------------------------------------
// Two-pass y transform for the long lines (64 = 8 x 8, 128 = 16 x 8, 256 = 16 x 16), single-rank runs: the scheme of the
// k-space pass (kspace_kernel.cu) without its arithmetic.  Tiles of N rows x 128 (or 256) bytes arrive by TMA (one request per
// tile, two stages, no LDGSTS issue slots and no staging registers), each thread does one radix-R1 butterfly per outer
// pass with twiddles generated from two seeds, the other pass runs on registers and the results leave from registers as
// 128-byte rows: 2 loads + 1 store of the tile in shared memory per work item instead of 3 + 3 (cp.async staging
// included) in the three-pass kernel above.
// ------------------------------------------------------------------------------------------------
template <int N> struct YPlan2 { enum { OK = 0, R1 = 1, R2 = 1 }; };
template <> struct YPlan2<64>  { enum { OK = 1, R1 = 8,  R2 = 8 }; };
template <> struct YPlan2<128> { enum { OK = 1, R1 = 16, R2 = 8 }; };
template <> struct YPlan2<256> { enum { OK = 1, R1 = 16, R2 = 16 }; };

template <int N, int CC>
struct Y2Cfg {
  enum { R1 = YPlan2<N>::R1, R2 = YPlan2<N>::R2, T = N / R1, NT = T * CC, NB = N / R2, IB = NB / T,
         ITEM = N * CC, TILE_BYTES = ITEM * (int)sizeof(cplx), SHM = 2 * TILE_BYTES + 64,
         FIT = 227 * 1024 / (SHM + 1024), CAP = (N >= 256) ? 2 : 4, MINB = FIT < CAP ? FIT : CAP };
};

template <int N, bool INV, int CC>
__global__ void __launch_bounds__(Y2Cfg<N, CC>::NT, Y2Cfg<N, CC>::MINB)
    fft_y2_kernel(const __grid_constant__ CUtensorMap tm, cplx* __restrict__ data, Twiddle tw,
                  const DevState* __restrict__ st, unsigned chunks_per_plane, size_t plane_stride, size_t es,
                  unsigned nitems) {
  if (st != nullptr && st->done) return;
  using K = Y2Cfg<N, CC>;
  constexpr int R1 = K::R1, R2 = K::R2, T = K::T, C = CC, S1 = N / R1, NB = K::NB, IB = K::IB;
  const int tid = threadIdx.x;
  const int col = tid % C, t = tid / C;
  const cplx a0 = tw(t), astep = tw(2 * t);          // exp(-i pi t / N) and its square: a[k1] = a0 * astep^k1
  cplx* stages = smem_dyn;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem_dyn + 2 * K::ITEM);
  auto issue = [&](unsigned it, int b) {
    mbar_arrive_expect_tx(&bars[b], K::TILE_BYTES);
    tma_load_2d(stages + b * K::ITEM, &tm, (int)((it % chunks_per_plane) * C * 2), (int)((it / chunks_per_plane) * N), &bars[b]);
  };
  if (tid == 0) {
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    mbar_fence_init();
  }
  __syncthreads();
  unsigned item = blockIdx.x;
  if (tid == 0 && item < nitems) issue(item, 0);
  unsigned n_done = 0;
  for (; item < nitems; item += gridDim.x, ++n_done) {
    const int b = n_done & 1;
    const unsigned next = item + gridDim.x;
    if (tid == 0 && next < nitems) issue(next, b ^ 1);   // (every thread left stage b ^ 1 before the barrier that ended the last item)
    cplx* sm = stages + b * K::ITEM + col;
    auto ld_sm = [&](int i) { return sm[i * C]; };
    auto st_sm = [&](int i, cplx v) { sm[i * C] = v; };
    cplx* base = data + (size_t)(item / chunks_per_plane) * plane_stride + (size_t)(item % chunks_per_plane) * C + col;
    mbar_wait(&bars[b], (n_done >> 1) & 1);
    if constexpr (!INV) {
      {                                              // pass A: half-integer shift, radix R1 over m1, twiddle
        cplx x[R1];
#pragma unroll
        for (int m1 = 0; m1 < R1; ++m1) x[m1] = ld_sm(m1 * S1 + t);
        HalfShiftAll<R1, -1>::run(x);
        Dft<R1, -1>::run(x);
        const PassATw<R1> a(a0, astep);
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) st_sm(k1 * S1 + t, cmul(x[k1], a.get(k1)));
      }
      __syncthreads();
#pragma unroll
      for (int i = 0; i < IB; ++i) {                 // pass B on registers, rows out in natural order
        const int blk = t + i * T;
        cplx x[R2];
#pragma unroll
        for (int m = 0; m < R2; ++m) x[m] = ld_sm(blk * R2 + m);
        Dft<R2, -1>::run(x);
#pragma unroll
        for (int k = 0; k < R2; ++k) base[(size_t)(blk + NB * k) * es] = x[k];
      }
    } else {
      cplx y[IB][R2];                                // first inverse stage: rows blk + NB k, natural order in the tile
#pragma unroll
      for (int i = 0; i < IB; ++i)
#pragma unroll
        for (int k = 0; k < R2; ++k) y[i][k] = ld_sm((t + i * T) + NB * k);
      __syncthreads();                               // every row has been read before any slot is rewritten
#pragma unroll
      for (int i = 0; i < IB; ++i) {
        Dft<R2, +1>::run(y[i]);
#pragma unroll
        for (int r = 0; r < R2; ++r) st_sm((t + i * T) * R2 + r, y[i][r]);
      }
      __syncthreads();
      {                                              // last stage: conjugate twiddle, radix R1 over k1, shift, 1/N
        cplx x[R1];
        const PassATw<R1> a(a0, astep);
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) x[k1] = cmulc(ld_sm(k1 * S1 + t), a.get(k1));
        Dft<R1, +1>::run(x);
        HalfShiftAll<R1, +1>::run(x);
        const double scale = 1.0 / (double)N;
#pragma unroll
        for (int m1 = 0; m1 < R1; ++m1) base[(size_t)(m1 * S1 + t) * es] = cscale(x[m1], scale);
      }
    }
    fence_proxy_async();                             // this item's st.shared writes to stage b come before the TMA load that
    __syncthreads();                                 // refills it (generic -> async proxy);  stage b is free again
  }
}

// complex columns per tile: 16 (256-byte rows, one 256-thread CTA per SM) for the 256-point lines -- fewer, longer
// requests in flight suit the memory system better than two CTAs fetching 128-byte rows (C4: 0.199 -> 0.177 ms per
// pass; profiles/README.md) -- 8 otherwise (at 128 points the two are level, at 512 the tile would not fit)
int y_tile_cols(const Grid& gr) { return (gr.ny == 256 && gr.q() % 16 == 0) ? 16 : COLS; }

template <int N, bool INV, int CC>
static int launch_y2_cc(const Grid& gr, const Buffers& b, bool use_state, cudaStream_t s) {
  if constexpr (YPlan2<N>::OK) {
    using K = Y2Cfg<N, CC>;
    const size_t Q = gr.q();
    const unsigned cpp = (unsigned)(Q / CC), nitems = (unsigned)gr.nxl * cpp;
    auto kern = fft_y2_kernel<N, INV, CC>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)K::SHM) != cudaSuccess) return 0;
    Twiddle tw{b.tw, gr.nmax / N, 2 * gr.nmax - 1};
    unsigned grid = (unsigned)(gr.num_sms * K::MINB);
    if (grid > nitems) grid = nitems;
    kern<<<grid, K::NT, K::SHM, s>>>(b.tm_ywork, b.work, tw, use_state ? b.state : nullptr, cpp, (size_t)gr.ny * Q, Q, nitems);
    return 1;
  } else {
    return 0;
  }
}
template <int N, bool INV>
static int launch_y2_n(const Grid& gr, const Buffers& b, bool use_state, cudaStream_t s) {
  if constexpr (N == 256) {
    if (y_tile_cols(gr) == 16) return launch_y2_cc<N, INV, 16>(gr, b, use_state, s);
  }
  return launch_y2_cc<N, INV, COLS>(gr, b, use_state, s);
}

// true when the y passes of this grid take the two-pass TMA kernel (the API layer then builds its tensor map)
bool y_uses_tma(int ny, int n_ranks) { return n_ranks == 1 && (ny == 64 || ny == 128 || ny == 256); }

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
  if (y_uses_tma(g.ny, g.n_ranks)) {
    switch (g.ny) {
      case 64: return launch_y2_n<64, false>(g, b, use_state, s);
      case 128: return launch_y2_n<128, false>(g, b, use_state, s);
      default: return launch_y2_n<256, false>(g, b, use_state, s);
    }
  }
#define CALL(N) k = launch_strided_n<N, false>(g, b, false, use_state, s)
  R3D_DISPATCH_N(g.ny, CALL)
#undef CALL
  return k;
}
int launch_y_inv(const Grid& g, const Buffers& b, bool use_state, cudaStream_t s) {
  int k = 0;
  if (y_uses_tma(g.ny, g.n_ranks)) {
    switch (g.ny) {
      case 64: return launch_y2_n<64, true>(g, b, use_state, s);
      case 128: return launch_y2_n<128, true>(g, b, use_state, s);
      default: return launch_y2_n<256, true>(g, b, use_state, s);
    }
  }
#define CALL(N) k = launch_strided_n<N, true>(g, b, false, use_state, s)
  R3D_DISPATCH_N(g.ny, CALL)
#undef CALL
  return k;
}
int launch_x_fwd(const Grid& g, const Buffers& b, cudaStream_t s) {
  int k = 0;
#define CALL(N) k = launch_strided_n<N, false>(g, b, true, false, s)
  R3D_DISPATCH_N(g.nx, CALL)
#undef CALL
  return k;
}
int launch_x_inv(const Grid& g, const Buffers& b, cudaStream_t s) {
  int k = 0;
#define CALL(N) k = launch_strided_n<N, true>(g, b, true, false, s)
  R3D_DISPATCH_N(g.nx, CALL)
#undef CALL
  return k;
}

// ------------------------------------------------------------------------------------------------
// z passes.  A tile = LP = COLS/nv adjacent (ix,iy) lines x nv sites = COLS columns of NZ = n/2 complex points;
// column index = (line in tile) * nv + site, so the k-space rows [p][site] of one line are contiguous.
// Complex tile pitch COLS+1 (conflict-free transposing stores), real tile pitch n+2.
// ------------------------------------------------------------------------------------------------
constexpr int ZP = COLS + 1;

// Configuration of the z kernels per line length NZ = n/2: radix plan (R1, R2, R3, T threads per column), column
// groups per CTA and resident CTAs per SM the kernel is compiled for (register cap), separately for closure_zfwd
// (GF, MBF) and zinv_residual (GI, MBI).  The large lines run 3-pass plans of small radices: few registers per thread,
// so that 768-1024 threads per SM hide the latency of the closure's exp() chains and of the streaming loads.
template <int NZ> struct ZPlan : FftCfg<NZ> { enum { GF = FftCfg<NZ>::G, MBF = 1, GI = FftCfg<NZ>::G, MBI = 1, MBG = 1 }; };
template <> struct ZPlan<64>  { enum { R1 = 8, R2 = 8, R3 = 1, T = 8, G = 4, GF = 2, MBF = 4, GI = 2, MBI = 8, MBG = 5 }; };
template <> struct ZPlan<128> { enum { R1 = 4, R2 = 4, R3 = 8, T = 16, G = 2, GF = 1, MBF = 4, GI = 1, MBI = 8, MBG = 5 }; };
template <> struct ZPlan<256> { enum { R1 = 4, R2 = 8, R3 = 8, T = 32, G = 1, GF = 1, MBF = 3, GI = 1, MBI = 4, MBG = 3 }; };

__device__ __forceinline__ double2 ld2(const double* p) { return *reinterpret_cast<const double2*>(p); }
__device__ __forceinline__ void st2(double* p, double2 v) { *reinterpret_cast<double2*>(p) = v; }

// closure + forward z.  One tile per CTA.  Stage-in with 16-byte loads (two adjacent z points of both half lines
// per thread, two such quads in flight), closure, packing u_m = (c_m - i c_{m+n/2}) exp(-i pi m / n) into the
// shared-memory tile, then the n/2-point complex line FFTs.
// DYN: the damping follows the residual; the Z slots then hold X_i and the update forms X_i + b R_i from both histories
template <int NZ, int G, int MINB, bool DYN>
__global__ void __launch_bounds__(ZPlan<NZ>::T* G* COLS, MINB)
    closure_zfwd_kernel(double* __restrict__ tau_cur, const double* __restrict__ w, const double* __restrict__ raw,
                        const double* __restrict__ Z, const double* __restrict__ Rh, cplx* __restrict__ work,
                        Twiddle tw_shift, Twiddle tw, const DevState* __restrict__ st, int nv, size_t npts, size_t field,
                        int closure, int order) {
  if (raw == nullptr && st->done) return;
  // pending MDIIS update (step 6 of the previous iteration): tau = sum_i c_i Z_i is formed here, on the way in,
  // and written back once, instead of by a separate pass that this kernel would then re-read
  __shared__ int s_ulist[MAX_M];
  __shared__ double s_ucoef[MAX_M];
  __shared__ int s_um;
  __shared__ double s_bdyn;
  if (threadIdx.x == 0) {
    const int m = raw ? 0 : st->upd_m;
    s_um = m;
    s_bdyn = st->b_dyn;
    for (int i = 0; i < m; ++i) { s_ulist[i] = st->upd_list[i]; s_ucoef[i] = st->upd_coef[i]; }
  }
  __syncthreads();
  const int um = s_um;
  const double bdyn = s_bdyn;
  using Cfg = ZPlan<NZ>;
  constexpr int T = Cfg::T, R1 = Cfg::R1, R2 = Cfg::R2, R3 = Cfg::R3, C = COLS, n = 2 * NZ;
  constexpr int NT = T * G * C, HP = NZ / 2, U = 2;
  const int tid = threadIdx.x;
  const int LP = C / nv, GL = G * LP;                 // lines per column group, lines per CTA
  const size_t line0 = (size_t)blockIdx.x * GL;
  const double* tau = raw ? raw : tau_cur;
  const int total = GL * nv * HP;

  for (int e0 = tid; e0 < total; e0 += U * NT) {
    double2 t0[U], t1[U], w0[U], w1[U];
    size_t off[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int e = e0 + u * NT;
      if (e < total) {
        const int mp = e % HP, lc = e / HP;
        const int site = lc / GL, l = lc % GL;
        off[u] = (size_t)site * npts + (line0 + l) * n + 2 * mp;
        if (um == 0) {
          t0[u] = ld2(tau + off[u]);
          t1[u] = ld2(tau + off[u] + NZ);
        } else {
          // products and sums rounded one by one, in the order of the oracle's loop (Eq. 40 as read in Q7)
          double2 a0 = make_double2(0.0, 0.0), a1 = make_double2(0.0, 0.0);
#pragma unroll 5
          for (int k = 0; k < um; ++k) {
            const double* Zk = Z + (size_t)s_ulist[k] * field + off[u];
            double2 z0 = __ldcs(reinterpret_cast<const double2*>(Zk));
            double2 z1 = __ldcs(reinterpret_cast<const double2*>(Zk + NZ));
            if constexpr (DYN) {                       // X_i + b R_i with the current b, rounded as the oracle's expression
              const double* Rk = Rh + (size_t)s_ulist[k] * field + off[u];
              const double2 r0 = __ldcs(reinterpret_cast<const double2*>(Rk));
              const double2 r1 = __ldcs(reinterpret_cast<const double2*>(Rk + NZ));
              z0 = make_double2(__dadd_rn(z0.x, __dmul_rn(bdyn, r0.x)), __dadd_rn(z0.y, __dmul_rn(bdyn, r0.y)));
              z1 = make_double2(__dadd_rn(z1.x, __dmul_rn(bdyn, r1.x)), __dadd_rn(z1.y, __dmul_rn(bdyn, r1.y)));
            }
            const double ck = s_ucoef[k];
            a0.x = __dadd_rn(a0.x, __dmul_rn(ck, z0.x));
            a0.y = __dadd_rn(a0.y, __dmul_rn(ck, z0.y));
            a1.x = __dadd_rn(a1.x, __dmul_rn(ck, z1.x));
            a1.y = __dadd_rn(a1.y, __dmul_rn(ck, z1.y));
          }
          t0[u] = a0;
          t1[u] = a1;
          st2(tau_cur + off[u], a0);
          st2(tau_cur + off[u] + NZ, a1);
        }
        if (!raw) {
          w0[u] = ld2(w + off[u]);
          w1[u] = ld2(w + off[u] + NZ);
        }
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int e = e0 + u * NT;
      if (e < total) {
        const int mp = e % HP, lc = e / HP;
        const int site = lc / GL, l = lc % GL;
        double2 c0 = t0[u], c1 = t1[u];
        if (!raw) {                                    // g = closure(w + tau), c_sr = g - 1 - tau  (Eq. 15-16, 31)
          c0.x = closure_g(w0[u].x + t0[u].x, closure, order) - 1.0 - t0[u].x;
          c0.y = closure_g(w0[u].y + t0[u].y, closure, order) - 1.0 - t0[u].y;
          c1.x = closure_g(w1[u].x + t1[u].x, closure, order) - 1.0 - t1[u].x;
          c1.y = closure_g(w1[u].y + t1[u].y, closure, order) - 1.0 - t1[u].y;
        }
        cplx* tile = smem_dyn + (l / LP) * (NZ * ZP) + (l % LP) * nv + site;
        tile[(2 * mp) * ZP] = cmul(make_double2(c0.x, -c1.x), tw_shift(2 * mp));
        tile[(2 * mp + 1) * ZP] = cmul(make_double2(c0.y, -c1.y), tw_shift(2 * mp + 1));
      }
    }
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
  using Cfg = ZPlan<NZ>;
  constexpr int G = ZPlan<NZ>::GF;
  const int LP = COLS / gr.nv, GL = G * LP;
  const size_t nlines = (size_t)gr.nxl * gr.ny;
  const int threads = Cfg::T * G * COLS;
  const size_t shm = (size_t)G * NZ * ZP * sizeof(cplx);
  auto kern = sp.dyn_b ? closure_zfwd_kernel<NZ, G, ZPlan<NZ>::MBF, true> : closure_zfwd_kernel<NZ, G, ZPlan<NZ>::MBF, false>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shm) != cudaSuccess) return 0;
  const int ez = gr.nmax / gr.nz;
  Twiddle tws{b.tw, ez, 2 * gr.nmax - 1}, tw{b.tw, 2 * ez, 2 * gr.nmax - 1};
  kern<<<(unsigned)(nlines / GL), threads, shm, s>>>(b.tau, b.w, raw, b.Z, b.R, b.work, tws, tw, b.state, gr.nv,
                                                       gr.npts, gr.field, sp.closure, sp.pse_order);
  return 1;
}

int launch_closure_zfwd(const Grid& g, const Buffers& b, const SolverParams& sp, const double* raw, cudaStream_t s) {
  int k = 0;
  switch (g.nz / 2) {
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

// inverse z + residual.  One tile per CTA: inverse line FFTs in shared memory, the last stage leaves
// (f_m, f_{m+n/2}) in place of complex element m, then a streaming phase with 16-byte accesses forms R = tau' - tau
// (Eq. 33) and Z = tau + b R (the form Eq. 40 needs this entry in) and stores both into history slot `cur`.
// MAXO >= 0: the Gram row <R, R_i> over the (at most MAXO = M - 1) stored residuals is accumulated in the streaming
// phase as well, and the kernel ends with the partial-sum reduction and the MDIIS solve (mdiis_device.cuh).
// MAXO = -1: transform only (debug hook, raw_out).
struct GramArgs {
  double* part1;
  double* part2;
  unsigned* tickets;
  const double* weight;  // [nv] weights 1/rho_g of the modified Anderson inner product (Eq. 38); unused otherwise
  double n_values;       // grid points x site types of the caller: the N n_v of Eq. 41 (phantom types do not count)
  AccelArgs aa;
  GramExchange xr;       // slab runs: where this rank's row goes (mdiis_device.cuh)
};

template <int NZ, int G, int MINB, int MAXO, bool WEIGHTED>
__global__ void __launch_bounds__(ZPlan<NZ>::T* G* COLS, MINB)
    zinv_residual_kernel(const cplx* __restrict__ work, const double* __restrict__ tau_cur, double* __restrict__ Z,
                         double* __restrict__ R, double* __restrict__ raw_out, Twiddle tw_shift, Twiddle tw,
                         DevState* __restrict__ st, int nv, size_t npts, size_t field, double bdamp, GramArgs ga) {
  if (raw_out == nullptr && st->done) return;
  constexpr bool GRAM = (MAXO >= 0);
  constexpr int NACC = GRAM ? MAXO + 1 : 1;
  __shared__ int s_other[MAX_M];
  __shared__ int s_nother, s_m, s_flag;
  __shared__ double s_row[MAX_M + 2];
  __shared__ SolveScratch s_solve;
  if (GRAM && threadIdx.x == 0) {
    const int m = st->m;
    const int skip = (m == ga.aa.M) ? 1 : 0;              // a full history drops its oldest entry this iteration
    s_nother = m - skip;
    s_m = m;
    for (int i = 0; i < m - skip; ++i) s_other[i] = st->list[i + skip];
  }
  using Cfg = ZPlan<NZ>;
  constexpr int T = Cfg::T, R1 = Cfg::R1, R2 = Cfg::R2, R3 = Cfg::R3, C = COLS, n = 2 * NZ;
  constexpr int NT = T * G * C;
  constexpr int HP = NZ / 2;                           // pairs (m, m+1) per half line
  const int tid = threadIdx.x;
  const int LP = C / nv, GL = G * LP;
  cplx* smc = smem_dyn;                                // [G][NZ][ZP] complex
  const int cur = raw_out ? 0 : st->cur;

  const int col = tid % C, t = (tid / C) % T, grp = tid / (C * T);
  cplx* sm = smc + grp * (NZ * ZP) + col;
  auto ld_sm = [&](int i) { return sm[i * ZP]; };
  auto st_sm = [&](int i, cplx v) { sm[i * ZP] = v; };
  const double scale = 1.0 / (double)NZ;
  const size_t line0 = (size_t)blockIdx.x * GL;
  {
    const size_t line = line0 + (size_t)grp * LP + col / nv;
    const cplx* src = work + line * NZ * nv + (col % nv);
    auto in = [&](int p, int) { return src[(size_t)p * nv]; };
    if constexpr (R3 == 1) {
      inv_stage_first<NZ, R2, R1>(t, T, tw, false, in, st_sm);
      __syncthreads();
    } else {
      inv_stage_first<NZ, (R3 == 1 ? R2 : R3), R1>(t, T, tw, false, in, st_sm);
      __syncthreads();
      inv_stage_mid<NZ, R1, R2, false>(t, T, tw, ld_sm, st_sm);
      __syncthreads();
    }
    // u_m exp(+i pi m/n) / NZ = f_m - i f_{m+n/2}; every thread rewrites exactly the elements it has just read
    auto out = [&](int m, cplx v) {
      const cplx f = cscale(cmulc(v, tw_shift(m)), scale);
      sm[m * ZP] = make_double2(f.x, -f.y);
    };
    inv_stage_last<NZ, R1, false>(t, T, tw, ld_sm, out);
  }
  __syncthreads();

  const double* Xc = tau_cur;
  double* Rc = raw_out ? nullptr : R + (size_t)cur * field;
  double* Zc = raw_out ? nullptr : Z + (size_t)cur * field;
  const int nother = GRAM ? s_nother : 0;              // (written before the barriers of the transform)
  double acc[NACC], acc_u = 0.0;                        // acc_u: unweighted <R, R> of a weighted run (for the rms)
#pragma unroll
  for (int j = 0; j < NACC; ++j) acc[j] = 0.0;

  // streaming phase: thread <-> (site, line, pair of adjacent z points); 16-byte accesses, z fastest
  for (int e = tid; e < GL * nv * HP; e += NT) {
    const int mp = e % HP, lc = e / HP;
    const int site = lc / GL, l = lc % GL;
    const size_t off = (size_t)site * npts + (line0 + l) * n + 2 * mp;
    const cplx* tile = smc + (l / LP) * (NZ * ZP) + (l % LP) * nv + site;
    const cplx a = tile[(2 * mp) * ZP], b = tile[(2 * mp + 1) * ZP];
    const double2 tlo = make_double2(a.x, b.x), thi = make_double2(a.y, b.y);   // tau' at off.., off+NZ..
    if (raw_out) {
      st2(raw_out + off, tlo);
      st2(raw_out + off + NZ, thi);
    } else {
      const double2 xlo = ld2(Xc + off), xhi = ld2(Xc + off + NZ);
      const double2 rlo = make_double2(tlo.x - xlo.x, tlo.y - xlo.y);          // R = tau' - tau  (Eq. 33)
      const double2 rhi = make_double2(thi.x - xhi.x, thi.y - xhi.y);
      st2(Rc + off, rlo);
      st2(Rc + off + NZ, rhi);
      // Z = X + b R (Eq. 40 / Q7); mul and add rounded separately, as the oracle's X[i] + b*R[i]
      st2(Zc + off, make_double2(__dadd_rn(xlo.x, __dmul_rn(bdamp, rlo.x)), __dadd_rn(xlo.y, __dmul_rn(bdamp, rlo.y))));
      st2(Zc + off + NZ, make_double2(__dadd_rn(xhi.x, __dmul_rn(bdamp, rhi.x)), __dadd_rn(xhi.y, __dmul_rn(bdamp, rhi.y))));
      if constexpr (GRAM) {
        // weighted inner product (modified Anderson, Eq. 38): one side of every product carries the weight of this
        // element's site; the unweighted <R, R> is kept as well, for the rms
        double2 vlo = rlo, vhi = rhi;
        if constexpr (WEIGHTED) {
          const double wg = ga.weight[site];
          vlo = make_double2(wg * rlo.x, wg * rlo.y);
          vhi = make_double2(wg * rhi.x, wg * rhi.y);
          acc_u = fma(rlo.x, rlo.x, fma(rlo.y, rlo.y, fma(rhi.x, rhi.x, fma(rhi.y, rhi.y, acc_u))));
        }
        acc[MAXO] = fma(vlo.x, rlo.x, fma(vlo.y, rlo.y, fma(vhi.x, rhi.x, fma(vhi.y, rhi.y, acc[MAXO]))));
#pragma unroll
        for (int j = 0; j < MAXO; ++j)
          if (j < nother) {
            const double* Rj = R + (size_t)s_other[j] * field + off;
            const double2 qlo = __ldcs(reinterpret_cast<const double2*>(Rj));
            const double2 qhi = __ldcs(reinterpret_cast<const double2*>(Rj + NZ));
            acc[j] = fma(vlo.x, qlo.x, fma(vlo.y, qlo.y, fma(vhi.x, qhi.x, fma(vhi.y, qhi.y, acc[j]))));
          }
      }
    }
  }
  if constexpr (GRAM) {
    // per-thread fp64 sums (<= 64 elements each) -> double-double across the warp (fixed tree) and the warps
    __syncthreads();                                   // the tile is dead: its memory holds the warp sums
    double* s_part = reinterpret_cast<double*>(smem_dyn);
    constexpr int NW = NT / 32;
    const int lane = tid & 31, wid = tid >> 5;
#pragma unroll
    for (int j = 0; j <= MAXO + 1; ++j) {              // j = MAXO + 1: the unweighted self product
      if (j < nother || j == MAXO || (j == MAXO + 1 && WEIGHTED)) {
        double hi = (j <= MAXO) ? acc[j < NACC ? j : 0] : acc_u, lo = 0.0;
        for (int o = 16; o > 0; o >>= 1) {
          const double h2 = __shfl_down_sync(0xffffffffu, hi, o), l2 = __shfl_down_sync(0xffffffffu, lo, o);
          dd_add(hi, lo, h2, l2);
        }
        if (lane == 0) {
          s_part[(j * NW + wid) * 2] = hi;
          s_part[(j * NW + wid) * 2 + 1] = lo;
        }
      }
    }
    __syncthreads();
    if (tid <= MAXO + 1 && (tid < nother || tid == MAXO || (tid == MAXO + 1 && WEIGHTED))) {
      double hi = 0.0, lo = 0.0;
      for (int w = 0; w < NW; ++w) dd_add(hi, lo, s_part[(tid * NW + w) * 2], s_part[(tid * NW + w) * 2 + 1]);
      dd_norm(hi, lo);
      const int j = (tid < MAXO) ? tid : (tid == MAXO ? MAX_M : MAX_M - 1);
      *reinterpret_cast<double2*>(ga.part1 + ((size_t)j * gridDim.x + blockIdx.x) * 2) = make_double2(hi, lo);
      __threadfence();
    }
    gram_finish<NT>(st, ga.part1, ga.part2, ga.tickets, s_m, nother, ga.aa, WEIGHTED, ga.n_values, s_row, &s_flag, s_solve,
                    ga.xr);
  }
}

static AccelArgs accel_args(const SolverParams& sp) {
  return AccelArgs{sp.M, sp.restart, sp.accel, sp.and_s1, sp.and_s2, sp.b_min, sp.dyn_b ? sp.b_max : 0.0};
}
static GramExchange gram_exchange(const Grid& gr, const Buffers& b) {
  GramExchange xr{};
  xr.rank = gr.rank;
  xr.n_dst = gr.n_ranks > 1 ? b.n_gram_dst : 0;
  for (int d = 0; d < xr.n_dst; ++d) xr.dst[d] = b.gram_dst[d];
  return xr;
}

template <int NZ, int MAXO, bool WEIGHTED>
static int launch_zinv_nm(const Grid& gr, const Buffers& b, const SolverParams& sp, double* raw_out, cudaStream_t s) {
  using Cfg = ZPlan<NZ>;
  constexpr int G = ZPlan<NZ>::GI;
  constexpr int MB = (MAXO >= 0) ? ZPlan<NZ>::MBG : ZPlan<NZ>::MBI;
  const int LP = COLS / gr.nv, GL = G * LP;
  const int threads = Cfg::T * G * COLS;
  size_t shm = (size_t)G * NZ * ZP * sizeof(cplx);
  const size_t red = (size_t)(MAX_M + 2) * (threads / 32 + 1) * 2 * sizeof(double);
  if (shm < red) shm = red;
  auto kern = zinv_residual_kernel<NZ, G, MB, MAXO, WEIGHTED>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shm) != cudaSuccess) return 0;
  const int ez = gr.nmax / gr.nz;
  Twiddle tws{b.tw, ez, 2 * gr.nmax - 1}, tw{b.tw, 2 * ez, 2 * gr.nmax - 1};
  GramArgs ga{b.gram_part, b.gram_part2, b.tickets, b.gram_w, (double)gr.npts_global * gr.nv_user, accel_args(sp),
              gram_exchange(gr, b)};
  // (dynamic damping: the Z slot takes X itself -- X + 0 R is exact -- and the update applies the current b)
  kern<<<(unsigned)((size_t)gr.nxl * gr.ny / GL), threads, shm, s>>>(b.work, b.tau, b.Z, b.R, raw_out, tws, tw, b.state,
                                                                   gr.nv, gr.npts, gr.field, sp.dyn_b ? 0.0 : sp.b, ga);
  return 1;
}

// raw_out != nullptr: transform only; otherwise the variant compiled for M - 1 stored residuals
template <int NZ>
static int launch_zinv_n(const Grid& gr, const Buffers& b, const SolverParams& sp, double* raw_out, cudaStream_t s) {
  if (raw_out) return launch_zinv_nm<NZ, -1, false>(gr, b, sp, raw_out, s);
  if (sp.accel == RISM3D_ACCEL_ANDERSON) return launch_zinv_nm<NZ, 2, true>(gr, b, sp, raw_out, s);   // 3 stored pairs
  // compiled for a few history sizes only (each bounds the unrolled Gram loop); M - 1 rounds up to the next one
  const int mo = sp.M - 1;
  if (mo <= 0) return launch_zinv_nm<NZ, 0, false>(gr, b, sp, raw_out, s);
  if (mo <= 2) return launch_zinv_nm<NZ, 2, false>(gr, b, sp, raw_out, s);
  if (mo <= 4) return launch_zinv_nm<NZ, 4, false>(gr, b, sp, raw_out, s);
  if (mo <= 7) return launch_zinv_nm<NZ, 7, false>(gr, b, sp, raw_out, s);
  if (mo <= 9) return launch_zinv_nm<NZ, 9, false>(gr, b, sp, raw_out, s);
  return launch_zinv_nm<NZ, MAX_M - 1, false>(gr, b, sp, raw_out, s);
}

template <int NZ>
static int zinv_ctas_n(const Grid& gr) {
  const int LP = COLS / gr.nv, GL = ZPlan<NZ>::GI * LP;
  return (int)((size_t)gr.nxl * gr.ny / GL);
}
int zinv_ctas(const Grid& g) {
  switch (g.nz / 2) {
    case 4: return zinv_ctas_n<4>(g);
    case 8: return zinv_ctas_n<8>(g);
    case 16: return zinv_ctas_n<16>(g);
    case 32: return zinv_ctas_n<32>(g);
    case 64: return zinv_ctas_n<64>(g);
    case 128: return zinv_ctas_n<128>(g);
    case 256: return zinv_ctas_n<256>(g);
    default: return 0;
  }
}

int launch_zinv_residual(const Grid& g, const Buffers& b, const SolverParams& sp, double* raw_out, cudaStream_t s) {
  int k = 0;
  switch (g.nz / 2) {
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

// ------------------------------------------------------------------------------------------------
// Slab-decomposed runs: the second half of the MDIIS step.  gram_x holds one row of double-double totals per rank
// (written by the last-arriving CTA of every rank's zinv_residual, moved by the caller's all-gather or stored straight
// into the peers' arrays); one warp adds them in rank order and runs the same bookkeeping and solve as a single rank.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(32)
    gram_solve_kernel(DevState* __restrict__ st, const double* __restrict__ gram_x, int n_ranks, AccelArgs aa,
                      int weighted, double n_values) {
  if (st->done) return;
  __shared__ SolveScratch s_solve;
  __shared__ double s_row[MAX_M + 2];
  const int lane = threadIdx.x;
  const int m = st->m;
  const int nother = m - ((m == aa.M) ? 1 : 0);          // as zinv_residual saw it: a full history drops its oldest entry
  const int nent = nother + (weighted ? 2 : 1);
  if (lane < nent) {
    double hi = 0.0, lo = 0.0;
    for (int r = 0; r < n_ranks; ++r) {
      const double2 p = __ldcg(reinterpret_cast<const double2*>(gram_x) + (size_t)r * GRAM_SLOT + lane);
      dd_add(hi, lo, p.x, p.y);
    }
    s_row[lane] = hi + lo;
  }
  __syncwarp();
  mdiis_bookkeeping_and_solve(st, s_solve, s_row, m, nother, aa, weighted ? s_row[nother + 1] : s_row[nother], n_values);
}

// the same for any array of double-double rows [n_rows][GRAM_SLOT][2] (the 1D solver's per-CTA partial sums)
int launch_gram_solve_rows(DevState* st, const double* rows, int n_rows, const SolverParams& sp, double n_values,
                           cudaStream_t s) {
  gram_solve_kernel<<<1, 32, 0, s>>>(st, rows, n_rows, accel_args(sp), sp.accel == RISM3D_ACCEL_ANDERSON ? 1 : 0, n_values);
  return 1;
}

int launch_gram_solve(const Grid& gr, const Buffers& b, const SolverParams& sp, cudaStream_t s) {
  gram_solve_kernel<<<1, 32, 0, s>>>(b.state, b.gram_x, gr.n_ranks, accel_args(sp), sp.accel == RISM3D_ACCEL_ANDERSON ? 1 : 0,
                                     (double)gr.npts_global * gr.nv_user);
  return 1;
}

// In-stream barrier across the ranks of a peer-mapped slab run: every rank stores its next epoch into slot `rank` of
// every rank's flag array (release, system scope: the stores of the kernels before it in the stream are visible to
// whoever sees the flag) and waits until all slots of its own array have reached that epoch.  All ranks enqueue the same
// sequence of kernels, so epochs agree without any host involvement; the kernel is graph-capturable.
// The wait is BOUNDED: a rank that never arrives (its process died, it enqueued fewer barriers, its context was
// re-created without a new rism3d_slab_set_peers on every rank) would otherwise leave the others spinning inside a
// kernel for ever.  After timeout_ns without all arrivals the function gives up and returns false.
struct FlagPtrs { unsigned long long* p[MAX_RANKS]; };

__device__ __forceinline__ unsigned long long global_timer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;\n" : "=l"(t));
  return t;
}

// one warp per rank (blockDim.x == 32); `mine` = this rank's [MAX_RANKS + 1] flags (the last entry is its epoch counter)
__device__ __forceinline__ bool xbarrier_arrive_and_wait(unsigned long long* mine, const FlagPtrs& peers, int n_ranks,
                                                         int rank, unsigned long long timeout_ns) {
  const int lane = threadIdx.x;
  unsigned long long epoch = 0;
  if (lane == 0) {
    epoch = mine[MAX_RANKS] + 1;
    mine[MAX_RANKS] = epoch;
  }
  epoch = __shfl_sync(0xffffffffu, epoch, 0);
  __threadfence_system();
  bool ok = true;
  if (lane < n_ranks) {
    asm volatile("st.release.sys.global.u64 [%0], %1;\n" ::"l"(peers.p[lane] + rank), "l"(epoch) : "memory");
    const unsigned long long t0 = global_timer_ns();
    unsigned spins = 0;
    for (;;) {
      unsigned long long seen;
      asm volatile("ld.acquire.sys.global.u64 %0, [%1];\n" : "=l"(seen) : "l"(mine + lane) : "memory");
      if (seen >= epoch) break;
      if ((++spins & 63u) == 0u && global_timer_ns() - t0 > timeout_ns) { ok = false; break; }
    }
  }
  return __all_sync(0xffffffffu, ok);
}

// On a timeout the rank's solver state is marked: done = 1 makes every later loop kernel of the call return at once,
// status = RISM3D_ERR_PEER is what rism3d_iterate reports; later barriers of the same call do not wait again (the epochs
// of the ranks no longer agree: the run has to be reconnected with rism3d_slab_set_peers on every rank).
__global__ void __launch_bounds__(32)
    xbarrier_kernel(unsigned long long* __restrict__ mine, FlagPtrs peers, int n_ranks, int rank, DevState* st,
                    unsigned long long timeout_ns) {
  if (st->status == RISM3D_ERR_PEER) return;
  const bool ok = xbarrier_arrive_and_wait(mine, peers, n_ranks, rank, timeout_ns);
  if (!ok && threadIdx.x == 0) {
    st->status = RISM3D_ERR_PEER;
    st->done = 1;
  }
}

int launch_xbarrier(const Grid& gr, const Buffers& b, cudaStream_t s) {
  FlagPtrs fp{};
  for (int r = 0; r < gr.n_ranks; ++r) fp.p[r] = b.flag_dst[r];
  xbarrier_kernel<<<1, 32, 0, s>>>(b.xflags, fp, gr.n_ranks, gr.rank, b.state, b.peer_timeout_ns);
  return 1;
}

// Self-test of the barrier on ONE GPU (rism3d_debug_peer_barrier_selftest).  Kernels that wait on one another must not be
// run as separate launches on one device -- nothing guarantees that they are resident together -- so the ranks are the
// blocks of one cooperative launch: block r is rank r, with its own flag array in `flags` ([n_ranks][MAX_RANKS + 1],
// zero on entry), and runs the same xbarrier_arrive_and_wait as the production kernel `epochs` times.  Before barrier e
// rank r publishes data[r] = e * 1000 + r with a plain store; after it, every rank must see at least that value from
// every other rank (the release / acquire pair orders it).  absent_rank >= 0: that block leaves at once, every other
// rank must give up within timeout_ns and reports it.  result[0] += ordering errors, result[1] += ranks that timed out.
__global__ void __launch_bounds__(32)
    xbarrier_selftest_kernel(unsigned long long* flags, volatile unsigned long long* data, int* result, int n_ranks,
                             int epochs, int absent_rank, unsigned long long timeout_ns) {
  const int rank = blockIdx.x, lane = threadIdx.x;
  if (rank == absent_rank) return;
  FlagPtrs fp{};
  for (int r = 0; r < n_ranks; ++r) fp.p[r] = flags + (size_t)r * (MAX_RANKS + 1);
  for (int e = 1; e <= epochs; ++e) {
    if (lane == 0) data[rank] = (unsigned long long)e * 1000ull + rank;
    __syncwarp();
    if (!xbarrier_arrive_and_wait(fp.p[rank], fp, n_ranks, rank, timeout_ns)) {
      if (lane == 0) atomicAdd(result + 1, 1);
      return;
    }
    if (lane < n_ranks) {
      const unsigned long long v = data[lane];
      if (v < (unsigned long long)e * 1000ull + lane || v % 1000ull != (unsigned long long)lane) atomicAdd(result, 1);
    }
    __syncwarp();
  }
}

// d_scratch: >= 4096 bytes, zeroed here on `s`; h_result[2] (pinned or pageable) receives (errors, timeouts) after a sync
cudaError_t run_xbarrier_selftest(void* d_scratch, int n_ranks, int epochs, int absent_rank, unsigned long long timeout_ns,
                                  int h_result[2], cudaStream_t s) {
  cudaError_t e = cudaMemsetAsync(d_scratch, 0, 4096, s);
  if (e != cudaSuccess) return e;
  unsigned long long* flags = (unsigned long long*)d_scratch;                       // 8 x 9 x 8 = 576 bytes
  unsigned long long* data = flags + (size_t)MAX_RANKS * (MAX_RANKS + 1);            // 64 bytes
  int* result = (int*)(data + MAX_RANKS);
  void* args[] = {&flags, &data, &result, &n_ranks, &epochs, &absent_rank, &timeout_ns};
  e = cudaLaunchCooperativeKernel((const void*)xbarrier_selftest_kernel, dim3(n_ranks), dim3(32), args, 0, s);
  if (e != cudaSuccess) return e;
  e = cudaMemcpyAsync(h_result, result, 2 * sizeof(int), cudaMemcpyDeviceToHost, s);
  if (e != cudaSuccess) return e;
  return cudaStreamSynchronize(s);
}

}  // namespace r3d
