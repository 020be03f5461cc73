// kspace_kernel.cu -- steps 3b-5a of the loop in ONE pass over the k-space work array:
//   forward FFT along x  ->  c(k) = c_sr(k) - q_g phi~(k)          (Eq. 32)
//                        ->  h_g(k) = sum_g' c_g'(k) chi_g'g(|k|)   (Eq. 13)
//                        ->  tau'(k) = h(k) - c_sr(k)               (Eq. 33 in k space; Q14)
//                        ->  inverse FFT along x, in place.
// The last forward pass and the first inverse stage work on the same register set (decimation in frequency
// forward, decimation in time inverse), so the k-space arithmetic happens in registers between them; the n_v
// sites of one k point sit in n_v adjacent lanes (site-interleaved layout) and are exchanged by warp shuffles.
// chi(|k|) comes from the per-shell table built in set_solvent_chi: |k|^2 = dk^2 (s + 3/4) with
// s = sum_axis j'(j'+1), j' the folded index.
#include "async_copy.cuh"
#include "fft_core.cuh"
#include "rism3d_internal.h"
#include "tma.cuh"

namespace r3d {

extern __shared__ __align__(128) double2 smem_dyn[];
constexpr int COLS = 8;

// geometry of the k-space slab this context transforms along x: work is [nx][nyl][nzh][nv] complex, row jy_l stands for
// j_y = jy0 + jy_l of the whole grid (nyl = ny, jy0 = 0 without a slab decomposition)
struct KGeom {
  int nzh;               // nz / 2 stored j_z = 2p
  int nyl, jy0;
  int ny, nz;            // whole-grid lengths: folded index j' = j < n/2 ? j : n - 1 - j
  int wx, wy, wz;        // weights of the shell index (Grid)
  __device__ __forceinline__ int s_yz(int jy_l, int p) const {
    const int jy = jy0 + jy_l;
    const int jyf = 2 * jy < ny ? jy : ny - 1 - jy;
    const int jzf = 4 * p < nz ? 2 * p : nz - 1 - 2 * p;
    return wy * jyf * (jyf + 1) + wz * jzf * (jzf + 1);
  }
};
static KGeom make_kgeom(const Grid& g) { return KGeom{g.nz / 2, g.nyl, g.jy0, g.ny, g.nz, g.wx, g.wy, g.wz}; }

// shared-memory layout of one pipeline stage: [G][N][COLS] data tile, then [G][N][COLS/NV] phi~ values
template <int N, int NV>
struct KspaceCfg {
  enum { NT = FftCfg<N>::T * FftCfg<N>::G * COLS,
         ITEM = FftCfg<N>::G * N * COLS,                  // complex data elements per work item
         PHI = FftCfg<N>::G * N * (COLS / NV),            // phi~ values per work item
         STAGE = ITEM + PHI,
         MIDT = (FftCfg<N>::R3 == 1) ? 0 : (N / FftCfg<N>::R1 / FftCfg<N>::R2) * FftCfg<N>::R2,   // mid-pass twiddle table
         SHM = (2 * STAGE + MIDT) * (int)sizeof(cplx),
         MINB = (SHM > 110 * 1024) ? 1 : ((SHM > 72 * 1024) ? 2 : 3) };
};

// Eq. 32 + Eq. 13 + Eq. 33 (in k space) for ONE k point, the NV sites of which sit in NV adjacent lanes:
//   c = c_sr - q_g phi~ ;  h_g = sum_g' c_g' chi_g'g ;  returns tau'(k) = h_g - c_sr.
// ch: this lane's row of the per-shell table, chi_shell[shell][g][k] = chi_{(g xor k) g}: entry k multiplies the c of
// lane (g xor k), so the own value needs no shuffle and the others come by NV - 1 butterfly exchanges.
template <int NV>
__device__ __forceinline__ cplx kspace_point(cplx csr, cplx ph, double qg, const double* __restrict__ ch) {
  const cplx c = make_double2(csr.x - qg * ph.x, csr.y - qg * ph.y);          // Eq. 32
  double chv[NV];                                                             // one 8*NV-byte row, 16-byte loads
  if constexpr (NV == 1) {
    chv[0] = __ldg(ch);
  } else {
#pragma unroll
    for (int i = 0; i < NV / 2; ++i) {
      const double2 v = __ldg(reinterpret_cast<const double2*>(ch) + i);
      chv[2 * i] = v.x;
      chv[2 * i + 1] = v.y;
    }
  }
  double hx = c.x * chv[0], hy = c.y * chv[0];
#pragma unroll
  for (int k = 1; k < NV; ++k) {
    const double cx = __shfl_xor_sync(0xffffffffu, c.x, k);
    const double cy = __shfl_xor_sync(0xffffffffu, c.y, k);
    hx = fma(cx, chv[k], hx);                                                  // Eq. 13
    hy = fma(cy, chv[k], hy);
  }
  return make_double2(hx - csr.x, hy - csr.y);                                // tau'(k) = h - c_sr
}

template <int N, int NV>
__device__ __forceinline__ void stage_kspace(cplx* buf, const cplx* data, const cplx* phik, const KGeom& kg, size_t item,
                                             int tid) {
  using Cfg = FftCfg<N>;
  using K = KspaceCfg<N, NV>;
  constexpr int C = COLS, PC = C / NV;
  const size_t Q = (size_t)kg.nzh * NV, ES = (size_t)kg.nyl * Q;
#pragma unroll
  for (int k = 0; k < K::ITEM / K::NT; ++k) {
    const int idx = tid + k * K::NT;
    const int grp = idx / (N * C), rem = idx % (N * C), row = rem / C, col = rem % C;
    const size_t chunk = item * Cfg::G + grp;
    cp_async16(buf + idx, data + chunk * C + (size_t)row * ES + col);
  }
#pragma unroll
  for (int k = 0; k < (K::PHI + K::NT - 1) / K::NT; ++k) {
    const int idx = tid + k * K::NT;
    if (idx < K::PHI) {
      const int grp = idx / (N * PC), rem = idx % (N * PC), row = rem / PC, c = rem % PC;
      const size_t q2 = (item * Cfg::G + grp) * C;       // flattened (jy_l, p, site) of the tile's first column
      const size_t jy = q2 / Q, p0 = (q2 % Q) / NV;
      cp_async16(buf + K::ITEM + idx, phik + ((size_t)row * kg.nyl + jy) * kg.nzh + p0 + c);
    }
  }
}

template <int N, int NV>
__global__ void __launch_bounds__(KspaceCfg<N, NV>::NT, KspaceCfg<N, NV>::MINB)
    kspace_x_kernel(cplx* __restrict__ data, const cplx* __restrict__ phik, const double* __restrict__ chi_shell,
                    const double* __restrict__ qv, Twiddle tw, const DevState* __restrict__ st, KGeom kg, unsigned nitems) {
  if (st->done) return;
  using Cfg = FftCfg<N>;
  using K = KspaceCfg<N, NV>;
  constexpr int T = Cfg::T, R1 = Cfg::R1, R2 = Cfg::R2, R3 = Cfg::R3, C = COLS;
  constexpr int RL = (R3 == 1) ? R2 : R3;            // radix of the innermost digit
  constexpr int NB = N / RL, RMID = NB / R1;
  constexpr int NZ = N / 2, PC = C / NV;             // NZ: folding point of the x index
  const size_t Q = (size_t)kg.nzh * NV;              // complex elements per (jx, jy) row
  const size_t ES = (size_t)kg.nyl * Q;              // stride of the x axis
  const int tid = threadIdx.x;
  const int col = tid % C, t = (tid / C) % T, grp = tid / (C * T);
  const int site = col % NV;
  const double qg = qv[site];
  // this thread's twiddles are the same for every tile: pass-A set in registers, middle-pass set in a shared table
  using Tw = LineTw<N, R1, R2, R3, T, false>;
  cplx* mid_table = smem_dyn + 2 * K::STAGE;
  Tw::fill_mid_table(mid_table, tw, tid, K::NT);
  Tw w;
  w.init(t, tw, mid_table);
  int b = 0;
  size_t item = blockIdx.x;
  if (item < nitems) stage_kspace<N, NV>(smem_dyn, data, phik, kg, item, tid);
  cp_async_commit();
  for (; item < nitems; item += gridDim.x) {
    const size_t next = item + gridDim.x;
    if (next < nitems) stage_kspace<N, NV>(smem_dyn + (b ^ 1) * K::STAGE, data, phik, kg, next, tid);
    cp_async_commit();
    cp_async_wait<1>();
    __syncthreads();
    cplx* sm = smem_dyn + b * K::STAGE + grp * (N * C) + col;
    const cplx* sph = smem_dyn + b * K::STAGE + K::ITEM + grp * (N * PC) + col / NV;
    const size_t q2 = (item * Cfg::G + grp) * C + col;   // flattened (jy, p, site)
    cplx* base = data + q2;
    const int s_yz = kg.s_yz((int)(q2 / Q), (int)((q2 % Q) / NV));   // folded indices: |k_axis| = dk (j' + 1/2)
    auto ld_sm = [&](int i) { return sm[i * C]; };
    auto st_sm = [&](int i, cplx v) { sm[i * C] = v; };

    fwd_a_c(t, w, tw, ld_sm, st_sm);
    __syncthreads();
    if constexpr (R3 != 1) {
      fwd_mid_c(t, w, ld_sm, st_sm);
      __syncthreads();
    }
    // innermost digit: forward DFT, k-space arithmetic, inverse DFT, all on the same registers
    for (int blk = t; blk < NB; blk += T) {
      cplx x[RL];
#pragma unroll
      for (int m = 0; m < RL; ++m) x[m] = ld_sm(blk * RL + m);
      Dft<RL, -1>::run(x);
      const int k1 = blk / RMID, k2 = blk % RMID;
      const int j0 = k1 + R1 * k2;
#pragma unroll
      for (int k = 0; k < RL; ++k) {
        const int jx = j0 + NB * k;
        const int jxf = jx < NZ ? jx : N - 1 - jx;
        const int shell = (kg.wx * jxf * (jxf + 1) + s_yz) >> 1;
        x[k] = kspace_point<NV>(x[k], sph[jx * PC], qg, chi_shell + (size_t)shell * (NV * NV) + site * NV);
      }
      Dft<RL, +1>::run(x);                             // first inverse stage; its twiddles are applied by the loads of the next
#pragma unroll
      for (int r = 0; r < RL; ++r) st_sm(blk * RL + r, x[r]);
    }
    __syncthreads();
    if constexpr (R3 != 1) {
      inv_mid_c(t, w, ld_sm, st_sm);
      __syncthreads();
    }
    const double scale = 1.0 / (double)N;
    inv_last_c(t, w, tw, ld_sm, [&](int m, cplx v) { base[m * ES] = cscale(v, scale); });
    __syncthreads();                                   // stage b is free again
    b ^= 1;
  }
}

// ------------------------------------------------------------------------------------------------
// Two-pass variant for the line lengths that factor into two radices <= 32 (64 = 8 x 8, 128 = 16 x 8, 256 = 16 x 16,
// 512 = 32 x 16):
// half the shared-memory passes of the three-pass plan (3 loads + 2 stores of the tile per work item instead of 5 + 5),
// which is what bounds this kernel (L1 / shared data pipe).  T = N / R1 threads per column, one
// radix-R1 butterfly each in the outer passes; the pass-A twiddles exp(-2 pi i (k1 + 1/2) t / N), k1 = 0..R1-1, are a
// geometric sequence in k1 and are generated from two seeds per thread instead of being held in 4 R1 registers.
// One tile (N x 8 complex = 128-byte rows) per CTA at a time, single-buffered: several small CTAs per SM overlap
// their load, arithmetic and store phases with each other.
// ------------------------------------------------------------------------------------------------
template <int N> struct KPlan2 { enum { OK = 0, R1 = 1, R2 = 1, STAGES = 2 }; };
template <> struct KPlan2<64>  { enum { OK = 1, R1 = 8,  R2 = 8,  STAGES = 2 }; };
template <> struct KPlan2<128> { enum { OK = 1, R1 = 16, R2 = 8,  STAGES = 2 }; };
template <> struct KPlan2<256> { enum { OK = 1, R1 = 16, R2 = 16, STAGES = 2 }; };
// 512 = 32 x 16: the 64 KB tile is single-buffered so that two CTAs fit on an SM and overlap each other's load,
// arithmetic and store phases
template <> struct KPlan2<512> { enum { OK = 1, R1 = 32, R2 = 16, STAGES = 1 }; };

constexpr int TMA_BOX_ROWS = 256;                           // a TMA box holds at most 256 elements per dimension

template <int N, int NV>
struct Kspace2Cfg {
  enum { R1 = KPlan2<N>::R1, R2 = KPlan2<N>::R2, STAGES = KPlan2<N>::STAGES, T = N / R1, NT = T * COLS,
         ITEM = N * COLS, PHI = N * (COLS / NV),
         TILE_BYTES = ITEM * (int)sizeof(cplx), PHI_BYTES = PHI * (int)sizeof(cplx),
         STAGE = ITEM + PHI,                                // complex elements of one pipeline stage: tile, then phi~
         SHM = STAGES * (TILE_BYTES + PHI_BYTES) + 64,      // the stages and their mbarriers
         BOX_ROWS = N < TMA_BOX_ROWS ? N : TMA_BOX_ROWS, NBOX = N / BOX_ROWS,
         FIT = 227 * 1024 / (SHM + 1024), CAP = (N >= 256) ? 2 : 8,   // long lines want all 255 registers
         MINB = FIT < CAP ? FIT : CAP };
};

// L2 policy of the chi gathers: keep the shell table resident (evict_last) under the streaming tiles -- at 512^3 the
// table is 12.5 MB and, without the hint, a tenth of the pass's DRAM reads were table rows coming back
__device__ __forceinline__ uint64_t l2_keep_policy() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;\n" : "=l"(pol));
  return pol;
}

template <int NV>
struct ChiRow {
  double v[NV];
  __device__ __forceinline__ void load(const double* __restrict__ ch, uint64_t pol) {
    if constexpr (NV == 1) {
      v[0] = __ldg(ch);
    } else if constexpr (NV == 2) {
      const double2 t = __ldg(reinterpret_cast<const double2*>(ch));
      v[0] = t.x;
      v[1] = t.y;
    } else {
      // 32-byte rows: one 256-bit load each (sm_100: LDG.E.256), half the requests of two 128-bit loads
#pragma unroll
      for (int i = 0; i < NV / 4; ++i)
        asm volatile("ld.global.nc.L2::cache_hint.v4.f64 {%0, %1, %2, %3}, [%4], %5;\n"
                     : "=d"(v[4 * i]), "=d"(v[4 * i + 1]), "=d"(v[4 * i + 2]), "=d"(v[4 * i + 3])
                     : "l"(ch + 4 * i), "l"(pol));
    }
  }
};

template <int NV>
__device__ __forceinline__ cplx kspace_point_row(cplx csr, cplx ph, double qg, const ChiRow<NV>& row) {
  const cplx c = make_double2(csr.x - qg * ph.x, csr.y - qg * ph.y);          // Eq. 32
  double hx = c.x * row.v[0], hy = c.y * row.v[0];
#pragma unroll
  for (int k = 1; k < NV; ++k) {
    const double cx = __shfl_xor_sync(0xffffffffu, c.x, k);
    const double cy = __shfl_xor_sync(0xffffffffu, c.y, k);
    hx = fma(cx, row.v[k], hx);                                                // Eq. 13
    hy = fma(cy, row.v[k], hy);
  }
  return make_double2(hx - csr.x, hy - csr.y);                                // tau'(k) = h - c_sr
}

template <int N, int NV>
__global__ void __launch_bounds__(Kspace2Cfg<N, NV>::NT, Kspace2Cfg<N, NV>::MINB)
    kspace2_kernel(const __grid_constant__ CUtensorMap tm_work, const __grid_constant__ CUtensorMap tm_phik,
                   cplx* __restrict__ work, const double* __restrict__ chi_shell, const double* __restrict__ qv, Twiddle tw,
                   const DevState* __restrict__ st, KGeom kg, unsigned nitems) {
  if (st->done) return;
  using K = Kspace2Cfg<N, NV>;
  constexpr int R1 = K::R1, R2 = K::R2, T = K::T, C = COLS;
  constexpr int S1 = N / R1, NB = N / R2;            // S1 == T: one pass-A butterfly per thread
  constexpr int NZ = N / 2, PC = C / NV;             // NZ: folding point of the x index
  const unsigned Q = (unsigned)kg.nzh * NV;          // complex elements per (jx, jy) row
  constexpr int PFMAX = (NV > 4) ? 4 : 8;            // chi rows in flight per thread (a row is NV doubles)
  constexpr int PF = (R2 < PFMAX) ? R2 : PFMAX;
  const int tid = threadIdx.x;
  const int col = tid % C, t = tid / C;
  const int site = col % NV;
  const double qg = qv[site];
  const cplx a0 = tw(t), astep = tw(2 * t);          // exp(-i pi t / N) and its square: a[k1] = a0 * astep^k1
  constexpr int STAGES = K::STAGES;
  cplx* stages = smem_dyn;                           // [STAGES] x ([N][8] tile, [N][8 / NV] phi~)
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem_dyn + STAGES * K::STAGE);   // one per stage
  const double scale = 1.0 / (double)N;
  const uint64_t chi_policy = l2_keep_policy();
  // the boxes of work item `it` into stage b; TMA coordinates: innermost = doubles along the flattened (jy, p[, site])
  auto issue = [&](unsigned it, int b) {
    const unsigned q0 = it * C;
    mbar_arrive_expect_tx(&bars[b], K::TILE_BYTES + K::PHI_BYTES);
#pragma unroll
    for (int bx = 0; bx < K::NBOX; ++bx) {
      tma_load_2d(stages + b * K::STAGE + bx * K::BOX_ROWS * C, &tm_work, (int)(q0 * 2), bx * K::BOX_ROWS, &bars[b]);
      tma_load_2d(stages + b * K::STAGE + K::ITEM + bx * K::BOX_ROWS * PC, &tm_phik,
                  (int)((q0 / Q * kg.nzh + (q0 % Q) / NV) * 2), bx * K::BOX_ROWS, &bars[b]);
    }
  };
  if (tid == 0) {
#pragma unroll
    for (int b = 0; b < STAGES; ++b) mbar_init(&bars[b], 1);
    mbar_fence_init();
  }
  __syncthreads();
  unsigned item = blockIdx.x;
  if (tid == 0 && item < nitems) issue(item, 0);
  unsigned n_done = 0;
  for (; item < nitems; item += gridDim.x, ++n_done) {
    const int b = (STAGES == 2) ? (int)(n_done & 1) : 0;
    const unsigned next = item + gridDim.x;
    if constexpr (STAGES == 2) {
      if (tid == 0 && next < nitems) {
        tma_wait_read();                             // the store of the previous item has left stage b ^ 1
        issue(next, b ^ 1);
      }
    }                                                // (one stage: the next tile is requested inside the last pass)
    cplx* sm = stages + b * K::STAGE + col;
    const cplx* sph = stages + b * K::STAGE + K::ITEM + col / NV;
    auto ld_sm = [&](int i) { return sm[i * C]; };
    auto st_sm = [&](int i, cplx v) { sm[i * C] = v; };
    const unsigned q2 = item * C + col;              // flattened (jy, p, site)
    const int s_yz = kg.s_yz((int)(q2 / Q), (int)((q2 % Q) / NV));   // folded indices: |k_axis| = dk (j' + 1/2)
    auto chi_row = [&](int jx) {
      const int jxf = jx < NZ ? jx : N - 1 - jx;
      return chi_shell + (size_t)((kg.wx * jxf * (jxf + 1) + s_yz) >> 1) * (NV * NV) + site * NV;
    };
    mbar_wait(&bars[b], (STAGES == 2) ? ((n_done >> 1) & 1) : (n_done & 1));

    {                                                // forward pass A: radix R1 over m1, half-integer shift, twiddle
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
    // inner digit: forward DFT, k-space arithmetic, inverse DFT, all on the same registers; the chi rows of the next
    // PF k points are in flight while one is used
    for (int blk = t; blk < NB; blk += T) {
      ChiRow<NV> ring[PF];
#pragma unroll
      for (int k = 0; k < PF; ++k) ring[k].load(chi_row(blk + NB * k), chi_policy);
      cplx x[R2];
#pragma unroll
      for (int m = 0; m < R2; ++m) x[m] = ld_sm(blk * R2 + m);
      Dft<R2, -1>::run(x);
#pragma unroll
      for (int k = 0; k < R2; ++k) {
        const int jx = blk + NB * k;
        x[k] = kspace_point_row<NV>(x[k], sph[jx * PC], qg, ring[k % PF]);
        if (k + PF < R2) ring[k % PF].load(chi_row(blk + NB * (k + PF)), chi_policy);
      }
      Dft<R2, +1>::run(x);
#pragma unroll
      for (int r = 0; r < R2; ++r) st_sm(blk * R2 + r, x[r]);
    }
    __syncthreads();
    {                                                // inverse last stage: conjugate twiddle, radix R1 over k1, shift
      cplx x[R1];
      const PassATw<R1> a(a0, astep);
#pragma unroll
      for (int k1 = 0; k1 < R1; ++k1) x[k1] = cmulc(ld_sm(k1 * S1 + t), a.get(k1));
      if constexpr (STAGES == 1) {
        // single-buffered tiles (n = 512): once every thread holds its values the stage is free -- the next tile is
        // requested now and lands under this pass's arithmetic; the results leave from registers (128-byte rows).
        // The stage was last written with ordinary st.shared (pass B): order those generic-proxy writes before the
        // async-proxy write of the TMA load (a CTA barrier alone does not order the two proxies in the PTX model)
        fence_proxy_async();
        __syncthreads();
        if (tid == 0 && next < nitems) issue(next, 0);
      }
      Dft<R1, +1>::run(x);
      HalfShiftAll<R1, +1>::run(x);
      if constexpr (STAGES == 1) {
        cplx* dst = work + (size_t)item * C + col;
        const size_t ES = (size_t)kg.nyl * Q;          // stride of the x axis
#pragma unroll
        for (int m1 = 0; m1 < R1; ++m1) dst[(size_t)(m1 * S1 + t) * ES] = cscale(x[m1], scale);
      } else {
#pragma unroll
        for (int m1 = 0; m1 < R1; ++m1) st_sm(m1 * S1 + t, cscale(x[m1], scale));   // in place: the slots this thread read
      }
    }
    if constexpr (STAGES == 2) {
      fence_proxy_async();
      __syncthreads();
      if (tid == 0) {
#pragma unroll
        for (int bx = 0; bx < K::NBOX; ++bx)
          tma_store_2d(&tm_work, (int)(item * C * 2), bx * K::BOX_ROWS, stages + b * K::STAGE + bx * K::BOX_ROWS * C);
        tma_commit();
      }
    }
  }
  if (STAGES == 2 && tid == 0) tma_wait_all();
}

template <int N, int NV>
static int launch_kspace2_nv(const Grid& gr, const Buffers& b, cudaStream_t s) {
  using K = Kspace2Cfg<N, NV>;
  const unsigned nitems = (unsigned)((size_t)gr.nyl * gr.q() / COLS);
  auto kern = kspace2_kernel<N, NV>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)K::SHM) != cudaSuccess) return 0;
  Twiddle tw{b.tw, gr.nmax / N, 2 * gr.nmax - 1};
  unsigned grid = (unsigned)(gr.num_sms * K::MINB);
  if (grid > nitems) grid = nitems;
  kern<<<grid, K::NT, K::SHM, s>>>(b.tm_work, b.tm_phik, b.kbuf, b.chi_shell, b.qv, tw, b.state, make_kgeom(gr), nitems);
  return 1;
}

// true when launch_kspace_x takes the TMA path for this grid (the API layer then builds the tensor maps)
bool kspace_uses_tma(int n) {
  switch (n) {
    case 64: return KPlan2<64>::OK;
    case 128: return KPlan2<128>::OK;
    case 256: return KPlan2<256>::OK;
    case 512: return KPlan2<512>::OK;
    default: return false;
  }
}

template <int N, int NV>
static int launch_kspace_nv(const Grid& gr, const Buffers& b, cudaStream_t s) {
  using Cfg = FftCfg<N>;
  using K = KspaceCfg<N, NV>;
  const size_t nchunks = (size_t)gr.nyl * gr.q() / COLS;
  const unsigned nitems = (unsigned)(nchunks / Cfg::G);
  auto kern = kspace_x_kernel<N, NV>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)K::SHM) != cudaSuccess) return 0;
  Twiddle tw{b.tw, gr.nmax / N, 2 * gr.nmax - 1};
  unsigned grid = (unsigned)(gr.num_sms * K::MINB);
  if (grid > nitems) grid = nitems;
  kern<<<grid, K::NT, K::SHM, s>>>(b.kbuf, b.phik, b.chi_shell, b.qv, tw, b.state, make_kgeom(gr), nitems);
  return 1;
}

template <int N, int NV>
static int launch_kspace_pick(const Grid& g, const Buffers& b, cudaStream_t s) {
  if constexpr (KPlan2<N>::OK) return launch_kspace2_nv<N, NV>(g, b, s);
  else return launch_kspace_nv<N, NV>(g, b, s);
}

template <int N>
static int launch_kspace_n(const Grid& g, const Buffers& b, cudaStream_t s) {
  switch (g.nv) {
    case 1: return launch_kspace_pick<N, 1>(g, b, s);
    case 2: return launch_kspace_pick<N, 2>(g, b, s);
    case 4: return launch_kspace_pick<N, 4>(g, b, s);
    case 8: return launch_kspace_pick<N, 8>(g, b, s);
    default: return 0;
  }
}

int launch_kspace_x(const Grid& g, const Buffers& b, cudaStream_t s) {
  switch (g.nx) {
    case 8: return launch_kspace_n<8>(g, b, s);
    case 16: return launch_kspace_n<16>(g, b, s);
    case 32: return launch_kspace_n<32>(g, b, s);
    case 64: return launch_kspace_n<64>(g, b, s);
    case 128: return launch_kspace_n<128>(g, b, s);
    case 256: return launch_kspace_n<256>(g, b, s);
    case 512: return launch_kspace_n<512>(g, b, s);
    default: return 0;
  }
}

template <int N, int NV>
static constexpr int kspace_smem_nv() {
  if constexpr (KPlan2<N>::OK) return Kspace2Cfg<N, NV>::SHM;
  else return KspaceCfg<N, NV>::SHM;
}
template <int N>
static int kspace_smem_n(int nv) {
  switch (nv) {
    case 1: return kspace_smem_nv<N, 1>();
    case 2: return kspace_smem_nv<N, 2>();
    case 4: return kspace_smem_nv<N, 4>();
    case 8: return kspace_smem_nv<N, 8>();
    default: return 0;
  }
}

int kspace_smem_bytes(int n, int nv) {
  switch (n) {
    case 8: return kspace_smem_n<8>(nv);
    case 16: return kspace_smem_n<16>(nv);
    case 32: return kspace_smem_n<32>(nv);
    case 64: return kspace_smem_n<64>(nv);
    case 128: return kspace_smem_n<128>(nv);
    case 256: return kspace_smem_n<256>(nv);
    case 512: return kspace_smem_n<512>(nv);
    default: return 0;
  }
}

}  // namespace r3d
