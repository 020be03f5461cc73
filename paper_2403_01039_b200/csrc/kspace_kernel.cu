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

namespace r3d {

extern __shared__ double2 smem_dyn[];
constexpr int COLS = 8;

// shared-memory layout of one pipeline stage: [G][N][COLS] data tile, then [G][N][COLS/NV] phi~ values
template <int N, int NV>
struct KspaceCfg {
  enum { NT = FftCfg<N>::T * FftCfg<N>::G * COLS,
         ITEM = FftCfg<N>::G * N * COLS,                  // complex data elements per work item
         PHI = FftCfg<N>::G * N * (COLS / NV),            // phi~ values per work item
         STAGE = ITEM + PHI,
         MIDT = (FftCfg<N>::R3 == 1) ? 0 : (N / FftCfg<N>::R1 / FftCfg<N>::R2) * FftCfg<N>::R2,   // mid-pass twiddle table
         SHM = (2 * STAGE + MIDT) * (int)sizeof(cplx),
#ifdef R3D_KSPACE_MINB
         MINB = R3D_KSPACE_MINB };
#else
         MINB = (SHM > 110 * 1024) ? 1 : ((SHM > 72 * 1024) ? 2 : 3) };
#endif
};

template <int N, int NV>
__device__ __forceinline__ void stage_kspace(cplx* buf, const cplx* data, const cplx* phik, size_t item, int tid) {
  using Cfg = FftCfg<N>;
  using K = KspaceCfg<N, NV>;
  constexpr int C = COLS, NZ = N / 2, PC = C / NV;
  constexpr size_t Q = (size_t)NZ * NV, ES = (size_t)N * Q;
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
      const size_t q2 = (item * Cfg::G + grp) * C;       // flattened (jy, p, site) of the tile's first column
      const size_t jy = q2 / Q, p0 = (q2 % Q) / NV;
      cp_async16(buf + K::ITEM + idx, phik + (size_t)row * N * NZ + jy * NZ + p0 + c);
    }
  }
}

template <int N, int NV>
__global__ void __launch_bounds__(KspaceCfg<N, NV>::NT, KspaceCfg<N, NV>::MINB)
    kspace_x_kernel(cplx* __restrict__ data, const cplx* __restrict__ phik, const double* __restrict__ chi_shell,
                    const double* __restrict__ qv, Twiddle tw, const DevState* __restrict__ st, unsigned nitems) {
  if (st->done) return;
  using Cfg = FftCfg<N>;
  using K = KspaceCfg<N, NV>;
  constexpr int T = Cfg::T, R1 = Cfg::R1, R2 = Cfg::R2, R3 = Cfg::R3, C = COLS;
  constexpr int RL = (R3 == 1) ? R2 : R3;            // radix of the innermost digit
  constexpr int NB = N / RL, RMID = NB / R1;
  constexpr int NZ = N / 2, PC = C / NV;
  constexpr size_t Q = (size_t)NZ * NV;              // complex elements per (jx, jy) row
  constexpr size_t ES = (size_t)N * Q;               // stride of the x axis
  const int tid = threadIdx.x;
  const int col = tid % C, t = (tid / C) % T, grp = tid / (C * T);
  const int site = col % NV;
  const int lane = tid & 31;
  const int lane0 = lane & ~(NV - 1);
  const double qg = qv[site];
  // this thread's twiddles are the same for every tile: pass-A set in registers, middle-pass set in a shared table
  using Tw = LineTw<N, R1, R2, R3, T, false>;
  cplx* mid_table = smem_dyn + 2 * K::STAGE;
  Tw::fill_mid_table(mid_table, tw, tid, K::NT);
  Tw w;
  w.init(t, tw, mid_table);
  int b = 0;
  size_t item = blockIdx.x;
  if (item < nitems) stage_kspace<N, NV>(smem_dyn, data, phik, item, tid);
  cp_async_commit();
  for (; item < nitems; item += gridDim.x) {
    const size_t next = item + gridDim.x;
    if (next < nitems) stage_kspace<N, NV>(smem_dyn + (b ^ 1) * K::STAGE, data, phik, next, tid);
    cp_async_commit();
    cp_async_wait<1>();
    __syncthreads();
    cplx* sm = smem_dyn + b * K::STAGE + grp * (N * C) + col;
    const cplx* sph = smem_dyn + b * K::STAGE + K::ITEM + grp * (N * PC) + col / NV;
    const size_t q2 = (item * Cfg::G + grp) * C + col;   // flattened (jy, p, site)
    cplx* base = data + q2;
    const int jy = (int)(q2 / Q);
    const int p = (int)((q2 % Q) / NV);
    const int jyf = jy < NZ ? jy : N - 1 - jy;         // folded indices: |k_axis| = dk (j' + 1/2)
    const int jzf = (2 * p) < NZ ? 2 * p : N - 1 - 2 * p;
    const int s_yz = jyf * (jyf + 1) + jzf * (jzf + 1);
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
        const int shell = (jxf * (jxf + 1) + s_yz) >> 1;
        const cplx ph = sph[jx * PC];
        const cplx csr = x[k];
        const cplx c = make_double2(csr.x - qg * ph.x, csr.y - qg * ph.y);     // Eq. 32
        const double* ch = chi_shell + (size_t)shell * (NV * NV) + site * NV;  // chi_{g' site}, g' = 0..NV-1
        double chv[NV];                                                         // one 8*NV-byte row, 16-byte loads
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
        double hx = 0.0, hy = 0.0;
#pragma unroll
        for (int gp = 0; gp < NV; ++gp) {
          const double cx = __shfl_sync(0xffffffffu, c.x, lane0 + gp);
          const double cy = __shfl_sync(0xffffffffu, c.y, lane0 + gp);
          hx += cx * chv[gp];                                                   // Eq. 13
          hy += cy * chv[gp];
        }
        x[k] = make_double2(hx - csr.x, hy - csr.y);                            // tau'(k) = h - c_sr
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

template <int N, int NV>
static int launch_kspace_nv(const Grid& gr, const Buffers& b, cudaStream_t s) {
  using Cfg = FftCfg<N>;
  using K = KspaceCfg<N, NV>;
  const size_t Q = (size_t)(gr.n / 2) * gr.nv;
  const size_t nchunks = (size_t)gr.n * Q / COLS;
  const unsigned nitems = (unsigned)(nchunks / Cfg::G);
  auto kern = kspace_x_kernel<N, NV>;
  cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)K::SHM);
  Twiddle tw{b.tw, 1, 2 * gr.n - 1};
  unsigned grid = (unsigned)resident_ctas(K::MINB);
  if (grid > nitems) grid = nitems;
  kern<<<grid, K::NT, K::SHM, s>>>(b.work, b.phik, b.chi_shell, b.qv, tw, b.state, nitems);
  return 1;
}

template <int N>
static int launch_kspace_n(const Grid& g, const Buffers& b, cudaStream_t s) {
  switch (g.nv) {
    case 1: return launch_kspace_nv<N, 1>(g, b, s);
    case 2: return launch_kspace_nv<N, 2>(g, b, s);
    case 4: return launch_kspace_nv<N, 4>(g, b, s);
    case 8: return launch_kspace_nv<N, 8>(g, b, s);
    default: return 0;
  }
}

int launch_kspace_x(const Grid& g, const Buffers& b, cudaStream_t s) {
  switch (g.n) {
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

}  // namespace r3d
