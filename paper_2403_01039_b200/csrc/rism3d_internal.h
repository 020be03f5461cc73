// rism3d_internal.h -- shared declarations of the CUDA side of librism3d.so (not part of the ABI).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/rism3d.h"

namespace r3d {

constexpr int MAX_M = 16;            // MDIIS history slots (rism3d_params.mdiis_nvec <= 16)
constexpr int MAX_NV = 8;            // solvent site types
constexpr int RMS_HIST_CAP = 65536;
constexpr int FE_BLOCKS = 148 * 4;        // CTAs of the free-energy reduction
constexpr int MAX_RANKS = 8;              // processes of a slab-decomposed run (rism3d_params.n_ranks)
constexpr int GRAM_SLOT = MAX_M + 2;      // double-double Gram entries one rank hands to the others per iteration

constexpr double K_BOLTZMANN = 0.001987204259;   // kcal/(mol K)     (Q3)
constexpr double COULOMB = 332.06371;            // kcal A/(mol e^2) (Q3)

// Device-resident solver state: the whole MDIIS bookkeeping lives on the GPU so that an iteration is a
// fixed sequence of launches (graph-capturable) and `iterate` never has to synchronise per iteration.
struct DevState {
  // ---- header: the first 64 bytes are what rism3d_iterate copies back to the host ----
  int done;                    // 1: converged or diverged -> all loop kernels return immediately
  int status;                  // rism3d_status
  int n_done;                  // iterations completed by the current rism3d_iterate call
  int hist_n;                  // total iterations since set_solute
  int m;                       // filled history entries
  int cur;                     // physical history slot that receives the (Z, R) pair of the running iteration
  int upd_m;                   // entries to combine in the update kernel (0: skip)
  unsigned ticket;             // first-level group adders of the Gram reduction that have finished
  double tol;
  double rms_last;
  double b_dyn;                // damping of the pending update when it follows the residual (SolverParams.dyn_b)
  double pad_[1];
  // ---- MDIIS bookkeeping ----
  int list[MAX_M];             // physical slot of each entry, oldest first
  int upd_list[MAX_M];
  double upd_coef[MAX_M];
  double S[MAX_M][MAX_M];      // Gram matrix of the stored residuals, indexed like `list`
  double rms[MAX_M];           // rms of each entry
  double rms_hist[RMS_HIST_CAP];
};
struct StateHeader {           // mirrors the first 64 bytes of DevState
  int done, status, n_done, hist_n, m, cur, upd_m; unsigned ticket;
  double tol, rms_last, b_dyn, pad_[1];
};

struct Grid {
  int nx, ny, nz;        // points per axis of the WHOLE grid: powers of two, one spacing (the box need not be cubic)
  int nmax;              // the largest of the three: the twiddle table and the |k| shell table are built for it
  int wx, wy, wz;        // (nmax / n_axis)^2: with dk0 = 2 pi / (nmax h), |k|^2 = dk0^2 (s + (wx + wy + wz) / 4),
                         // s = sum_axis w_axis j'(j' + 1) an even integer (j' the folded index): shell index s / 2
  int nshell;            // entries of the shell table: largest s / 2, plus one
  int nv;                // site types as the kernels see them: nv_user rounded up to a power of two (1, 2, 4, 8); the
                         // extra "phantom" types have zero charge, LJ, density and chi, stay exactly 0 and cost bandwidth only
  int nv_user;           // site types of the caller (rism3d_params.n_sites)
  double h;              // spacing
  double origin[3];      // position of grid point (0, 0, 0) of the whole grid
  // slab decomposition over n_ranks processes (n_ranks = 1: this context holds the whole grid).  r space and the z / y
  // passes: planes ix0 .. ix0 + nxl - 1;  the k-space pass (x lines): rows jy0 .. jy0 + nyl - 1.
  int n_ranks, rank;
  int nxl, ix0;
  int nyl, jy0;
  size_t npts;           // r-space points of THIS context: nxl * ny * nz
  size_t field;          // nv * npts doubles in one field-set
  size_t npts_global;    // nx * ny * nz
  int num_sms;           // SMs of the device the context lives on (grid size of the persistent kernels)
  int smem_optin;        // largest dynamic shared memory a kernel may opt in to on that device, bytes
  __host__ __device__ size_t q() const { return (size_t)(nz / 2) * nv; }   // complex elements per (ix, iy) row of `work`
};

// Device pointers carved from the caller's workspace.
struct Buffers {
  DevState* state;
  double* Z;             // [M][field]   MDIIS history: Z_i = X_i + b R_i (the only form Eq. 40 needs X_i in)
  double* R;             // [M][field]   MDIIS residuals R_i = Y_i - X_i
  double* tau;           // [field]      current input X (tau = t - f)
  double* w;             // [field]      -beta u + f
  double2* work;         // [nxl][ny][nz/2][nv] complex   k-space work array (x lines: [nx][nyl][nz/2][nv])
  double* phi;           // [npts]       phi(r)
  double2* phik;         // [nx][nyl][nz/2]  phi~(k) exp(+i k.r0) / dV
  double* chi_shell;     // [nshell][nv][nv]   chi_shell[s][g][k] = chi_{(g xor k) g}(k_s)
  double2* tw;           // [2 nmax]     exp(-i pi j / nmax)
  double* gram_part;     // [MAX_M+1][gram_blocks][2]  double-double partial sums, one per zinv_residual CTA
  double* gram_part2;    // [MAX_M+1][groups][2]  first-level sums of groups of 64 partials
  unsigned* tickets;     // [groups] arrival counters of the partial-sum reduction (zero between launches)
  size_t n_tickets;
  double* scratch;       // [field] temporary (get_field, setup tables); aliases `work`
  double* qv;            // [nv] solvent charges
  double* rhov;          // [nv]
  double* gram_w;        // [nv] weights of the inner product: 1 (MDIIS) or 1/rho_g (modified Anderson, Eq. 38)
  double* fe_part;       // [FE_BLOCKS][MAX_NV][2]
  // ---- slab decomposition (n_ranks > 1; with one rank kbuf == work and the tables are unused) ----
  double2* kbuf;         // [nx][nyl][nz/2][nv] complex   this rank's k-space slab: x lines complete
  double2* stage;        // [n_ranks][nxl][nyl][nz/2][nv] staging buffer of the two transposes when a library collective
                         // moves the blocks (rism3d_slab_local); unused once rism3d_slab_set_peers has been called
  double* gram_x;        // [n_ranks][GRAM_SLOT][2]  every rank's double-double Gram row, summed in rank order by the solve
  unsigned long long* xflags;   // [MAX_RANKS + 1] arrival epochs of the in-stream barrier (peer mode) + this rank's epoch counter
  double2* fwd_dst[MAX_RANKS];        // y_fwd writes the rows j_y of rank d's slab of plane ix_l to fwd_dst[d] + (ix_l nyl + jy_l) Q
  const double2* bwd_src[MAX_RANKS];  // y_inv reads them back from bwd_src[s] + (ix_l nyl + jy_l) Q
  double* gram_dst[MAX_RANKS];        // copies of gram_x this rank writes its slot into (itself; every peer in peer mode)
  unsigned long long* flag_dst[MAX_RANKS];   // peer mode: xflags of every rank
  int n_gram_dst;
  bool peer_mode;
  unsigned long long peer_timeout_ns;        // longest wait of one in-stream barrier (rism3d_slab_set_peer_timeout)
  // TMA descriptors of the k-space pass (built by rism3d_init when kspace_uses_tma(n)): `work` as a 2D array of doubles
  // [jx][2 n Q] with boxes of n rows x 128 bytes, `phik` as [jx][2 n n/2] with boxes of n rows x (8 / nv) complex
  CUtensorMap tm_work, tm_phik;
  // the y passes (single-rank runs, ny = 64, 128, 256): `work` as [nxl * ny][2 Q] doubles, boxes of ny rows x 128 bytes
  CUtensorMap tm_ywork;
};

struct SolverParams {
  int closure;           // rism3d_closure
  int pse_order;
  int M;
  double b;
  double restart;
  double beta, kT, kappa, r_min;
  bool dyn_b;            // damping follows the residual, b = clamp(-0.2 log10 rms, b_min, b_max); the history then holds X_i
  double b_min, b_max;   //   in the Z slots (stored with b = 0) and the update forms X_i + b R_i from both fields
  int accel;             // rism3d_accelerator (ANDERSON: M = 3 stored pairs = the newest + two histories)
  double and_s1, and_s2; // tuning parameters of Eq. 34-35
};

// dynamic shared memory of kspace_x for this grid (0: unsupported n / nv); the API layer checks it against the device
int kspace_smem_bytes(int nx, int nv);
bool kspace_uses_tma(int nx);
bool y_uses_tma(int ny, int n_ranks);
int y_tile_cols(const Grid&);

// ---- launchers (each returns the number of kernels it launched; errors surface via cudaGetLastError) ----
// fft_kernels.cu
int launch_closure_zfwd(const Grid&, const Buffers&, const SolverParams&, const double* d_raw_in, cudaStream_t);
int launch_y_fwd(const Grid&, const Buffers&, bool use_state, cudaStream_t);   // slab runs: writes through fwd_dst
int launch_x_fwd(const Grid&, const Buffers&, cudaStream_t);
int launch_x_inv(const Grid&, const Buffers&, cudaStream_t);
int launch_kspace_x(const Grid&, const Buffers&, cudaStream_t);
int launch_y_inv(const Grid&, const Buffers&, bool use_state, cudaStream_t);   // slab runs: reads through bwd_src
int launch_gram_solve(const Grid&, const Buffers&, const SolverParams&, cudaStream_t);   // slab runs: sum the ranks' rows, solve
int launch_gram_solve_rows(DevState*, const double* rows, int n_rows, const SolverParams&, double n_values, cudaStream_t);
int launch_xbarrier(const Grid&, const Buffers&, cudaStream_t);                // peer mode: all ranks have reached this point
cudaError_t run_xbarrier_selftest(void* d_scratch, int n_ranks, int epochs, int absent_rank, unsigned long long timeout_ns,
                                  int h_result[2], cudaStream_t);
int launch_zinv_residual(const Grid&, const Buffers&, const SolverParams&, double* d_raw_out, cudaStream_t);
int zinv_ctas(const Grid&);                      // CTAs of zinv_residual (it writes one Gram partial per CTA)
// mdiis_kernels.cu
int launch_mdiis_update(const Grid&, const Buffers&, const SolverParams&, cudaStream_t);
// setup_kernels.cu
int launch_chi_shell(const Grid&, const Buffers&, const double* d_chi_table, int n_k, double k0, double dk,
                     cudaStream_t);
int launch_potential(const Grid&, const Buffers&, const SolverParams&, int n_atoms, const double* d_atoms,
                     const double* d_pair, double rcut, cudaStream_t);
int launch_w_cells(const Grid&, const Buffers&, const SolverParams&, const double* d_atoms, const double* d_pair,
                   const int* d_cell_start, const int nc[3], const double lo[3], double edge, double rcut, cudaStream_t);
int launch_phi(const Grid&, const Buffers&, const SolverParams&, int n_atoms, const double* d_atoms, cudaStream_t);
int launch_phi_tilde(const Grid&, const Buffers&, const SolverParams&, int n_atoms, const double* d_atoms,
                     double2* d_phase, cudaStream_t);
int launch_gradient(const Grid&, const Buffers&, const SolverParams&, int n_atoms, double* d_gw, const double* d_atoms,
                    const double* d_pair, double* d_partial, int nchunks, double* d_out, cudaStream_t);
double measure_dfma_peak(int num_sms, double* d_scratch, cudaStream_t);
int launch_free_energy(const Grid&, const Buffers&, const SolverParams&, double* d_out, cudaStream_t);
int launch_get_field(const Grid&, const Buffers&, const SolverParams&, int which, int site, double* d_dst,
                     cudaStream_t);

// double-double helpers (used by the Gram and free-energy reductions)
__device__ __forceinline__ void dd_add_prod(double& hi, double& lo, double a, double b) {
  const double p = __dmul_rn(a, b);        // kept out of FMA contraction: the error-free split needs the rounded product
  const double e = __fma_rn(a, b, -p);
  const double s = hi + p;
  const double bb = s - hi;
  const double err = (hi - (s - bb)) + (p - bb);
  hi = s;
  lo += err + e;
}
__device__ __forceinline__ void dd_add(double& hi, double& lo, double h2, double l2) {
  const double s = hi + h2;
  const double bb = s - hi;
  const double err = (hi - (s - bb)) + (h2 - bb);
  hi = s;
  lo += err + l2;
}
__device__ __forceinline__ void dd_norm(double& hi, double& lo) {
  const double s = hi + lo;
  lo = lo - (s - hi);
  hi = s;
}

// Sum of `count` double-double partials part[i * stride], i < count, by ONE warp, in a fixed order: lane l adds l, l + 32, ...,
// then the shuffle tree.  Result (hi, lo) in lane 0.
__device__ __forceinline__ void warp_sum_partials(const double* part, int count, int lane, double& hi, double& lo,
                                                  int stride = 1) {
  hi = 0.0;
  lo = 0.0;
  for (int i = lane; i < count; i += 32) {
    const double2 p = __ldcg(reinterpret_cast<const double2*>(part) + (size_t)i * stride);
    dd_add(hi, lo, p.x, p.y);
  }
  for (int o = 16; o > 0; o >>= 1) {
    const double h2 = __shfl_down_sync(0xffffffffu, hi, o), l2 = __shfl_down_sync(0xffffffffu, lo, o);
    dd_add(hi, lo, h2, l2);
  }
}

// closure g(d) (Q1, Q2): HNC exp(d); KH/PSE-n: exp(d) for d <= 0, sum_{i<=n} d^i/i! for d > 0
__device__ __forceinline__ double closure_g(double d, int closure, int order) {
  if (closure == RISM3D_HNC) return exp(d);
  if (d > 0.0) {
    // Horner form 1 + d/1 (1 + d/2 (1 + ... (1 + d/n))), every product and sum rounded separately (as the oracle's
    // numpy expression); orders 1 and 2 need no division (x/1 and x/2 are exact as x and 0.5 x)
    if (order == 1) return __dadd_rn(1.0, d);
    if (order == 2) return __dadd_rn(1.0, __dmul_rn(__dadd_rn(1.0, __dmul_rn(d, 0.5)), d));
    double s = 1.0;
    for (int i = order; i >= 1; --i) s = __dadd_rn(1.0, __ddiv_rn(__dmul_rn(s, d), (double)i));
    return s;
  }
  return exp(d);
}

}  // namespace r3d
