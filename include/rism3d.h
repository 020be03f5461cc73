/* rism3d.h -- C ABI of the B200-native 3D-RISM solver core (librism3d.so).
 *
 * The library runs the self-consistent 3D-RISM iteration of arxiv 2403.01039 (RISMiCal),
 * PAPER.md:222-254 "numerical procedure", on one GPU in fp64:
 *
 *   setup (once per solute)   w_g(r) = -beta u_g(r) + f_g(r)      Eq. 22 + Eq. 29
 *                             phi~(k), f~_g = q_g phi~             Eq. 30
 *   loop  step 2              g = closure(w + tau),  c_sr = g-1-tau  Eq. 15-16, 31
 *         step 3              c_sr(k) = FFT3D[c_sr] on the half-integer k grid
 *                             c(k) = c_sr(k) - f~(k)                Eq. 32
 *         step 4              h_g(k) = sum_g' c_g'(k) chi_g'g(|k|)  Eq. 13
 *         step 5              tau' = FFT3D^-1[h(k) - c_sr(k)]       Eq. 33
 *         step 6              MDIIS over M stored (tau, R = tau' - tau) pairs  Eq. 40
 *         step 7              rms = sqrt(sum R^2 / (N n_v)) < tol    Eq. 41
 *   post                      solvation free energy                 Eq. 17-18
 *
 * tau_g(r) = t_g(r) - f_g(r) is the short-range part of the paper's iteration variable t = h - c.
 * The readings of the places where the paper is garbled or silent (KH branches, Eq. 40, Eq. 41,
 * PSE-n, chi interpolation, units) are listed in DESIGN.md "Readings" Q1-Q16.
 *
 * Conventions
 *   - Units: Angstrom, e, kcal/mol, K.  k_B = 0.001987204259 kcal/(mol K), Coulomb constant
 *     332.06371 kcal A/(mol e^2).
 *   - Every function returns RISM3D_OK (0) or a negative rism3d_status; nothing throws or aborts.
 *     rism3d_last_error() gives the message of the last failure on that context.
 *   - HOST pointers are borrowed for the duration of the call and copied.  DEVICE pointers are
 *     said so explicitly.  The caller owns the device workspace and the CUDA stream (PyTorch
 *     allocates them); the library owns only its small host-side context.
 *   - All GPU work is enqueued on the stream given to rism3d_init; calls that return host values
 *     synchronise that stream before returning.
 *   - Real 3D fields are laid out [site][ix][iy][iz], iz fastest, n_sites*nx*ny*nz doubles;
 *     grid point (ix,iy,iz) sits at origin + spacing*(ix,iy,iz).
 *     In a slab-decomposed run (rism3d_params.n_ranks > 1) a context holds nx/n_ranks planes: "Slab decomposition".
 *   - There is no CPU fallback: without a CUDA device rism3d_init fails with RISM3D_ERR_CUDA.
 */
#ifndef RISM3D_H
#define RISM3D_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rism3d_ctx rism3d_ctx;   /* opaque; created by rism3d_init, freed by rism3d_destroy */

typedef enum {
  RISM3D_OK            =  0,
  RISM3D_ERR_ARG       = -1,   /* NULL pointer, negative count, unknown enum value                 */
  RISM3D_ERR_SIZE      = -2,   /* an axis not a power of two in 8..512, n_sites outside 1..8, mdiis_nvec outside
                                  1..16, r_min or mdiis_b not positive, (nz/2)*n_sites(padded) not a multiple of 8,
                                  or a slab decomposition the grid does not divide into (rism3d_params.n_ranks) */
  RISM3D_ERR_ORDER     = -3,   /* call out of order (set_solute before set_solvent_chi, ...)       */
  RISM3D_ERR_CHI_RANGE = -4,   /* chi table does not cover the 3D |k| range, or is too coarse      */
  RISM3D_ERR_NEUTRAL   = -5,   /* sum_g rho_g q_g != 0 (1e-12)                                     */
  RISM3D_ERR_WORKSPACE = -6,   /* workspace smaller than rism3d_workspace_bytes()                  */
  RISM3D_ERR_CUDA      = -7,   /* a CUDA call failed; message carries cudaGetErrorString           */
  RISM3D_ERR_DIVERGED  = -8,   /* non-finite residual; tau is left at the last input               */
  RISM3D_ERR_PEER      = -9    /* peer mode: another rank did not reach an in-stream barrier within the wait limit
                                  (rism3d_slab_set_peer_timeout); the iteration was abandoned on this rank          */
} rism3d_status;

typedef enum { RISM3D_KH = 1, RISM3D_PSE = 2, RISM3D_HNC = 3 } rism3d_closure;

/* convergence accelerator: MDIIS with mdiis_nvec stored pairs (Eq. 40), or the paper's modified
 * Anderson method with two histories (Eq. 34-39; three stored pairs, inner product weighted with 1/rho_g) */
typedef enum { RISM3D_ACCEL_MDIIS = 0, RISM3D_ACCEL_ANDERSON = 1 } rism3d_accelerator;

/* which-codes of rism3d_get_field */
typedef enum {
  RISM3D_FIELD_G    = 0,   /* g = closure(w + tau)                                                 */
  RISM3D_FIELD_H    = 1,   /* g - 1                                                                */
  RISM3D_FIELD_C_SR = 2,   /* g - 1 - tau                         (Eq. 31)                         */
  RISM3D_FIELD_T    = 3,   /* t = tau + q_g phi(r)                (the paper's variable)           */
  RISM3D_FIELD_TAU  = 4,   /* the iteration variable as stored                                     */
  RISM3D_FIELD_W    = 5,   /* -beta u + f                                                          */
  RISM3D_FIELD_PHI  = 6    /* phi(r) of Eq. 29 (site argument ignored)                             */
} rism3d_field;

typedef struct {
  int    nx, ny, nz;        /* grid points per axis: each a power of two in 8..512; they may differ (the box
                               need not be a cube), the spacing is the same on all axes                */
  double spacing;           /* grid spacing, A                                                     */
  double origin[3];         /* position of grid index (0,0,0), A                                   */
  int    n_sites;           /* n_v, number of solvent site TYPES, 1..8 (3, 5, 6, 7 run padded to 4 or 8 with
                               phantom types of zero charge, LJ, density and chi: same results, the bandwidth
                               of the padded count)                                                */
  int    closure;           /* rism3d_closure                                                      */
  int    pse_order;         /* n of PSE-n (>= 1; 1 is KH); ignored for KH / HNC                    */
  double temperature;       /* K                                                                   */
  int    mdiis_nvec;        /* M, 1..16 (1 = damped Picard iteration)                              */
  double mdiis_b;           /* damping b of Eq. 40                                                 */
  double mdiis_restart;     /* restart when rms > this * (smallest rms in the history); <= 0: never */
  double kappa;             /* kappa of Eq. 29-30, 1/A (the paper: 1)                              */
  double r_min;             /* distance clamp of the short-range potential, A (Q11)      */
  int    device;            /* CUDA device ordinal                                                 */
  int    accelerator;       /* rism3d_accelerator; ANDERSON ignores mdiis_nvec / mdiis_restart and uses
                               mdiis_b as the mixing parameter b of Eq. 39                         */
  double anderson_s[2];     /* tuning parameters s_1, s_2 of Eq. 34-35 (the paper's GPU code: 0.2, 0)      */
  int    mdiis_dynamic_b;   /* != 0 (MDIIS only): b = -0.2 log10(rms) clamped to [mdiis_b_min, mdiis_b_max] every
                               iteration instead of the static mdiis_b (Q18).  The
                               history then keeps X_i and R_i apart and the update reads both: M more words per
                               grid point, site and iteration                                       */
  double mdiis_b_min, mdiis_b_max;
  int    n_ranks, rank;     /* slab decomposition over n_ranks GPUs, one context per GPU and process (0 or 1: the
                               whole grid on this GPU).  See "Slab decomposition" below.             */
} rism3d_params;

/* Bytes of DEVICE memory the caller must provide to rism3d_init (0 if the parameters are invalid). */
size_t rism3d_workspace_bytes(const rism3d_params* params);

/* Create a context.  d_workspace: DEVICE pointer, 256-byte aligned, `bytes` long, owned by the
 * caller and kept alive until rism3d_destroy.  cuda_stream: a cudaStream_t (NULL = legacy default
 * stream).  Builds the twiddle tables; no field is valid before set_solvent_chi + set_solute. */
int rism3d_init(rism3d_ctx** out, const rism3d_params* params, void* d_workspace, size_t bytes,
                void* cuda_stream);

/* Solvent description (X_g'g = omega_g'g + rho_g' h_g'g from a 1D-RISM solve).
 * HOST arrays.  q, sigma, eps, rho: [n_sites] (rho = number density of the site type, 1/A^3).
 * chi: [n_k][n_sites][n_sites] with chi[m][g'][g] tabulated at k_m = k0 + m*dk (g' is the index
 * summed in Eq. 13).  chi(|k|) is taken from the table by 4-point Lagrange interpolation
 * (Q6), evaluated once per distinct |k| of the grid into a device table. */
int rism3d_set_solvent_chi(rism3d_ctx* ctx, const double* q, const double* sigma, const double* eps,
                           const double* rho, int n_k, double dk, double k0, const double* chi);

/* Solute (Eq. 22).  HOST arrays xyz [n_atoms][3], q, sigma, eps [n_atoms].
 * rcut <= 0: all pairs (the paper's definition); rcut > 0: the short-range remainder
 * -beta [C q q exp(-kappa r)/r + LJ] only counts pairs with r < rcut (Q12); the
 * long-range functions phi, phi~ are never cut.  With rcut > 0 the atoms are binned into cells of edge rcut / 2 and
 * every grid point visits only the cells within reach (same pair set as the plain loop over all atoms with the test
 * r < rcut).  Runs the setup kernels, sets tau = 0 (the paper's
 * initial guess t = f) and clears the MDIIS history.  setup_ms (may be NULL)
 * receives the GPU time of the setup kernels in milliseconds (CUDA events). */
int rism3d_set_solute(rism3d_ctx* ctx, int n_atoms, const double* xyz, const double* q,
                      const double* sigma, const double* eps, double rcut, float* setup_ms);

/* GPU time, in milliseconds, of the deferred phi(r) kernel of the current solute (Eq. 29): with rcut > 0 set_solute
 * computes only what the loop reads (w from a cell list, phi~); phi(r), which is never cut off and costs an all-pairs
 * pass, is computed by the first call that needs it (free_energy, pmv, get_field T / PHI).  0 while it has not run
 * or when set_solute computed it (rcut <= 0). */
int rism3d_phi_ms(rism3d_ctx* ctx, float* ms);

/* Run the loop (single rank, or a slab run in peer mode).  tol <= 0: exactly max_iter iterations.  tol > 0: stop after the first iteration
 * whose rms residual is below tol (tau is then left unchanged by that iteration) or after max_iter.
 * n_done (may be NULL): iterations performed by this call; rms (may be NULL): last residual.
 * Returns RISM3D_ERR_DIVERGED when the residual became non-finite. */
int rism3d_iterate(rism3d_ctx* ctx, int max_iter, double tol, int* n_done, double* rms);

/* Solvation free energy of the current tau (Eq. 18 KH / Eq. 17 HNC / PSE-n, Q2, Q10),
 * kcal/mol.  dmu_site: HOST [n_sites] or NULL. */
int rism3d_free_energy(rism3d_ctx* ctx, double* dmu_total, double* dmu_site);

/* Partial molar volume of the solute (Eq. 19), A^3:
 *   V = k_B T chi_T (1 - sum_g rho_g int c_g(r) dr),
 * chi_t = isothermal compressibility of the pure solvent in A^3 mol/kcal (it comes from the solvent's own RISM
 * solve, like chi).  Plain grid sum; the long-range part -q_g phi(r) of c_g drops out of the density-weighted sum by
 * neutrality, so only c_sr enters.  c_int_site (HOST [n_sites] or NULL) receives dV sum_r c_sr,g(r) in A^3. */
int rism3d_pmv(rism3d_ctx* ctx, double chi_t, double* pmv, double* c_int_site);

/* Pressure-correction term of the solvation free energy (Eq. 21), kcal/mol:  dmu_PC = -P V,  V the partial
 * molar volume of Eq. 19 (returned in *pmv when not NULL, A^3).  chi_t (A^3 mol/kcal) and pressure (the bulk pressure of
 * Eq. 20, kcal/(mol A^3)) are properties of the bulk solvent and come from its own 1D-RISM solve, like chi. */
int rism3d_pressure_correction(rism3d_ctx* ctx, double chi_t, double pressure, double* dmu_pc, double* pmv);

/* Solvent-induced gradient of the free energy on the solute atoms (the equation after Eq. 23;
 * common to HNC and KH):  d(dmu)/dR_a = sum_g rho_g int g_g(r) du_g(r)/dR_a dr,  kcal/(mol A), with u of Eq. 22, all
 * pairs (no cutoff), the distance clamp r_min as in the potential.  grad: HOST [n_atoms][3] of the last set_solute.
 * The force on atom a is minus this.  Uses the k-space work array and the history slot the next iteration overwrites
 * anyway as scratch (no effect on a later iterate). */
int rism3d_gradient(rism3d_ctx* ctx, double* grad);

/* Copy one field of one site (nx*ny*nz doubles, [ix][iy][iz]) to dst; dst_is_device selects a
 * DEVICE or HOST destination. */
int rism3d_get_field(rism3d_ctx* ctx, int which, int site, double* dst, int dst_is_device);

/* Overwrite tau of one site (warm start); clears the MDIIS history. */
int rism3d_set_tau(rism3d_ctx* ctx, int site, const double* src, int src_is_device);

/* rms residual of every iteration since the last set_solute (at most the last 65536), HOST dst. */
int rism3d_get_rms_history(rism3d_ctx* ctx, double* dst, int cap, int* n);

/* Number of kernels the library has launched on this context so far (for bench.py's gpu_launches). */
long long rism3d_launch_count(const rism3d_ctx* ctx);

/* Measured fp64 FMA peak of the context's device in TFLOP/s (2 flops per FMA; a microbenchmark of independent DFMA
 * chains, best of 4 launches, CUDA events): the roofline denominator of the setup kernels (S0) and of
 * rism3d_gradient, which are bound by plain fp64 arithmetic. */
int rism3d_measure_dfma_peak(rism3d_ctx* ctx, double* tflops);

/* Per-kernel GPU time of the loop kernels (CUDA events on the context's stream, one before and one after
 * every kernel of an iteration).  set_profiling(1) clears the sums and switches the events on,
 * set_profiling(0) switches them off; both synchronise the stream.  get_timings synchronises, then writes
 * ms_total[k], k < RISM3D_N_LOOP_KERNELS (HOST, cap >= RISM3D_N_LOOP_KERNELS): the summed milliseconds of
 * loop kernel k over *n_iterations profiled iterations, in launch order (names: rism3d_loop_kernel_name). */
#define RISM3D_N_LOOP_KERNELS 5
int rism3d_set_profiling(rism3d_ctx* ctx, int enable);
/* (SURVEY.md section 8(b) sketched this call as (float*, int); it returns double sums and the iteration count instead, so
 * that a caller can form per-iteration means without a second call.) */
int rism3d_get_timings(rism3d_ctx* ctx, double* ms_total, int cap, long long* n_iterations);
const char* rism3d_loop_kernel_name(int k);             /* static strings; "" when k is out of range */

/* Debug / test hooks: run the shifted 3D transform pair alone on a caller-supplied field.  n_sites below is the PADDED
 * site count (n_sites rounded up to 1, 2, 4 or 8).
 * forward: real DEVICE field [n_sites][nx][ny][nz] -> complex DEVICE spectrum
 *   [jx][jy][p][site] (re, im interleaved), p = 0..nz/2-1 standing for jz = 2p, holding
 *   sum_n f(r_n) exp(-i k_j.(r_n - origin)) with k_j = dk (j + 1/2) per axis (no dV factor).
 * inverse: the exact inverse of that map (includes 1/(nx ny nz)). */
int rism3d_debug_fft_forward(rism3d_ctx* ctx, const double* d_real_in, double* d_spec_out);
int rism3d_debug_fft_inverse(rism3d_ctx* ctx, const double* d_spec_in, double* d_real_out);

/* ---- Slab decomposition over several GPUs ("2D decomposition 3D-FFT"; one level of it) -----------
 *
 * n_ranks = P (a power of two, <= 8; nx/P and ny/P multiples of 8) contexts, one per GPU, share one solve.  Rank r holds
 * the planes ix in [r nx/P, (r+1) nx/P) of every real field ([site][ix_l][iy][iz]; get_field / set_tau move that slab)
 * and runs the closure, the z and the y transforms on them.  The x transform, Eq. 32, Eq. 13 and the inverse x transform
 * need whole x lines: rank r does them for the rows jy in [r ny/P, (r+1) ny/P) of the spectrum, array "K" =
 * complex [jx][jy_l][p][site].  As in the paper (its steps 6-7, which "can be canceled out") k space is
 * left in that transposed distribution: one exchange on the way in, one on the way out, both of nx/P x ny/P x (nz/2 n_v)
 * complex blocks between every pair of ranks, and one exchange of a row of <= 18 double-double Gram sums.
 *
 * The exchanges happen INSIDE the transform kernels' loads and stores, through per-rank base pointers:
 *   forward   the y pass of rank r writes the rows of rank d's slab to   F_d + (ix_l ny/P + jy_l) nz/2 n_v
 *   backward  the inverse y pass of rank r reads the rows of rank s from B_s + (ix_l ny/P + jy_l) nz/2 n_v
 * Two ways to provide F and B:
 *   staged (default)   F_d = stage + d*block, B_s = stage + s*block in this rank's own staging array; the CALLER moves
 *                      stage -> K of every rank after phase 0 and K -> stage after phase 1 with an all-to-all of equal,
 *                      contiguous blocks (torch.distributed.all_to_all_single over NCCL), and all-gathers the Gram rows
 *                      after phase 2.  rism3d_slab_local gives the addresses.
 *   peer               after rism3d_slab_set_peers (device pointers of every rank's K, Gram and flag arrays, mapped into
 *                      this process: CUDA IPC / torch symmetric memory over NVLink), F_d = K_d + r*block and
 *                      B_s = K_s + r*block: the y pass stores straight into the destination GPU's K and the inverse y
 *                      pass loads straight from the source GPU's K -- the transposes overlap the transforms tile by
 *                      tile and no staging copy exists.  rism3d_iterate then runs whole iterations with in-stream
 *                      barriers (a flag per rank, release/acquire at system scope) where the phases meet.
 * Phases of one iteration (rism3d_slab_phase), every rank the same sequence:
 *   0  pending MDIIS update, closure, forward z, forward y (-> F)          [exchange: forward blocks]
 *   1  forward x, Eq. 32, Eq. 13, inverse x on K, in place                 [exchange: backward blocks]
 *   2  inverse y (<- B), inverse z, residual, Gram row of this slab        [exchange: Gram rows]
 *   3  sum of the ranks' rows in rank order, rms, restart rule, MDIIS solve (identical on every rank)
 * set_solvent_chi and set_solute take the same arguments on every rank (each computes its slabs of w, phi, phi~).
 * free_energy, pmv, pressure_correction and gradient return THIS SLAB'S share of the grid sums: the caller adds the
 * ranks' numbers (dmu, the site integrals, gradient components).  The debug FFT hooks are single-rank only. */

/* Host-only: the slab of rank params->rank (no context, no GPU needed).  Real fields of the rank: planes ix0 .. ix0+nxl-1;
 * its k-space slab: rows jy0 .. jy0+nyl-1; row_elems = (nz/2) * n_sites_padded complex numbers per (ix, iy) row of the
 * spectrum; block_elems = nxl * nyl * row_elems complex numbers per block of the transposes.  Returns RISM3D_ERR_SIZE
 * when the parameters are invalid.  With n_ranks <= 1 the slab is the whole grid. */
typedef struct {
  int nxl, ix0, nyl, jy0;
  int n_sites_padded;
  size_t row_elems, block_elems;
} rism3d_slab_info;
int rism3d_slab_plan(const rism3d_params* params, rism3d_slab_info* out);

/* Addresses of this rank's exchange arrays (DEVICE pointers inside the workspace) and the block size of the transposes:
 * K and stage hold n_ranks blocks of block_bytes each (block s <-> rank s); gram holds n_ranks rows of gram_row_bytes;
 * flags is the barrier array of peer mode.  Any output pointer may be NULL. */
int rism3d_slab_local(rism3d_ctx* ctx, void** d_K, void** d_stage, void** d_gram, void** d_flags, size_t* block_bytes,
                      size_t* gram_row_bytes);

/* Switch to peer mode: d_K[r], d_gram[r], d_flags[r] are the arrays rism3d_slab_local returned on rank r, as DEVICE
 * pointers valid in this process (HOST arrays of n_ranks pointers; entry `rank` is this rank's own).
 * EXPERIMENTAL: peer mode has been checked for numerics with the ranks' phases ordered by the host, and its barrier by
 * the self-test below; a peer-mode rism3d_iterate has not yet run on two GPUs.
 * The call also zeroes this rank's barrier flags and epoch counter.  EVERY rank must call it (again) whenever any rank's
 * context has been (re)created, and the ranks must then meet on the host (a process-group barrier) before the first
 * rism3d_iterate: the in-stream barriers count epochs from that point and rely on every rank enqueueing the same
 * sequence of iterations (same max_iter and tol on every rank). */
int rism3d_slab_set_peers(rism3d_ctx* ctx, void* const* d_K, void* const* d_gram, void* const* d_flags);

/* Longest time one in-stream barrier of a peer-mode rism3d_iterate waits for the other ranks, seconds (0.001..3600;
 * default 30).  When a rank does not arrive in time -- its process died, it enqueued fewer iterations, it was re-created
 * without a new rism3d_slab_set_peers everywhere -- the waiting rank stops iterating instead of spinning inside a kernel
 * for ever: the remaining kernels of the call return at once and rism3d_iterate returns RISM3D_ERR_PEER.  tau is then
 * undefined for the abandoned iteration, and further rism3d_iterate calls fail with RISM3D_ERR_PEER until every rank has
 * called rism3d_slab_set_peers again. */
int rism3d_slab_set_peer_timeout(rism3d_ctx* ctx, double seconds);

/* Test hook: runs the barrier code of peer mode on ONE GPU, the n_ranks (1..8) ranks being the blocks of one cooperative
 * launch (kernels that wait on one another must not be separate launches on one device).  `epochs` barriers in a row;
 * before each, every rank publishes a value that every other rank must see after it.  absent_rank >= 0: that rank never
 * arrives and every other rank must give up after timeout_s (0.001..60).  d_scratch: DEVICE, >= 4096 bytes, overwritten.
 * *n_errors: ordering violations seen (must be 0); *n_timeouts: ranks that gave up (0, or n_ranks - 1 with an absent
 * rank).  Synchronises cuda_stream. */
int rism3d_debug_peer_barrier_selftest(int device, void* d_scratch, size_t bytes, void* cuda_stream, int n_ranks, int epochs,
                                       int absent_rank, double timeout_s, int* n_errors, int* n_timeouts);

/* Mapping the peers' arrays into this process (CUDA IPC; one GPU per process on one node).  A workspace that is to
 * be exported must be an allocation of its own: peer_alloc is a plain cudaMalloc on `device` (a sub-block of a caching
 * allocator cannot be exported).  peer_export fills a 64-byte handle that another process turns into a DEVICE pointer
 * valid in ITS address space with peer_open (which also enables peer access from `device` to the owner's GPU); the
 * arrays of rism3d_slab_local sit at the same offsets in every rank's workspace. */
int rism3d_peer_alloc(int device, size_t bytes, void** d_ptr);
int rism3d_peer_free(int device, void* d_ptr);
int rism3d_peer_export(int device, void* d_ptr, unsigned char handle[64]);
int rism3d_peer_open(int device, const unsigned char handle[64], void** d_ptr);
int rism3d_peer_close(int device, void* d_ptr);

/* Phase calls of a staged run (also usable in peer mode when the caller orders the ranks itself):
 * begin sets the tolerance of the iterations that follow (as rism3d_iterate's tol) and clears the call's counters;
 * phase(0..3) enqueues that phase of one iteration; end applies the pending update (tau is then the new input), reads
 * the state back and reports like rism3d_iterate.  status (rism3d_slab_status): cheap look at the device state between
 * iterations -- *done != 0 once an iteration has met the tolerance or diverged (further phases return immediately). */
int rism3d_slab_begin(rism3d_ctx* ctx, double tol);
int rism3d_slab_phase(rism3d_ctx* ctx, int phase);
int rism3d_slab_status(rism3d_ctx* ctx, int* done, int* n_done, double* rms);
int rism3d_slab_end(rism3d_ctx* ctx, int* n_done, double* rms);

/* Slab runs: free_energy, pmv, pressure_correction and gradient return THIS rank's share of a grid sum; the whole-grid
 * value is the sum of the ranks' shares.  The caller gathers the shares (an all-gather: data movement only) and this call
 * adds them, in rank order, so that every rank gets the same bits whatever the collective library does:
 * per_rank: HOST [n_ranks][n_values], out: HOST [n_values], out[j] = sum_r per_rank[r][j] (r = 0, 1, ...).  Host-only. */
int rism3d_slab_combine(const double* per_rank, int n_ranks, int n_values, double* out);

const char* rism3d_last_error(const rism3d_ctx* ctx);   /* valid until the next call on ctx */
const char* rism3d_status_string(int status);           /* static strings                    */

/* Frees the host context (not the workspace).  NULL is allowed. */
void rism3d_destroy(rism3d_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* RISM3D_H */
