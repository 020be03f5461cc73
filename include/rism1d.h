/* rism1d.h -- C ABI of the 1D solvent-solvent RISM solve on the GPU (part of librism3d.so).
 *
 * Produces what the 3D path takes as input: the solvent susceptibility chi_ab(k) = w_ab(k) + rho_a h_ab(k)
 * ("X = omega + rho h, obtained by the 1D-RISM calculation for a pure solvent system"), and the
 * bulk properties of Eq. 19-21 (isothermal compressibility chi_T, pressure P).  The paper gives the
 * equations (Eq. 4 the 1D-RISM equation; closures Eq. 5-7) and defers the numerics to its
 * ref. 7; the procedure is the one of DESIGN.md "O-1D" (SURVEY.md section 8(f) NEXT-4 "GPU 1D-RISM"):
 *
 *   full-site formulation, n_sites x n_sites pair functions on the radial grid r_i = i dr, k_j = j dk, i, j = 1..M-1,
 *   dr dk = pi / M;  iteration variable tau_ab(r) = t_ab - f_ab (t = h - c), the analytic long-range split of
 *   Eq. 29-30 per pair;  one pass:
 *     g = closure(w + tau),  w = -beta [LJ + C q_a q_b exp(-kappa r)/r]            Eq. 5-7
 *     c_sr = g - 1 - tau ;   C_sr(k) by the radial sine transform ;  C = C_sr - F    Eq. 29-30
 *     H(k) = (I - W C R)^-1 W C W,  W = intramolecular matrix, R = diag(rho_a)      Eq. 4 solved for h at each k
 *     tau'(r) from H - C_sr, symmetrised in (a, b);  residual, MDIIS (Eq. 40)
 *   radial transforms: F(k_j) = (4 pi dr / k_j) sum_i r_i f(r_i) sin(pi i j / M) and its mirror image, as type-I
 *   sine transforms through a complex FFT of the odd extension (length 2M).
 *
 * Same conventions as rism3d.h: HOST pointers unless said otherwise, negative rism3d_status codes on failure, the
 * caller owns the device workspace and the stream, no CPU fallback.  Units: A, e, kcal/mol, K.
 */
#ifndef RISM1D_H
#define RISM1D_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rism1d_ctx rism1d_ctx;

typedef struct {
  int    n_sites;           /* full solvent sites (every site of every species), 1..8                          */
  int    n_points;          /* M: power of two in 512..16384; the radial grid has M - 1 points                   */
  double dr;                /* radial spacing, A                                                                 */
  double temperature;       /* K                                                                                 */
  double kappa;             /* kappa of Eq. 29-30, 1/A                                                           */
  int    closure;           /* rism3d_closure (KH = 1, PSE = 2, HNC = 3)                                          */
  int    pse_order;
  int    mdiis_nvec;        /* 1..16                                                                             */
  double mdiis_b;           /* damping b of Eq. 40                                                               */
  double mdiis_restart;     /* restart factor; <= 0: never                                                       */
  int    device;
} rism1d_params;

size_t rism1d_workspace_bytes(const rism1d_params* params);   /* 0 when the parameters are invalid */

/* d_workspace: DEVICE, 256-byte aligned, kept alive by the caller until rism1d_destroy.  tau starts at 0. */
int rism1d_init(rism1d_ctx** out, const rism1d_params* params, void* d_workspace, size_t bytes, void* cuda_stream);

/* q, sigma, eps [n_sites]; rho [n_sites]: number density of the SPECIES site a belongs to, 1/A^3; species [n_sites]:
 * species index of each site; bond [n_sites][n_sites]: intramolecular distance of two sites of one species, A (ignored
 * on the diagonal and across species).  Lorentz-Berthelot mixing (Q4). */
int rism1d_set_solvent(rism1d_ctx* ctx, const double* q, const double* sigma, const double* eps, const double* rho,
                       const int* species, const double* bond);

/* Iterate from the current tau with all charges scaled by charge_scale (a charge ramp 0 -> 1 is the usual way to reach
 * the solution of a polar liquid: call repeatedly with growing scale; every call starts a fresh MDIIS history).
 * Stops after the first iteration whose rms residual sqrt(sum R^2 / (n_sites^2 (M - 1))) is below tol (tau is then left
 * unchanged by it), or after max_iter.  n_done / rms may be NULL.  RISM3D_ERR_DIVERGED on a non-finite residual. */
int rism1d_solve(rism1d_ctx* ctx, double charge_scale, int max_iter, double tol, int* n_done, double* rms);

/* Pair functions of the current tau: which = 0: g_ab(r), 1: tau_ab(r), 2: c_sr,ab(r);  dst: [n_sites][n_sites][M - 1]. */
int rism1d_get_pair(rism1d_ctx* ctx, int which, double* dst);

/* chi_ab(k_j) = w_ab(k_j) + rho_a h_ab(k_j) of the current tau, j = 1..M-1, k_j = j pi / (M dr):  dst [M - 1][n][n]. */
int rism1d_get_chi(rism1d_ctx* ctx, double* dst);

/* The same reduced to site TYPES (what rism3d_set_solvent_chi takes; Q15): site_type [n_sites] maps every
 * site to a type 0..n_types-1;  chi_{g'g} = sum over the sites a of type g' of chi_ab, b any one site of type g.
 * dst [M - 1][n_types][n_types]. */
int rism1d_get_chi_types(rism1d_ctx* ctx, int n_types, const int* site_type, double* dst);

/* Bulk thermodynamics of the solved liquid (Q19, Q20):
 *   1 / (k_B T chi_T) = sum_species rho - sum_ab rho_a rho_b int c_ab dr              (chi_t, A^3 mol / kcal)
 *   P = k_B T [ sum_species rho (n_species_sites + 1) / 2 - (1/2) sum_ab rho_a rho_b int c_ab dr ]   (Eq. 20, kcal/(mol A^3))
 * with int c_ab dr = 4 pi dr sum_i r_i^2 c_sr,ab(r_i) (the long-range parts cancel for a neutral solvent).
 * c0 (may be NULL): [n_sites][n_sites] the integrals themselves. */
int rism1d_thermo(rism1d_ctx* ctx, double* chi_t, double* pressure, double* c0);

long long rism1d_launch_count(const rism1d_ctx* ctx);
const char* rism1d_last_error(const rism1d_ctx* ctx);
void rism1d_destroy(rism1d_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* RISM1D_H */
