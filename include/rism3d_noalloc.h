/* rism3d_noalloc.h -- one entry point of librism3d.so that needs no device memory from anyone.
 *
 * Why it exists.  Everything else in this library works out of a workspace the caller allocates and hands to
 * rism3d_init (rism3d.h): the solvation-free-energy sum of Eq. 17-18, for one, parks its per-block
 * partial sums in a corner of that workspace.  Some users of a 3D-RISM result cannot provide such a buffer:
 *   - an MD or QM host program that calls 3D-RISM every step (MM/3D-RISM) and whose own memory pool
 *     has taken the whole GPU at start-up -- a cudaMalloc from a plug-in then simply fails;
 *   - code that sits between other people's asynchronous work on the same GPU, where cudaMalloc / cudaFree would
 *     stall every stream of the device while they run;
 *   - an analysis step that holds tau, w and phi of a finished solve in buffers it was GIVEN (by the solver, by another
 *     process) and has no allocator of its own.
 * For them the same sum is offered here with its scratch in a fixed array that is part of the library image: a
 * file-scope `static __device__` array of RISM3D_NOALLOC_SCRATCH_BYTES.  Every GPU that loads librism3d.so carries that
 * array from the moment the CUDA runtime loads the library's device code until the process exits, whether or not this
 * function is ever called.  The function calls no cudaMalloc, cudaFree, cudaMallocHost or any library routine that
 * allocates; the caller passes the input fields and the place for the result, nothing else.
 */
#ifndef RISM3D_NOALLOC_H
#define RISM3D_NOALLOC_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RISM3D_NOALLOC_MAX_SITES  8            /* solvent site types per call                                        */
#define RISM3D_NOALLOC_MAX_POINTS 134217728    /* grid points per call: 512^3, the largest grid of rism3d_init       */
#define RISM3D_NOALLOC_SCRATCH_BYTES 151552    /* 2 sums x 592 blocks x 8 sites x (hi, lo) x 8 bytes = 148 KiB/GPU   */

/* Solvation free energy per solvent site type from fields the caller already has on the device (Eq. 18 KH, Eq. 17 HNC,
 * PSE-n as DESIGN.md Q2 / Q10 -- the same integrand, block shape and summation order as rism3d_free_energy):
 *
 *   d_out[g]           = k_B T rho_g dV sum_r [ -c_sr - h c / 2 + h^2 / 2 - B ],   kcal/mol
 *   d_out[n_sites + g] = dV sum_r c_sr,g(r),  A^3   (the integrals Eq. 19 needs, as rism3d_pmv's c_int_site)
 *   with g = closure(w + tau), h = g - 1, c_sr = h - tau, c = c_sr - q_g phi, dV = spacing^3,
 *   B = h^2/2 where h > 0 (KH), d^(n+1)/(n+1)! where d = w + tau > 0 (PSE-n), 0 (HNC).
 *
 * Arguments
 *   device         CUDA device ordinal the pointers below belong to; it is made current for the call and the caller's
 *                  current device is restored before returning.
 *   cuda_stream    a cudaStream_t of that device (NULL = legacy default stream).  The two kernels are ENQUEUED on it and
 *                  the function returns without waiting: d_out is valid once the stream has passed them.
 *   n_points       grid points per field, 1..RISM3D_NOALLOC_MAX_POINTS (any shape: the sum does not care).
 *   spacing        grid spacing, A (> 0).          temperature   K (> 0).
 *   n_sites        1..RISM3D_NOALLOC_MAX_SITES.    closure / pse_order   rism3d_closure and the n of PSE-n (>= 1).
 *   q, rho         HOST [n_sites]: site charges (e) and number densities (1/A^3); copied into the launch parameters.
 *   d_tau, d_w     DEVICE [n_sites][n_points] doubles: tau = t - f and w = -beta u + f (rism3d_get_field TAU / W).
 *   d_phi          DEVICE [n_points]: phi(r) of Eq. 29 (rism3d_get_field PHI).  Inputs are only read.
 *   d_out          DEVICE [2][n_sites] doubles, written as above.  Caller-owned like the inputs.
 *   err, err_cap   optional HOST buffer for the message of a failure (may be NULL / 0).
 *
 * Errors (nothing is enqueued when one is returned)
 *   RISM3D_ERR_ARG   a NULL pointer, an unknown closure, a device ordinal that does not exist
 *   RISM3D_ERR_SIZE  n_sites or n_points outside the limits above -- the scratch array has a slot for 8 site types per
 *                    block and cannot grow, so a larger request is refused, never truncated -- or spacing /
 *                    temperature / pse_order not positive
 *   RISM3D_ERR_CUDA  the address of the scratch array could not be obtained, or a launch failed
 *
 * First call on a device.  The scratch array is addressed from host code through a device pointer that the library
 * looks up (cudaGetSymbolAddress, with that device current) the first time this function runs on each device, and keeps.
 * That look-up may make the CUDA runtime load the library's device code, so let the first call on a device happen during
 * start-up: outside any stream capture, and before the part of the program that must not stall.
 *
 * Sharing.  There is ONE array per GPU and every call on that GPU uses it, from any thread, stream or context of the
 * process.  Nothing in it has to be zero on entry -- each call first overwrites every slot it later reads, so whatever the
 * previous call left behind (also from a call with more site types) is harmless.  But two calls that are in flight on the
 * same GPU at the same time -- on different streams, or from different threads -- write the same slots and BOTH results
 * are garbage: keep the calls of one GPU on one stream, or order them with events.  Calls on different GPUs are
 * independent.  The existing rism3d_free_energy is unchanged and remains the path for callers who own a workspace.
 */
int rism3d_noalloc_free_energy(int device, void* cuda_stream, size_t n_points, double spacing, int n_sites, int closure,
                               int pse_order, double temperature, const double* q, const double* rho,
                               const double* d_tau, const double* d_w, const double* d_phi, double* d_out,
                               char* err, size_t err_cap);

#ifdef __cplusplus
}
#endif
#endif /* RISM3D_NOALLOC_H */
