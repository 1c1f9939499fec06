/* sn_weno.h -- C ABI of the WENO-5 / global Lax-Friedrichs flux reconstruction of arXiv 1507.08549 (SURVEY.md section
 * 8f, NEXT-3).
 *
 * What it computes (eqs. 1-4, left-hand sides: the paper's "WENO scheme" subroutine, Table 2 at
 * PAPER.md:155-160; "a fifth-order scheme ... finite-difference formulation ... First we separate the
 * hydro flux into a positive flux and a negative flux by a global Lax-Friedrichs splitting.  Then we apply the WENO
 * reconstruction on the two fluxes by an upwinding scheme.  The numerical flux is obtained by summing the reconstructed
 * positive and negative fluxes"; gamma-law EOS, Courant number 0.5):
 *     L(U) = -(Fhat_{i+1/2} - Fhat_{i-1/2}) / dr - (Ghat_{j+1/2} - Ghat_{j-1/2}) / dz        (Cartesian; no source terms)
 * Readings W1..W9: U[c][j][i], c = (rho, rho v_r, rho v_z, tau), planes of nz x nr, r fastest;
 * p = (gamma-1)(tau - (m_r^2 + m_z^2)/(2 rho)); alpha_r = max_cells(|v_r| + c_s), alpha_z likewise (GLOBAL maxima);
 * F+- = (F +- alpha U)/2 per component; Jiang-Shu WENO-5 (eps = 1e-6, weights 0.1/0.6/0.3); three ghost cells per side
 * with bc[4] = {r-low, r-high, z-low, z-high}, each 0 outflow (edge copy), 1 reflecting (mirror, normal momentum
 * flipped), 2 periodic; time step: SSP-RK3 with alpha recomputed per stage, dt = cfl / (alpha_r/dr + alpha_z/dz).
 *
 * Layout / ownership: U, L are DEVICE pointers to 4*nr*nz contiguous fp64 (component-major).  The handle owns the stage
 * buffers and the device scalars (alpha, dt); the caller owns U / L and the stream.  Everything runs in hand-written
 * sm_100a CUDA kernels (global-maximum reduction, tiled flux reconstruction with the Runge-Kutta stage update fused
 * into its epilogue); no CPU fallback.  One call in flight per handle.  Errors: -1 bad argument, -2 CUDA error,
 * message via sn_weno_last_error.
 */
#ifndef SN_WENO_H
#define SN_WENO_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sn_weno sn_weno; /* opaque */

/* nr, nz >= 1 (with >= 3 cells along an axis whose boundary is periodic or reflecting); dr, dz > 0; gamma > 1;
 * bc: 4 ints in {0, 1, 2}.  Returns NULL on bad arguments, allocation failure or no sm_100 device. */
sn_weno* sn_weno_create(int nr, int nz, double dr, double dz, double gamma, const int* bc);

/* alpha_host[0..1] = (alpha_r, alpha_z) of the state U (W4).  Synchronises `stream`. */
int sn_weno_max_speeds(sn_weno* h, const double* U, double* alpha_host, void* stream);

/* L = L(U).  alpha_r, alpha_z >= 0: splitting speeds to use; either < 0: the global maxima of U, computed on the
 * device (no host round trip).  U and L must not alias.  Asynchronous on `stream`. */
int sn_weno_rhs(sn_weno* h, const double* U, double* L, double alpha_r, double alpha_z, void* stream);

/* One SSP-RK3 step in place (W8): 3 x (global maxima -> flux reconstruction with the stage update fused).  *dt_host
 * (may be NULL) receives the step; the call synchronises `stream` only if dt_host != NULL. */
int sn_weno_step(sn_weno* h, double* U, double cfl, double* dt_host, void* stream);

/* March from t = 0 to t_end (the last step is shortened to land on it), at most max_steps steps.  The time and the
 * step, including the shortened last one, are formed on the device from the maxima the first stage computes anyway;
 * the host reads (dt, t, last-step flag) back once per step to decide whether to go on.  Returns the number of steps
 * (>= 0) or an error code (< 0).  Synchronises `stream`. */
int sn_weno_evolve(sn_weno* h, double* U, double cfl, double t_end, int max_steps, void* stream);

/* Same as sn_weno_rhs with HOST buffers (H2D of U, D2H of L inside the call). */
int sn_weno_rhs_host(sn_weno* h, const double* U_host, double* L_host, void* stream);

/* Counters of the last call: "rhs_ms" (device time of the flux-reconstruction kernel(s), CUDA events on the caller's
 * stream), "total_ms", "launches".  Returns 0 or -1. */
int sn_weno_get_stat(sn_weno* h, const char* key, double* out);

void sn_weno_destroy(sn_weno* h);
const char* sn_weno_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SN_WENO_H */
