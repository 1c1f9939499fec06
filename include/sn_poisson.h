/* sn_poisson.h -- C ABI of the B200-native self-gravity Poisson solve of arXiv 1507.08549.
 *
 * What it computes (§2.1: "Phi, the gravitational potential, satisfies the Poisson Equation
 * nabla^2 Phi = 4 pi G rho"; §2.1: "We use the successive overrelaxation method with the
 * Gauss-Seidel method to solve the Poisson equation in cylindrical coordinates. The iteration is stopped by
 * default when the relative changes of all grids reach below 1e-8. The inner boundaries are assumed to be
 * reflecting and the outer boundaries are fixed by using the Roche approximation Phi(r,z) = -GM/sqrt(r^2+z^2)
 * ... in general higher multipole terms are needed"; §2.3 / Table 2: the Poisson solver is
 * the largest of the subroutines the paper offloads to a GPU).
 *
 * One solve = (a-1) multipole moments M_l = sum rho (s/L0)^l P_l(cos theta) dV, l = 0..lmax, about the origin
 *           -> (a-1b) Dirichlet ghost values phi_b = -(1/L0) sum_l M_l P_l / (s/L0)^(l+1) one cell outside
 *              the east / north (/ south) edges (lmax = 0 is the paper's Roche boundary)
 *           -> (a-2) red-black SOR sweeps of the conservative cell-centred 5-point cylindrical Laplacian
 *           -> (a-3) per-sweep fused residual maxima and an on-device stopping decision.
 * The exact discretisation, orderings and pinned fp64 arithmetic are DESIGN.md §2-3 (readings R1..R14).
 * G = 1: the library solves nabla^2 phi = 4 pi rho; callers scale rho or phi.
 *
 * Grid and layout: uniform (r,z) grid, cell centres r_i = (i+1/2) dr, i in [0,nr);
 *   symmetry = 1 (half plane, reflecting equator): z_j = (j+1/2) dz;
 *   symmetry = 0 (full plane): z_j = (j+1/2 - nz/2) dz;  j in [0,nz).
 * Arrays rho and phi hold interior cells only (no ghost layer), fp64, contiguous, index j*nr + i (r fastest).
 *
 * Everything runs in hand-written sm_100a CUDA kernels.  There is no CPU fallback: every entry point fails
 * (NULL / status < 0, message via sn_poisson_last_error) when no CUDA device of compute capability 10.x is
 * usable.  No exceptions cross this boundary.  A handle supports one solve in flight at a time.
 */
#ifndef SN_POISSON_H
#define SN_POISSON_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sn_poisson sn_poisson; /* opaque handle; owns all device workspace */

/* Returned by value (16 bytes).
 *   sweeps   : full sweeps (red half-sweep + black half-sweep) applied to the returned phi
 *   status   : 0 converged (tol > 0) or fixed-sweep run completed (tol <= 0);
 *              1 hit max_sweeps without reaching tol (not an error);
 *             -1 bad argument / NULL (phi untouched); -2 CUDA error, or the resident kernel's watchdog tripped (a
 *                wait on another CTA exceeded its budget; phi unspecified); -3 non-finite residual
 *   residual : R_k of the last applied sweep k,
 *              R_k = max|res| / (max|4 pi rho| + (2/dr^2+2/dz^2) max|phi_new|)   (R9)            */
typedef struct {
    int32_t sweeps;
    int32_t status;
    double residual;
} sn_poisson_result;

/* Create a solver for an nr x nz grid.  nr, nz >= 2; dr, dz > 0 finite; symmetry in {0,1};
 * 0 <= lmax <= 64 (odd l are ignored when symmetry = 1; lmax = 0 reproduces PAPER.md:99's Roche boundary).
 * Binds to the current CUDA device.  The relaxation factor defaults to the closed form of DESIGN.md R8.
 * Returns NULL on bad arguments, allocation failure or no sm_100 device. */
sn_poisson* sn_poisson_create(int nr, int nz, double dr, double dz, int symmetry, int lmax);

/* Solve nabla^2 phi = 4 pi rho.
 *   rho        DEVICE pointer, nr*nz fp64, read-only, never modified.
 *   phi_inout  DEVICE pointer, nr*nz fp64: initial guess on entry (zeros = cold start, the previous potential
 *              = warm start), the iterate after `sweeps` sweeps on exit.
 *   tol > 0    stop after the first sweep k with R_k <= tol, or at max_sweeps.
 *   tol <= 0   run exactly max_sweeps sweeps.
 *   stream     cudaStream_t passed as void* (NULL = legacy default stream).  All work is enqueued on it and it
 *              is synchronised once before returning (the result is decided on the device).
 * Caller owns rho, phi and the stream; the handle owns everything else. */
sn_poisson_result sn_poisson_solve(sn_poisson* h, const double* rho, double* phi_inout, double tol,
                                   int max_sweeps, void* stream);

/* Same solve with HOST buffers (pageable or pinned): copies rho and phi to device workspace, solves, copies phi
 * back.  All copies are on `stream` and inside the call. */
sn_poisson_result sn_poisson_solve_host(sn_poisson* h, const double* rho_host, double* phi_inout_host,
                                        double tol, int max_sweeps, void* stream);

/* Limits: max_sweeps <= 4194304 (2^22) and max_sweeps x nbatch <= 2^26 -- the handle keeps 44 bytes of per-sweep
 * bookkeeping per member (maxima slots 16 + 8, equator-row slots of stop rule 1 8 + 4, R_k history 8), i.e. up to
 * 2.75 GiB at the limit, allocated for the largest max_sweeps x nbatch a handle has seen; larger values are rejected
 * with status -1. */

/* nbatch independent solves on the same grid geometry ([CFG 4a]).  rho, phi_inout: DEVICE pointers to nbatch
 * consecutive grids (member b at offset b*nr*nz).  out: HOST array of nbatch results.
 * Returns 0, or a negative status if the call itself failed. */
int sn_poisson_solve_batch(sn_poisson* h, int nbatch, const double* rho, double* phi_inout, double tol,
                           int max_sweeps, void* stream, sn_poisson_result* out);

/* sn_poisson_solve_batch with HOST buffers (pageable or pinned; layout as above).  rho is uploaded on `stream`,
 * phi's upload overlaps the moment / boundary kernels on an internal copy stream, phi's download is enqueued right
 * behind the relaxation; ONE stream synchronisation per call.  sn_poisson_solve_host is the nbatch = 1 case.
 * Device staging is grown on demand and kept on the handle.  Also on a negative return every copy the call enqueued
 * has finished.  Returns 0 or a negative status. */
int sn_poisson_solve_batch_host(sn_poisson* h, int nbatch, const double* rho_host, double* phi_inout_host,
                                double tol, int max_sweeps, void* stream, sn_poisson_result* out);

/* A warm-started SEQUENCE of nsteps solves on one grid ([CFG 3]: rho evolves, every solve starts from the previous
 * phi), HOST buffers:
 *   rho_seq_host    [nsteps][nr*nz]  the density of every step (read-only)
 *   phi_inout_host  [nr*nz]          initial guess of step 0 on entry, the potential of the LAST step on exit
 *   phi_seq_host    [nsteps][nr*nz]  the potential after every step, or NULL if only the last one is wanted
 *   out             [nsteps]         HOST array of results
 * Copy-compute overlap: rho_{t+1} is uploaded on an internal copy stream while solve t runs, and phi_t is downloaded
 * from a device snapshot while solve t+1 runs (moments are recomputed every step).  Stops early (returning 0) at the
 * first step t whose status is < 0; later entries of `out` are then untouched, phi_seq_host[0..t-1] are complete,
 * phi_seq_host[t..] are not written and phi_inout_host receives phi of the failed step as the device holds it (what
 * sn_poisson_solve leaves behind for that status; the last good potential is phi_seq_host[t-1]).  However the call
 * ends -- all steps, an early stop, or a negative return -- both the caller's stream and the internal copy stream have
 * been synchronised: no copy still reads or writes the host buffers afterwards.  Returns 0 or a negative status. */
int sn_poisson_solve_sequence_host(sn_poisson* h, int nsteps, const double* rho_seq_host, double* phi_inout_host,
                                   double* phi_seq_host, double tol, int max_sweeps, void* stream,
                                   sn_poisson_result* out);

void sn_poisson_destroy(sn_poisson* h);

/* ---- optional, additive --------------------------------------------------------------------------------- */

/* Override the relaxation factor (0 < omega < 2), e.g. [CFG 0]'s 1.9; omega <= 0 restores the default formula.
 * Returns 0 or -1. */
int sn_poisson_set_omega(sn_poisson* h, double omega);
double sn_poisson_get_omega(const sn_poisson* h);

/* NEXT-1: the paper-literal stopping rule.  rule = 0 (default): the residual ratio R_k of
 * DESIGN.md R9.  rule = 1: "The iteration is stopped by default when the relative changes of all grids reach
 * below 1e-8" -- reading R16: E_k = max|dphi| / max|phi_new| of sweep k, dphi = (omega/diag_j) res the change the update
 * applies to a cell; stop after the first sweep with E_k <= tol (the paper's default is tol = 1e-8; with lmax = 0 the
 * boundary is the paper's Roche formula).  `residual` and get_history then hold E_k.  All three sweep paths support
 * both rules.  Returns 0 or -1. */
int sn_poisson_set_stop_rule(sn_poisson* h, int rule);

/* NEXT-1: the gravity field g = -grad phi at the cell centres, the source term of the paper's
 * momentum and energy equations (eqs. 2-4).  Centred differences with the solver's boundary handling
 * (R15): reflecting axis, reflecting equator when symmetry = 1, elsewhere the ghost values of the LAST solve
 * / batch on this handle (or the injected ones).  phi, gr, gz: DEVICE pointers to nbatch consecutive grids (layout of
 * sn_poisson_solve_batch); gr, gz must not alias phi.  The kernel is enqueued on `stream` and NOT synchronised.
 * Returns 0, -1 (bad argument, or no ghost values for nbatch members yet), -2 (CUDA error). */
int sn_poisson_gravity(sn_poisson* h, int nbatch, const double* phi, double* gr, double* gz, void* stream);

/* Solve (as sn_poisson_solve_batch; nbatch = 1 for a single grid) AND emit the gravity field of the result in the same
 * call: gr, gz are DEVICE pointers to nbatch consecutive grids receiving g_r, g_z = -grad phi (definition and boundary
 * handling as sn_poisson_gravity).  On the resident path the epilogue is fused into the relaxation kernel: every thread
 * differences the patch of phi it still holds in registers right after its final store (neighbours outside the patch
 * from the stored result, after one grid barrier); on the blocked / streaming paths the standalone gravity kernel is
 * enqueued right behind the last sweep.  Bit-identical to sn_poisson_gravity on the returned phi.  gr, gz, phi_inout
 * must not alias.  gr / gz need only be 8-byte aligned: when either is not 16-byte aligned the resident path skips its
 * fused epilogue and the standalone kernel (scalar stores) runs behind it.  Returns 0 or a negative status. */
int sn_poisson_solve_gravity(sn_poisson* h, int nbatch, const double* rho, double* phi_inout, double* gr, double* gz,
                             double tol, int max_sweeps, void* stream, sn_poisson_result* out);

/* Test hooks.  All pointers are HOST pointers.
 * get_moments : M[0..lmax] of batch member 0 of the last solve (odd entries 0 when symmetry = 1).
 * set_boundary: inject ghost values bE[nz], bN[nr], bS[nr] (bS ignored when symmetry = 1) and skip the moment and
 *               boundary kernels in later solves; (NULL, NULL, NULL) restores the multipole boundary.
 * get_boundary: the ghost arrays used by batch member 0 of the last solve.
 * get_history : R_k for k = 1..min(n, sweeps) of batch member 0 of the last solve; returns the count copied.
 *               Paths 2 / 3 without the "exact" option track only the upper 32 bits of the maxima until the rule
 *               may have fired: entries before the last (exactly tracked) interval are lower bounds within 2^-19
 *               of R_k; the returned `residual` and the last entry are always exact. */
int sn_poisson_get_moments(sn_poisson* h, double* M);
int sn_poisson_set_boundary(sn_poisson* h, const double* bE, const double* bN, const double* bS);
int sn_poisson_get_boundary(sn_poisson* h, double* bE, double* bN, double* bS);
int sn_poisson_get_history(sn_poisson* h, double* R, int n);

/* Tuning knobs; unknown keys return -1.
 *   "path"        0 auto, 1 streaming kernels (one launch per colour), 2 resident persistent cooperative kernel
 *                 (phi on chip for the whole solve; every tile of every batch member co-resident), 3 blocked kernel
 *                 (one launch per m sweeps; any size, batches)
 *   "chunk"       launches enqueued between host polls of the device-side decision (paths 1 and 3)
 *   "tblock"      path 2 block mode / path 3: sweeps per halo exchange / per launch (temporal blocking depth m);
 *                 path 2 halo mode: sweeps per report / checkpoint interval; 0 = planner's choice
 *   "shape"       box shape index of path 2 / 3; -1 = planner's choice
 *   "halo"        path 2: 1 = halo mode (box == tile, edge exchange every half-sweep), 0 = block mode (margins of
 *                 2m cells, exchange every m sweeps), -1 = planner's choice
 *   "ds"          path 2 halo mode: 1 = all tiles of a member in one thread-block cluster (<= 16 tiles), edges through
 *                 distributed shared memory (st.async + mbarrier), one cluster per batch member (any batch size: the
 *                 clusters are independent); 0 = never; -1 = planner's choice
 *   "ring"        path 2 halo mode: 1 = ring duty (every box-edge cell is also updated, first thing in the half-sweep,
 *                 by the thread that receives on that edge, and sent at once, so that the packets travel during the
 *                 patch update), 0 = the owners of the edge cells send after their patch update, -1 = planner's
 *                 choice (on through L2 packets, off inside a cluster)
 *   "ll"          path 2 block mode: 1 = margins travel as tagged packets, 0 = tile flags + ring loads, -1 = auto
 *   "group"       batches on path 2: G > 0 = solve the batch in groups of G members, one resident launch after the
 *                 other; 0 = never group (all members co-resident or another path); -1 = group when the whole batch
 *                 cannot be co-resident and a group fills the chip in halo mode
 *   "exact"       1: paths 2 / 3 track the per-sweep maxima exactly in every interval / launch (exact R_k history)
 *   "prof"        1: path 2 records an in-kernel SM-clock profile (stats "prof_mean0..7", "prof_max0..7": total,
 *                 half-sweep compute, halo exchange, barrier, end of interval, margin refill, wait for the
 *                 decision, half-sweeps; mean / max over the CTAs, thread 0 of each)                         */
int sn_poisson_set_option(sn_poisson* h, const char* key, int64_t value);

/* Counters of the last solve / batch: "launches" (kernels launched), "sweep_launches" (those that ran relaxation
 * sweeps), "sweep_ms" (device time of the relaxation phase, CUDA events on the caller's stream), "setup_ms"
 * (moments + boundary), "path" (1, 2 or 3 as above), "ctas", "tile_w", "tile_h", "tblock", "shape", "halo", "ds", "ring",
 * "group" (members per resident launch), "redundancy" (cells updated per half-sweep / cells of the grid: 1 in halo
 * mode and on the streaming path, box cells / tile cells with temporal blocking).
 * Returns 0 or -1. */
int sn_poisson_get_stat(sn_poisson* h, const char* key, double* out);

/* Measurement aid (no handle, not part of the solve path): L2-resident bandwidth of this GPU in GB/s, measured with
 * two plain kernels of the library over a working set of 2 x `mib` MiB (copy: read + write bytes) / `mib` MiB (read).
 * the L2 peak is not in MEASURED_PEAKS.json and must be measured on the box; bench.py uses
 * the copy figure as the roofline denominator of the L2-bound rows.  Synchronises `stream`.  Returns 0 / -1 / -2. */
int sn_poisson_probe_l2(int mib, double* copy_gbs, double* read_gbs, void* stream);

/* Message of the last failure on this thread ("" if none). */
const char* sn_poisson_last_error(void);
const char* sn_poisson_version(void);

/* ---- NEXT-4: a faster-converging variant on the same stencil --------------------------------
 * Red-black-smoothed geometric multigrid (not in the paper, which relaxes the same equation by SOR).  Same
 * equation, discretisation, multipole ghosts and therefore the same converged potential as sn_poisson_solve; only the
 * iteration differs (readings M1..M8): V-cycles over the levels (nr / 2^l) x (nz / 2^l) (coarsened
 * while both counts are even and >= 8), red-black Gauss-Seidel smoothing (options "mg_nu1", "mg_nu2": sweeps before /
 * after the coarse-grid correction, default 1 / 1; "mg_nc": sweeps on the coarsest level, default 12), volume-weighted
 * restriction, bilinear prolongation, coarse Dirichlet ghosts extrapolated to the level-0 ghost centre.  After every
 * cycle the ratio R (rule R9) of the TRUE residual of the iterate is evaluated on the device; the solve stops after the
 * first cycle with R <= tol (tol <= 0: exactly max_cycles cycles).  Returns {cycles, status, R} like sn_poisson_solve
 * (`sweeps` = V-cycles applied); sn_poisson_get_history then returns R after every cycle.  rho / phi_inout: DEVICE
 * pointers as for sn_poisson_solve; any nr, nz >= 2 (a grid that cannot be coarsened runs plain Gauss-Seidel sweeps).
 * The stopping rule option (sn_poisson_set_stop_rule) does not apply.  One V-cycle is captured as a CUDA graph and
 * re-launched per cycle (option "mg_graph", default 1; re-captured when tol / max_cycles / the options change); with the legacy default stream the cycles run on a stream of the handle ordered between the caller's work.
 * Synchronises `stream`. */
sn_poisson_result sn_poisson_solve_mg(sn_poisson* h, const double* rho, double* phi_inout, double tol, int max_cycles,
                                      void* stream);
/* nbatch independent solves in one call (layout and `out` as for sn_poisson_solve_batch): every kernel of a cycle covers
 * all members, each member stops on its own ratio, the call returns when the last one has.  Member b's result is the
 * one sn_poisson_solve_mg gives for it alone, bit for bit.  Returns 0, or < 0 as sn_poisson_solve_batch. */
int sn_poisson_solve_mg_batch(sn_poisson* h, int nbatch, const double* rho, double* phi_inout, double tol, int max_cycles,
                              void* stream, sn_poisson_result* out);
/* The same as sn_poisson_solve_mg with HOST buffers (H2D of rho and phi, D2H of phi inside the call). */
sn_poisson_result sn_poisson_solve_mg_host(sn_poisson* h, const double* rho_host, double* phi_inout_host, double tol,
                                           int max_cycles, void* stream);
/* sn_poisson_solve_mg_batch with HOST buffers (pageable or pinned; layout as sn_poisson_solve_batch_host): rho goes up
 * on `stream`, phi's upload overlaps the moment / boundary kernels on the internal copy stream, phi comes back behind
 * the last cycle; one stream synchronisation.  sn_poisson_solve_mg_host is the nbatch = 1 case.  Also on a negative
 * return every copy the call enqueued has finished.  Returns 0 or a negative status. */
int sn_poisson_solve_mg_batch_host(sn_poisson* h, int nbatch, const double* rho_host, double* phi_inout_host, double tol,
                                   int max_cycles, void* stream, sn_poisson_result* out);

/* ---- Multipole moments without any device allocation ----------------------------------------------------------------
 * Who this is for.  Every other entry point works through a handle, and a handle gets its workspace from cudaMalloc
 * (at sn_poisson_create and again on the first solve).  Some hosts cannot do that: a hydro code that sized its grids to
 * fill the GPU at start-up and left no free memory to ask for; a framework in which all device memory belongs to one
 * pool and stray cudaMalloc calls are banned; a time-step loop that cannot accept cudaMalloc / cudaFree stalling the
 * whole device while other streams are busy.  For them this one call computes step (a-1) -- M_l, l = 0..lmax, and
 * max|4 pi rho| -- with no handle and without calling cudaMalloc, cudaFree or anything else that allocates.
 *
 * How.  The reduction needs a little global scratch between its two kernels (per-block partial sums and one control
 * block per member).  Here that scratch is a fixed array built into the library image: 520 KiB of device memory on
 * every GPU that loads the library, held until the process exits, whether or not this function is ever called.
 *
 * Arguments.  rho: DEVICE pointer, nbatch consecutive grids in the layout above (read only).  nr, nz, dr, dz, symmetry,
 * lmax: as for sn_poisson_create.  M_out: DEVICE pointer to nbatch * (lmax + 1) doubles, member b's M_l at
 * M_out[b * (lmax + 1) + l] (odd l are 0 when symmetry = 1).  maxf_out: DEVICE pointer to nbatch doubles receiving
 * max|4 pi rho| per member, or NULL.  The caller owns all three buffers.  stream: cudaStream_t or NULL.
 * The work is enqueued on `stream` and the call returns without waiting; results are valid once the stream reaches
 * that point.  Same kernels, block count and summation order as a handle uses, so M equals what
 * sn_poisson_get_moments reports after a solve of the same grid (the tests compare at the 1e-13 bar of the moment tests).
 *
 * Limits, checked up front.  1 <= nbatch <= SN_POISSON_STATIC_MAX_BATCH, and nbatch * B * NL <=
 * SN_POISSON_STATIC_MAX_DOUBLES, where B = min(ceil(nr * nz / 1024), 4 * SM count) blocks per member and NL = 9 / 17 /
 * 33 / 65 for lmax <= 8 / 16 / 32 / 64.  On a B200 (148 SMs) a single grid of any size fits at every lmax; large
 * grids fit up to 12 / 6 / 3 / 1 members per call.  A request beyond either limit returns -1 with the numbers in
 * sn_poisson_last_error; nothing is launched.  Other returns: 0 = enqueued, -1 = bad argument, -2 = CUDA error.
 *
 * Sharing.  All calls on one GPU use the same array, and it keeps the previous call's contents; the function clears the
 * part that has to start at zero itself (on `stream`), so back-to-back calls on ONE stream are safe.  Two calls whose
 * kernels can overlap on the GPU -- different streams, or different host threads without ordering between them --
 * race on the scratch and give wrong moments; serialise them (same stream, or an event).
 *
 * First call.  The first call on each device looks up the array's device address (cudaGetSymbolAddress, with that
 * device current) and caches it; make that first call in ordinary, non-capturing code, before any stream capture is
 * begun on the device.  Later calls do no set-up. */
#define SN_POISSON_STATIC_MAX_BATCH 64
#define SN_POISSON_STATIC_MAX_DOUBLES 65536
int sn_poisson_moments_static(const double* rho, int nbatch, int nr, int nz, double dr, double dz, int symmetry,
                              int lmax, double* M_out, double* maxf_out, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* SN_POISSON_H */
