/* sn_levelset.h -- C ABI of the level-set re-initialisation of arXiv 1507.08549.
 *
 * What it computes (section 2.2: "we enumerate all positions where the flame front cut the grid, by
 * finding all neighboring pairs of the scalar field where its values are of opposite signs.  The position of the flame
 * front is obtained by linear interpolation.  Then the distances of all grid points to the flame front positions are
 * compared, and the smallest one is chosen as the new value of S"; eqs. (6)-(7):
 *     S_new = H(d) S_old + (1 - H(d)) d,   H(d) = (1 - tanh((d - d0)/(Delta/3))) / (1 - tanh(-d0/(Delta/3))),  d0 = 3 Delta;
 * S lives on the cell CORNERS; Table 2: the paper's second-largest GPU routine).
 * Readings L1..L6: node (i, j) at (i dr, j dz); an edge is cut when one end is < 0 and the other
 * >= 0; crossing = fma(S_a/(S_a - S_b), h, x_a); d = copysign(sqrt(min (fma(dy, dy, dx dx))), S_old); H at |d|; no
 * crossing: S unchanged, return 0; no mirror images across the axis / equator.
 *
 * Layout: S_old, S_new, dist are DEVICE pointers to nx*ny fp64, index j*nx + i (x fastest), nx = nr + 1, ny = nz + 1.
 * Everything runs in hand-written sm_100a CUDA kernels (crossing enumeration -> pairwise minimum distance -> blend);
 * no CPU fallback.  The handle owns the crossing list and the partial-minimum workspace; the caller owns S and the
 * stream.  One call in flight per handle.
 */
#ifndef SN_LEVELSET_H
#define SN_LEVELSET_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sn_levelset sn_levelset; /* opaque */

/* nx, ny >= 2 nodes; dr, dz, delta > 0 finite (delta = the paper's grid size Delta, normally dr = dz).
 * Returns NULL on bad arguments, allocation failure or no sm_100 device (message: sn_levelset_last_error). */
sn_levelset* sn_levelset_create(int nx, int ny, double dr, double dz, double delta);

/* One re-initialisation.  S_old is read-only; S_new receives eq. (6); dist (may be NULL) receives the signed minimum
 * distance d.  S_new / dist must not alias S_old.  All work is enqueued on `stream` (cudaStream_t as void*), which is
 * synchronised before returning.  Returns the number of crossings (>= 0; 0 means S_new = S_old), -1 bad argument,
 * -2 CUDA error. */
int64_t sn_levelset_reinit(sn_levelset* h, const double* S_old, double* S_new, double* dist, void* stream);

/* Same with HOST buffers (H2D / D2H inside the call). */
int64_t sn_levelset_reinit_host(sn_levelset* h, const double* S_old_host, double* S_new_host, double* dist_host,
                                void* stream);

/* Counters of the last call: "crossings", "pairs" (nodes x crossings evaluated), "distance_ms" (device time of the
 * pairwise-distance kernel, CUDA events on the caller's stream), "total_ms", "launches".  Returns 0 or -1. */
int sn_levelset_get_stat(sn_levelset* h, const char* key, double* out);

void sn_levelset_destroy(sn_levelset* h);
const char* sn_levelset_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SN_LEVELSET_H */
