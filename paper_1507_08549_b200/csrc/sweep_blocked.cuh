// sweep_blocked.cuh -- steps a-2 + a-3 for grids / batches that do not fit on chip: temporal blocking with one
// launch per m sweeps.  PAPER.md:99 (SOR / Gauss-Seidel); PAPER.md:149 names the cost this removes ("data migration
// ... can take up even more time than using CPU solely"): every sweep of the plain streaming path moves 24 B per
// cell through L2/HBM, here it is (16 B x box + 8 B x tile) per m sweeps.  Design: DESIGN.md section 6.
//
//  * Every member grid is cut into tiles; one CTA per (tile, member) per launch.  The CTA loads its BW x BH box
//    (tile + a margin of 2m cells towards every neighbour) of phi into registers and f into shared memory, runs
//    n <= m full sweeps with the BoxEngine, and stores the tile (the part that is still exact) into the OTHER phi
//    buffer (Jacobi-style double buffering between launches, Gauss-Seidel red-black inside: bit-identical to the
//    oracle's ordering because a colour's updates are mutually independent, R10).
//  * a-3: per-sweep maxima go warp -> CTA -> atomicMax into per-sweep slots.  FAST tracking keeps only the upper 32
//    bits of |res| and |phi| (one FMNMX each per update instead of a 64-bit compare/select chain); that gives R_k
//    to within 2^-20, enough to know that the rule has NOT fired.  When it may have, the launch is re-run from the
//    untouched source buffer with EXACT tracking, the crossing sweep k* is found exactly, and if k* is inside the
//    launch the first k*-k0 sweeps are replayed once more (untracked).  The returned phi has exactly k* sweeps
//    applied and `residual` is the exact R_k*, like the oracle's.
//  * The "director": the last CTA of a member to finish a launch evaluates the slots and writes the member's next
//    action into its control block; the next launch just reads it.  The host only enqueues launches and polls
//    `done` a chunk behind.
#pragma once
#include "box_engine.cuh"
#include "tiling.h"

namespace snp {

struct BlkParams {
    Geom g;
    int ntx, nty;              // tiles in r and z
    int ow, oh;                // nominal owned tile size (multiples of 4 and H)
    int m;                     // sweeps per launch
    int max_sweeps;
    int force_exact;           // 1: always track exactly (exact history)
    int nbatch;
    const double* rho;         // [nbatch][nz][nr]
    double* buf[2];            // buf[0] = caller's phi_inout, buf[1] = workspace, both [nbatch][nz][nr]
    const double* bE;          // [nbatch][nz]
    const double* bN;          // [nbatch][nr]
    const double* bS;          // [nbatch][nr]
    unsigned int* slots_f;     // [nbatch][2*cap]  FAST maxima: upper words of max|res|, max|phi| per sweep
    unsigned long long* slots_x;   // [nbatch][2*cap]  EXACT maxima keys
    int slot_stride;           // 2*cap
    int hist_stride;           // cap
    Ctl* ctl;                  // [nbatch]
    double* hist;              // [nbatch][cap]
};

// First action of a member (after the moments pass has written maxf).  grid = nbatch, 1 thread.
static __global__ void k_blocked_init(Ctl* __restrict__ ctl, int m, int max_sweeps, int force_exact) {
    Ctl* c = ctl + blockIdx.x;
    if (threadIdx.x != 0) return;
    const int n = max_sweeps < m ? max_sweeps : m;
    c->action = kActAdvance;
    c->src = 0;
    c->k0 = 0;
    c->n = n;
    c->track = (force_exact || n == max_sweeps) ? kTrackExact : kTrackFast;
    c->arrived = 0u;
}

// The director: called by ONE thread of the last CTA of member `c` after a launch that executed (action, src, k0,
// n, track).  All maxima of the launch are final and visible.  Writes the next action (or the result).
__device__ inline void blocked_direct(const BlkParams& p, Ctl* c, int member, int action, int src, int k0, int n, int track,
                                      const unsigned int* sf, const unsigned long long* sx, double* hist) {
    const Geom& g = p.g;
    const unsigned int* s0f = g.slots0_f + (size_t)member * g.slots0_stride;      // rule 1: equator-row maxima
    const unsigned long long* s0x = g.slots0_x + (size_t)member * g.slots0_stride;
    auto finish = [&](int final_buf, int sweeps, int status, double R) {
        if (final_buf == 0) {
            c->sweeps = sweeps; c->status = status; c->residual = R;
            c->action = kActSkip;
            __threadfence();
            c->done = 1;
        } else {
            c->fin_sweeps = sweeps; c->fin_status = status; c->fin_R = R;
            c->action = kActCopy;
            c->src = final_buf;
        }
    };
    if (action == kActCopy || action == kActReplay) {
        // replay wrote buf[src^1]; copy wrote buf[0]
        const int final_buf = action == kActCopy ? 0 : (src ^ 1);
        finish(final_buf, c->fin_sweeps, c->fin_status, c->fin_R);
        return;
    }
    // action was kActAdvance or kActRedo: sweeps k0+1 .. k0+n were applied, new state in buf[src^1]
    double Rlast = 0.0;
    if (track == kTrackExact) {
        for (int s = 0; s < n; ++s) {
            const int k = k0 + s + 1;
            const double R = stop_value(g, __ldcg(sx + 2 * (k - 1)), __ldcg(sx + 2 * (k - 1) + 1),
                                        g.rule != 0 ? __ldcg(s0x + k - 1) : 0ull, c->maxf);
            hist[k - 1] = R;
            Rlast = R;
            const bool bad = is_nonfinite(R);
            if (bad || (g.tol > 0.0 && R <= g.tol)) {
                const int status = bad ? -3 : 0;
                if (s == n - 1) {
                    finish(src ^ 1, k, status, R);
                } else {                               // crossing inside the launch: replay k - k0 sweeps from buf[src]
                    c->fin_sweeps = k; c->fin_status = status; c->fin_R = R;
                    c->action = kActReplay;
                    c->n = k - k0;
                    c->track = kTrackNone;             // src, k0 unchanged
                }
                return;
            }
        }
    } else {
        // FAST: upper words only.  R_lo <= R_k (up to rounding, covered by the factor); the rule cannot have fired
        // at sweep k unless R_lo <= tol.  A poisoned (NaN) slot also makes the launch a candidate.
        bool candidate = false;
        for (int s = 0; s < n; ++s) {
            const int k = k0 + s + 1;
            const unsigned long long kr = (unsigned long long)__ldcg(sf + 2 * (k - 1)) << 32;
            const unsigned long long kp = ((unsigned long long)__ldcg(sf + 2 * (k - 1) + 1) << 32) | 0xffffffffull;
            const double R_lo = stop_value(g, kr, kp, g.rule != 0 ? (unsigned long long)__ldcg(s0f + k - 1) << 32 : 0ull, c->maxf);
            hist[k - 1] = R_lo;
            if (is_nonfinite(R_lo) || (g.tol > 0.0 && R_lo <= g.tol * 1.000000001)) candidate = true;
        }
        if (candidate) {                               // same launch again from the untouched source, exact maxima
            c->action = kActRedo;
            c->track = kTrackExact;                    // src, k0, n unchanged
            return;
        }
    }
    const int k1 = k0 + n;
    if (k1 >= p.max_sweeps) {                          // budget exhausted (the last launch is always EXACT)
        finish(src ^ 1, k1, g.tol > 0.0 ? 1 : 0, Rlast);
        return;
    }
    const int nn = (p.max_sweeps - k1 < p.m) ? p.max_sweeps - k1 : p.m;
    c->action = kActAdvance;
    c->src = src ^ 1;
    c->k0 = k1;
    c->n = nn;
    c->track = (p.force_exact || k1 + nn == p.max_sweeps) ? kTrackExact : kTrackFast;
}

template <int H, int TXN, int TYN>
struct BlkShape {
    using S = BoxShape<H, TXN, TYN>;
    static constexpr size_t smem_bytes = sizeof(double) * S::engine_doubles + sizeof(unsigned long long) * 2 * kMaxTB * S::NW;
};

// grid = (ntx*nty, nbatch), block = TXN*TYN threads.
template <int H, int TXN, int TYN, int MINB>
__global__ void __launch_bounds__(TXN* TYN, MINB) k_sor_blocked(const BlkParams p) {
    using S = BoxShape<H, TXN, TYN>;
    constexpr int BW = S::BW, BH = S::BH, NT = S::NT, NW = S::NW;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ int s_act[5];
    __shared__ unsigned int s_last;

    const int member = blockIdx.y;
    Ctl* c = p.ctl + member;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) {
        s_act[0] = c->action; s_act[1] = c->src; s_act[2] = c->k0; s_act[3] = c->n; s_act[4] = c->track;
    }
    __syncthreads();
    const int action = s_act[0], src = s_act[1], k0 = s_act[2], n = s_act[3], track = s_act[4];
    if (action == kActSkip) return;

    const Geom& g = p.g;
    const size_t ncell = (size_t)g.nr * g.nz;
    const int ntiles = p.ntx * p.nty;
    const int tile = blockIdx.x;
    const int tx = tile % p.ntx, ty = tile / p.ntx;
    const int h = 2 * p.m;
    // owned tile [x0,x1) x [y0,y1) and box origin (bx,by), all aligned to (4,H)
    const int x0 = tx * p.ow, x1 = min(g.nr, x0 + p.ow);
    const int y0 = ty * p.oh, y1 = min(g.nz, y0 + p.oh);
    const int bx = box_origin(x0, h, 4, BW, g.nr);
    const int by = box_origin(y0, h, H, BH, g.nz);

    BoxEngine<H, TXN, TYN, 0, group_rows_for(TXN * TYN, MINB)> E;
    E.carve(reinterpret_cast<double*>(smem_raw));
    unsigned long long* smax = reinterpret_cast<unsigned long long*>(E.exT + S::vert_doubles);   // [2*kMaxTB][NW]
    E.bind_thread(tid);
    const int gi0 = bx + 4 * E.a, gj0 = by + H * E.b;
    const bool own = gi0 >= x0 && gi0 < x1 && gj0 >= y0 && gj0 < y1;
    const bool row0_warp = __any_sync(0xffffffffu, g.symmetry == 1 && gj0 == 0);     // holds equator-row cells

    const double* srcp = p.buf[src] + (size_t)member * ncell;
    double* dstp = p.buf[src ^ 1] + (size_t)member * ncell;

    if (action == kActCopy) {
        if (own) {
            E.load_patch(srcp, g.nr, gi0, gj0);
            E.store_patch(dstp, g.nr, gi0, gj0);
        }
    } else {
        E.load_patch(srcp, g.nr, gi0, gj0);
        E.load_f(p.rho + (size_t)member * ncell, g.nr, gi0, gj0);
        E.load_coeffs(g, gi0, gj0);
        E.set_borders(g, bx, by, p.bE + (size_t)member * g.nz, p.bN + (size_t)member * g.nr,
                      p.bS + (size_t)member * g.nr, tid, NT);
        E.publish_all();
        __syncthreads();
        if (track == kTrackFast) {
            for (int s = 0; s < n; ++s) {
                E.reset_maxima();
                E.template half_sweep<0, kTrackFast>();
                E.template half_sweep<1, kTrackFast, false>();
                // warp reduction BEFORE the sweep's last barrier: its latency hides in the barrier wait
                if (g.rule != 0 && row0_warp) {          // rule 1 (R16): equator-row maximum, straight to its slot
                    const unsigned w0 = __reduce_max_sync(0xffffffffu, own ? __float_as_uint(E.mres0_f) : 0u);
                    if (lane == 0) atomicMax(g.slots0_f + (size_t)member * g.slots0_stride + k0 + s, w0);
                }
                const unsigned wr = __reduce_max_sync(0xffffffffu, own ? __float_as_uint(E.mres_f) : 0u);
                const unsigned wp = __reduce_max_sync(0xffffffffu, own ? __float_as_uint(E.mphi_f) : 0u);
                if (lane == 0) {
                    smax[(2 * s) * NW + warp] = wr;
                    smax[(2 * s + 1) * NW + warp] = wp;
                }
                E.sync();
            }
        } else if (track == kTrackExact) {
            for (int s = 0; s < n; ++s) {
                E.reset_maxima();
                E.template half_sweep<0, kTrackExact>();
                E.template half_sweep<1, kTrackExact, false>();
                if (g.rule != 0 && row0_warp) {
                    const unsigned long long w0 = warp_max_key(own ? E.mres0_k : 0ull);
                    if (lane == 0) atomicMax(g.slots0_x + (size_t)member * g.slots0_stride + k0 + s, w0);
                }
                const unsigned long long wr = warp_max_key(own ? E.mres_k : 0ull);
                const unsigned long long wp = warp_max_key(own ? E.mphi_k : 0ull);
                if (lane == 0) {
                    smax[(2 * s) * NW + warp] = wr;
                    smax[(2 * s + 1) * NW + warp] = wp;
                }
                E.sync();
            }
        } else {
            for (int s = 0; s < n; ++s) E.template sweep<kTrackNone>();
        }
        if (own) E.store_patch(dstp, g.nr, gi0, gj0);
        if (track != kTrackNone) {
            // any non-finite owned value persists (NaN/Inf never relax away): poison this launch's maxima
            const int anybad = __syncthreads_or(own && E.any_nonfinite());    // also orders the smax writes
            if (warp == 0) {
                for (int idx = lane; idx < 2 * n; idx += 32) {
                    unsigned long long v = 0ull;
                    for (int w = 0; w < NW; ++w) {
                        const unsigned long long t = smax[idx * NW + w];
                        v = t > v ? t : v;
                    }
                    const size_t slot = (size_t)member * p.slot_stride + 2 * (size_t)(k0 + (idx >> 1)) + (idx & 1);
                    if (track == kTrackFast) atomicMax(p.slots_f + slot, anybad ? 0x7ff80000u : (unsigned)v);
                    else atomicMax(p.slots_x + slot, anybad ? 0x7ff8000000000000ull : v);
                }
            }
        }
    }
    // arrive; the last CTA of this member directs the next launch
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = atomicAdd(&c->arrived, 1u);
    __syncthreads();
    if (s_last == (unsigned)(ntiles - 1) && tid == 0) {
        __threadfence();
        c->arrived = 0u;
        blocked_direct(p, c, member, action, src, k0, n, track, p.slots_f + (size_t)member * p.slot_stride,
                       p.slots_x + (size_t)member * p.slot_stride, p.hist + (size_t)member * p.hist_stride);
    }
}

}  // namespace snp
