// sweep_resident.cuh -- steps a-2 + a-3 as ONE persistent cooperative kernel with phi resident on chip.
//
// PAPER.md:99 "successive overrelaxation method with the Gauss-Seidel method"; PAPER.md:149 names the cost this
// design removes ("data migration, if not handled carefully, can take up even more time than using CPU solely").
// Discretisation / ordering / pinned arithmetic: DESIGN.md R1, R3, R7, R10.  Design: DESIGN.md §6.
//
//  * The grid is cut into tiles, one CTA per tile, all co-resident (cooperative launch).  A CTA works on a fixed
//    BW x BH "box" of cells = its owned tile plus a margin of 2m cells towards every neighbour.
//  * Thread (a,b) keeps a 4 x H patch of phi in REGISTERS for the whole solve; f = 4 pi rho sits in shared memory.
//    A red (black) update needs the 4 black (red) neighbours: inside the patch they are registers; across patch
//    edges they come from small shared-memory exchange arrays the owning thread publishes after each half-sweep.
//  * Temporal blocking: m full sweeps run between two inter-CTA exchanges.  Every box cell is updated every
//    half-sweep; cells closer than t to an interior box edge are stale after t half-sweeps, so after 2m
//    half-sweeps exactly the owned tile (distance >= 2m) is still exact -- no trapezoid bookkeeping, and a
//    colour's updates are mutually independent, so tiling cannot change a bit of the result.
//  * Exchange: owners store their patches to the global phi buffer of parity (epoch & 1), release a per-tile
//    epoch flag, acquire the flags of the tiles their box overlaps and reload the non-owned patches (L2 traffic,
//    ld.global.cg).  No grid-wide barrier on the critical path.
//  * a-3: every owned cell's pre-update |res| and post-update |phi| feed per-sweep maxima (DSETP/FSEL on |x|),
//    reduced warp -> CTA -> global atomicMax on order-preserving u64 keys in slot k.  The stopping decision for
//    the sweeps of epoch e-1 is taken by every CTA (identically) at the end of epoch e, one epoch late, so the
//    wait for the slowest CTA is off the critical path; the state two epochs back is still intact in the other
//    phi buffer, so the crossing sweep k* is then REPLAYED exactly from it (<= m sweeps): the returned phi has
//    exactly k* sweeps applied, like the oracle's.
#pragma once
#include "box_engine.cuh"
#include "sweep_blocked.cuh"
#include "tiling.h"

namespace snp {


struct ResParams {
    Geom g;
    int ntx, nty;              // tiles in r and z
    int ow, oh;                // nominal owned tile size (multiples of 4 and H)
    int m;                     // sweeps per epoch
    int max_sweeps;
    const double* rho;
    double* buf[3];            // state of epoch e lives in buf[e % 3]; buf[0] = caller's phi_inout (initial guess,
                               // final result), buf[1..2] = workspace
    const double* bE;
    const double* bN;
    const double* bS;
    unsigned long long* slots; // [2*max_sweeps] per-sweep (max|res|, max|phi|) keys
    Ctl* ctl;
    double* hist;
    unsigned int* flags;       // [ntiles] last epoch whose state this tile has published
    unsigned int* arrived;     // [nepochs+2] CTAs that have posted the maxima of epoch e
    unsigned int* gbar;        // single-use grid barrier counter
};

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u32(unsigned* p, unsigned v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void red_release_add_u32(unsigned* p, unsigned v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void spin_until_ge(const unsigned* p, unsigned want) {
    while (ld_acquire_u32(p) < want) __nanosleep(20);
}

template <int H, int TXN, int TYN>
struct ResShape {
    static constexpr int BW = 4 * TXN, BH = H * TYN, NT = TXN * TYN, NW = NT / 32;
    static constexpr int LS = TXN + 2;                         // row stride of the lateral exchange arrays
    static constexpr size_t smem_bytes =
        sizeof(double) * ((size_t)BH * BW + 2 * (size_t)BH * LS + 2 * (size_t)(TYN + 2) * BW) +
        sizeof(unsigned long long) * 2 * kMaxTB * NW;
};

// Position of column c of a 4-group in the colour-permuted layout [c0, c2, c1, c3].
__device__ __forceinline__ constexpr int perm4(int c) { return (c & 1) * 2 + (c >> 1); }

template <int H, int TXN, int TYN>
__global__ void __launch_bounds__(TXN* TYN, 1) k_sor_resident(const ResParams p) {
    using S = ResShape<H, TXN, TYN>;
    constexpr int BW = S::BW, BH = S::BH, NT = S::NT, NW = S::NW, LS = S::LS;
    static_assert(NT % 32 == 0 && H % 2 == 0 && H <= 8, "shape");

    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* fs = reinterpret_cast<double*>(smem_raw);          // [BH][BW]   f, colour-permuted per 4-group
    double* exL = fs + (size_t)BH * BW;                        // [BH][LS]   column 0 of thread a at [row][a+1]
    double* exR = exL + (size_t)BH * LS;                       // [BH][LS]   column 3 of thread a at [row][a+1]
    double* exB = exR + (size_t)BH * LS;                       // [TYN+2][BW] bottom row of thread-row b at [b+1]
    double* exT = exB + (size_t)(TYN + 2) * BW;                // [TYN+2][BW] top row of thread-row b at [b+1]
    unsigned long long* smax = reinterpret_cast<unsigned long long*>(exT + (size_t)(TYN + 2) * BW);  // [2*kMaxTB][NW]
    __shared__ int s_k;            // decision broadcast: crossing sweep (0 = none)
    __shared__ double s_R;

    const Geom& g = p.g;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int a = tid % TXN, b = tid / TXN;
    const int ntiles = p.ntx * p.nty;
    const int tile = blockIdx.x;
    const int tx = tile % p.ntx, ty = tile / p.ntx;
    const int m = p.m, h = 2 * m;

    // owned tile [x0,x1) x [y0,y1) and box origin (bx,by), all aligned to (4,H)
    const int x0 = tx * p.ow, x1 = min(g.nr, x0 + p.ow);
    const int y0 = ty * p.oh, y1 = min(g.nz, y0 + p.oh);
    const int bx = box_origin(x0, h, 4, BW, g.nr);
    const int by = box_origin(y0, h, H, BH, g.nz);
    const int gi0 = bx + 4 * a, gj0 = by + H * b;
    const bool own = gi0 >= x0 && gi0 < x1 && gj0 >= y0 && gj0 < y1;
    const int rowbase = H * b;

    // tiles whose owned cells this box overlaps (their flags gate the halo reload)
    const int ntx0 = bx / p.ow, ntx1 = (bx + BW - 1) / p.ow;
    const int nty0 = by / p.oh, nty1 = (by + BH - 1) / p.oh;
    const int nnb = (ntx1 - ntx0 + 1) * (nty1 - nty0 + 1);

    // per-thread constants
    double cEr[4], cWr[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        cEr[c] = g.cE[gi0 + c];
        cWr[c] = g.cW[gi0 + c];
    }
    const bool mirror0 = (g.symmetry == 1 && gj0 == 0);
    const double cS0 = mirror0 ? 0.0 : g.iz2;
    const double diag0 = mirror0 ? g.D0 : g.D;
    const double w0 = mirror0 ? g.wD0 : g.wD;

    double phi[H][4];

    auto load_patch = [&](const double* src) {
#pragma unroll
        for (int q = 0; q < H; ++q) {
            const double2* s2 = reinterpret_cast<const double2*>(src + (size_t)(gj0 + q) * g.nr + gi0);
            const double2 v0 = __ldcg(s2), v1 = __ldcg(s2 + 1);
            phi[q][0] = v0.x; phi[q][1] = v0.y; phi[q][2] = v1.x; phi[q][3] = v1.y;
        }
    };
    auto store_patch = [&](double* dst) {
#pragma unroll
        for (int q = 0; q < H; ++q) {
            double2* d2 = reinterpret_cast<double2*>(dst + (size_t)(gj0 + q) * g.nr + gi0);
            __stcg(d2, make_double2(phi[q][0], phi[q][1]));
            __stcg(d2 + 1, make_double2(phi[q][2], phi[q][3]));
        }
    };
    // publish every edge value of the patch (both colours) to the exchange arrays
    auto publish_all = [&]() {
#pragma unroll
        for (int q = 0; q < H; ++q) {
            exL[(rowbase + q) * LS + a + 1] = phi[q][0];
            exR[(rowbase + q) * LS + a + 1] = phi[q][3];
        }
        double* bb = exB + (size_t)(b + 1) * BW + 4 * a;
        double* tt = exT + (size_t)(b + 1) * BW + 4 * a;
        *reinterpret_cast<double2*>(bb) = make_double2(phi[0][0], phi[0][2]);
        *reinterpret_cast<double2*>(bb + 2) = make_double2(phi[0][1], phi[0][3]);
        *reinterpret_cast<double2*>(tt) = make_double2(phi[H - 1][0], phi[H - 1][2]);
        *reinterpret_cast<double2*>(tt + 2) = make_double2(phi[H - 1][1], phi[H - 1][3]);
    };

    // ---- one-time set-up: f into shared memory, constant borders of the exchange arrays, initial phi ----------
#pragma unroll
    for (int q = 0; q < H; ++q) {
        const double2* r2 = reinterpret_cast<const double2*>(p.rho + (size_t)(gj0 + q) * g.nr + gi0);
        const double2 v0 = __ldg(r2), v1 = __ldg(r2 + 1);
        double* fr = fs + (size_t)(rowbase + q) * BW + 4 * a;
        *reinterpret_cast<double2*>(fr) = make_double2(__dmul_rn(kFourPi, v0.x), __dmul_rn(kFourPi, v1.x));
        *reinterpret_cast<double2*>(fr + 2) = make_double2(__dmul_rn(kFourPi, v0.y), __dmul_rn(kFourPi, v1.y));
    }
    for (int r = tid; r < BH; r += NT) {
        exR[r * LS + 0] = 0.0;                                              // west of the box (cW = 0 on the axis)
        exL[r * LS + TXN + 1] = (bx + BW == g.nr) ? p.bE[by + r] : 0.0;     // east: Dirichlet ghost or stale margin
        exL[r * LS + 0] = 0.0;
        exR[r * LS + TXN + 1] = 0.0;
    }
    for (int c = tid; c < BW; c += NT) {
        const int gi = bx + (c & ~3) + ((c & 3) == 0 ? 0 : (c & 3) == 1 ? 2 : (c & 3) == 2 ? 1 : 3);  // inverse of perm4
        exT[c] = (by == 0 && g.symmetry == 0) ? p.bS[gi] : 0.0;             // south ghost (unused when mirrored)
        exB[(size_t)(TYN + 1) * BW + c] = (by + BH == g.nz) ? p.bN[gi] : 0.0;  // north ghost or stale margin
        exB[c] = 0.0;
        exT[(size_t)(TYN + 1) * BW + c] = 0.0;
    }
    load_patch(p.buf[0]);
    publish_all();
    __syncthreads();

    // ---- one half-sweep of colour COL over the thread's patch ------------------------------------------------
    double mres = 0.0, mphi = 0.0;
    auto half_sweep = [&](auto colTag, auto trackTag) {
        constexpr int COL = decltype(colTag)::value;
        constexpr bool TRACK = decltype(trackTag)::value;
        // vertical outer neighbours of the bottom (q=0) and top (q=H-1) rows: other-colour cells of the rows outside
        constexpr int pb = COL & 1, pt = (H - 1 + COL) & 1;                 // first updated column in those rows
        const double2 So = *reinterpret_cast<const double2*>(exT + (size_t)b * BW + 4 * a + 2 * pb);
        const double2 No = *reinterpret_cast<const double2*>(exB + (size_t)(b + 2) * BW + 4 * a + 2 * pt);
#pragma unroll
        for (int q = 0; q < H; ++q) {
            constexpr int dummy = 0;
            (void)dummy;
            const int pq = (q + COL) & 1;                                   // compile-time after unrolling
            const double outer = pq == 0 ? exR[(rowbase + q) * LS + a] : exL[(rowbase + q) * LS + a + 2];
            const double2 fv = *reinterpret_cast<const double2*>(fs + (size_t)(rowbase + q) * BW + 4 * a + 2 * pq);
            const double cS = q == 0 ? cS0 : g.iz2;
            const double dg = q == 0 ? diag0 : g.D;
            const double ww = q == 0 ? w0 : g.wD;
#pragma unroll
            for (int cc = 0; cc < 2; ++cc) {
                const int c = pq + 2 * cc;
                const double pW = c == 0 ? outer : phi[q][c == 0 ? 0 : c - 1];
                const double pE = c == 3 ? outer : phi[q][c == 3 ? 3 : c + 1];
                const double pN = q == H - 1 ? (cc == 0 ? No.x : No.y) : phi[q == H - 1 ? q : q + 1][c];
                const double pS = q == 0 ? (cc == 0 ? So.x : So.y) : phi[q == 0 ? 0 : q - 1][c];
                double res;
                const double pn = sor_update(cEr[c], cWr[c], g.iz2, cS, dg, ww, pE, pW, pN, pS, phi[q][c],
                                             cc == 0 ? fv.x : fv.y, res);
                phi[q][c] = pn;
                if (TRACK) {
                    const bool ur = own & (fabs(res) > mres);
                    mres = ur ? fabs(res) : mres;
                    const bool up = own & (fabs(pn) > mphi);
                    mphi = up ? fabs(pn) : mphi;
                }
            }
        }
        // publish the updated edge cells of this colour
#pragma unroll
        for (int q = 0; q < H; ++q) {
            const int pq = (q + COL) & 1;
            if (pq == 0) exL[(rowbase + q) * LS + a + 1] = phi[q][0];
            else exR[(rowbase + q) * LS + a + 1] = phi[q][3];
        }
        *reinterpret_cast<double2*>(exB + (size_t)(b + 1) * BW + 4 * a + 2 * pb) = make_double2(phi[0][pb], phi[0][pb + 2]);
        *reinterpret_cast<double2*>(exT + (size_t)(b + 1) * BW + 4 * a + 2 * pt) =
            make_double2(phi[H - 1][pt], phi[H - 1][pt + 2]);
        __syncthreads();
    };
    using C0 = std::integral_constant<int, 0>;
    using C1 = std::integral_constant<int, 1>;

    // Decision for the sweeps of epoch ee (all CTAs evaluate the same final slot values -> same answer).
    // Returns the first sweep k of that epoch whose ratio fires (non-finite, or <= tol when tol > 0), else 0.
    auto check_epoch = [&](int ee) -> int {
        const int kfirst = (ee - 1) * m + 1;
        const int nsw = min(m, p.max_sweeps - (ee - 1) * m);
        if (tid == 0) spin_until_ge(p.arrived + ee, (unsigned)ntiles);
        __syncthreads();
        if (warp == 0) {
            bool fire = false;
            double R = 0.0;
            if (lane < nsw) {
                const unsigned long long kr = __ldcg(p.slots + 2 * (size_t)(kfirst + lane - 1));
                const unsigned long long kp = __ldcg(p.slots + 2 * (size_t)(kfirst + lane - 1) + 1);
                R = stop_ratio(kr, kp, p.ctl->maxf, g.D);
                fire = is_nonfinite(R) || (g.tol > 0.0 && R <= g.tol);
            }
            const unsigned bal = __ballot_sync(0xffffffffu, fire);
            const int first = bal ? __ffs(bal) - 1 : -1;
            if (tile == 0 && lane < nsw && (first < 0 || lane <= first)) p.hist[kfirst + lane - 1] = R;
            if (lane == (first < 0 ? nsw - 1 : first)) {
                s_k = first < 0 ? 0 : kfirst + first;
                s_R = R;
            }
        }
        __syncthreads();
        return s_k;
    };

    // ---- epoch loop ------------------------------------------------------------------------------------------
    // End of epoch e:  store state e -> release flag  |  post maxima, arrive  |  acquire neighbour flags -> reload
    // margins  |  decide epoch e-1 while those loads are in flight.  State e overwrites state e-3, which nobody can
    // still be reading: the decision for epoch e-2 (taken during the end of epoch e-1) waited for every CTA to have
    // finished epoch e-2.  The state before any epoch whose sweeps are still undecided therefore stays intact.
    int done = 0, e = 0, kstar = 0, e_cross = 0;
    while (done < p.max_sweeps) {
        ++e;
        const int nsw = min(m, p.max_sweeps - done);
        for (int s = 0; s < nsw; ++s) {
            mres = 0.0;
            mphi = 0.0;
            half_sweep(C0{}, std::true_type{});
            half_sweep(C1{}, std::true_type{});
            const unsigned long long wr = warp_max_key(dbits(mres)), wp = warp_max_key(dbits(mphi));
            if (lane == 0) {
                smax[(2 * s) * NW + warp] = wr;
                smax[(2 * s + 1) * NW + warp] = wp;
            }
        }
        const bool last = done + nsw >= p.max_sweeps;
        double* cur = p.buf[e % 3];
        if (!last && own) store_patch(cur);
        // any non-finite owned value persists (NaN/Inf never relax away): poison this epoch's maxima
        bool bad = false;
        if (own) {
#pragma unroll
            for (int q = 0; q < H; ++q)
#pragma unroll
                for (int c = 0; c < 4; ++c) bad |= !(fabs(phi[q][c]) < INFINITY);
        }
        const int anybad = __syncthreads_or(bad);            // also: every thread's state stores are issued
        if (!last && tid == 0) st_release_u32(p.flags + tile, (unsigned)e);
        if (warp == 0) {
            for (int idx = lane; idx < 2 * nsw; idx += 32) {
                unsigned long long v = 0ull;
                for (int w = 0; w < NW; ++w) {
                    const unsigned long long t = smax[idx * NW + w];
                    v = t > v ? t : v;
                }
                if (anybad) v = 0x7ff8000000000000ull;
                atomicMax(p.slots + 2 * (size_t)(done + (idx >> 1)) + (idx & 1), v);
            }
            __syncwarp();
            if (lane == 0) red_release_add_u32(p.arrived + e, 1u);
        }
        done += nsw;
        if (last) {
            if (e >= 2) {
                kstar = check_epoch(e - 1);
                if (kstar) { e_cross = e - 1; break; }
            }
            kstar = check_epoch(e);
            if (kstar) e_cross = e;
            break;
        }
        if (warp == NW - 1) {
            for (int n = lane; n < nnb; n += 32) {
                const int nx = ntx0 + n % (ntx1 - ntx0 + 1), ny = nty0 + n / (ntx1 - ntx0 + 1);
                spin_until_ge(p.flags + ny * p.ntx + nx, (unsigned)e);
            }
        }
        __syncthreads();
        if (!own) load_patch(cur);
        if (e >= 2) {
            kstar = check_epoch(e - 1);
            if (kstar) { e_cross = e - 1; break; }
        }
        publish_all();
        __syncthreads();
    }

    // ---- finish ----------------------------------------------------------------------------------------------
    if (kstar && !(e_cross == e && kstar == done)) {
        // the rule fired at sweep kstar of epoch e_cross: replay it exactly from the state before that epoch
        const int es = e_cross - 1;
        const int r = kstar - es * m;
        load_patch(p.buf[es % 3]);
        __syncthreads();
        if (tid == 0) {                      // everyone has read its box before anyone overwrites buf[0]
            red_release_add_u32(p.gbar, 1u);
            spin_until_ge(p.gbar, (unsigned)ntiles);
        }
        __syncthreads();
        publish_all();
        __syncthreads();
        for (int s = 0; s < r; ++s) {
            half_sweep(C0{}, std::false_type{});
            half_sweep(C1{}, std::false_type{});
        }
    }
    if (own) store_patch(p.buf[0]);
    if (tile == 0 && tid == 0) {
        Ctl* c = p.ctl;
        const double R = s_R;
        if (kstar) {
            c->sweeps = kstar;
            c->residual = R;
            c->status = is_nonfinite(R) ? -3 : 0;
        } else {
            c->sweeps = p.max_sweeps;
            c->residual = R;
            c->status = g.tol > 0.0 ? 1 : 0;
        }
        c->done = 1;
    }
}

}  // namespace snp
