// box_engine.cuh -- the on-chip red-black SOR engine shared by the resident and the blocked sweep kernels
// (steps a-2 + a-3).  PAPER.md:99 "successive overrelaxation method with the Gauss-Seidel method"; ordering,
// coefficients and the pinned expression tree are DESIGN.md R1, R3, R7, R10; the stopping maxima are R9.
//
// One CTA owns a BW x BH "box" of cells.  Thread (a,b) keeps a 4 x H patch of phi in REGISTERS; f = 4 pi rho sits in
// shared memory.  A red (black) update needs the 4 black (red) neighbours: inside the patch they are registers;
// across patch edges they come from small shared-memory exchange arrays the owning thread publishes after each
// half-sweep (one __syncthreads per half-sweep).  Every box cell is updated every half-sweep; what the values
// outside the box are (Dirichlet ghosts, or stale margins that the caller discards) is the caller's business.
//
// Shared-memory layouts are chosen so that every 128-bit access of a warp has a 16-byte lane stride
// (conflict-free): f and the vertical exchange rows are split into two column-parity planes.
#pragma once
#include <type_traits>

#include "common.cuh"

namespace snp {

enum TrackMode : int {
    kTrackNone = 0,    // replay: no maxima
    kTrackExact = 1,   // exact max|res|, max|phi_new| as order-preserving u64 keys
    kTrackFast = 2,    // upper 32 bits only (a lower bound within 2^-20 relative); the exact value is recovered by an
                       // exact re-run of the few sweeps where it can matter
};

template <int H, int TXN, int TYN>
struct BoxShape {
    static constexpr int BW = 4 * TXN, BH = H * TYN, NT = TXN * TYN, NW = NT / 32;
    static constexpr int LS = TXN + 2;                         // row stride of the lateral exchange arrays
    static constexpr int PW = 2 * TXN;                         // doubles per parity plane of one row
    static constexpr size_t f_doubles = (size_t)BH * BW;
    static constexpr size_t lat_doubles = (size_t)BH * LS;
    static constexpr size_t vert_doubles = (size_t)(TYN + 2) * BW;
    static constexpr size_t engine_doubles = f_doubles + 2 * lat_doubles + 2 * vert_doubles;
    static_assert(NT % 32 == 0 && H % 2 == 0, "shape");
};

template <int H, int TXN, int TYN>
struct BoxEngine {
    using S = BoxShape<H, TXN, TYN>;
    static constexpr int BW = S::BW, BH = S::BH, LS = S::LS, PW = S::PW;

    // shared memory
    double* fs;     // [BH][2][PW]     f; plane p holds the columns with (c & 1) == p, thread a's pair at [2a, 2a+1]
    double* exL;    // [BH][LS]        column 0 of thread a at [row][a+1]
    double* exR;    // [BH][LS]        column 3 of thread a at [row][a+1]
    double* exB;    // [TYN+2][2][PW]  bottom row of thread-row b at [b+1]
    double* exT;    // [TYN+2][2][PW]  top row of thread-row b at [b+1]

    // per-thread state
    int a, b, rowbase;
    double phi[H][4];
    double cEr[4], cWr[4];
    double iz2, D, wD;          // interior rows
    double cS0, diag0, w0;      // row q = 0 of this patch (differs on the reflecting equator)
    // running maxima of the current sweep
    unsigned long long mres_k, mphi_k;     // exact keys
    float mres_f, mphi_f;                  // fast: |upper word| compared as fp32 (same order for finite values)

    __device__ __forceinline__ void carve(double* base) {
        fs = base;
        exL = fs + S::f_doubles;
        exR = exL + S::lat_doubles;
        exB = exR + S::lat_doubles;
        exT = exB + S::vert_doubles;
    }
    __device__ __forceinline__ void bind_thread(int tid) {
        a = tid % TXN;
        b = tid / TXN;
        rowbase = H * b;
    }
    // position of box column c inside its parity plane
    static __device__ __forceinline__ int plane_pos(int c) { return ((c >> 2) << 1) + ((c >> 1) & 1); }

    // coefficients of the 4 columns starting at global column gi0 and of patch row 0 at global row gj0
    __device__ __forceinline__ void load_coeffs(const Geom& g, int gi0, int gj0) {
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            cEr[c] = g.cE[gi0 + c];
            cWr[c] = g.cW[gi0 + c];
        }
        iz2 = g.iz2; D = g.D; wD = g.wD;
        const bool mirror0 = (g.symmetry == 1 && gj0 == 0);
        cS0 = mirror0 ? 0.0 : g.iz2;
        diag0 = mirror0 ? g.D0 : g.D;
        w0 = mirror0 ? g.wD0 : g.wD;
    }

    // f = 4 pi rho of this thread's patch into shared memory (rho row pitch nr, 16-byte aligned rows)
    __device__ __forceinline__ void load_f(const double* __restrict__ rho, int nr, int gi0, int gj0) {
#pragma unroll
        for (int q = 0; q < H; ++q) {
            const double2* r2 = reinterpret_cast<const double2*>(rho + (size_t)(gj0 + q) * nr + gi0);
            const double2 v0 = __ldg(r2), v1 = __ldg(r2 + 1);
            double* fr = fs + (size_t)(rowbase + q) * BW + 2 * a;
            *reinterpret_cast<double2*>(fr) = make_double2(__dmul_rn(kFourPi, v0.x), __dmul_rn(kFourPi, v1.x));
            *reinterpret_cast<double2*>(fr + PW) = make_double2(__dmul_rn(kFourPi, v0.y), __dmul_rn(kFourPi, v1.y));
        }
    }

    // Values just outside the box: Dirichlet ghosts where the box touches the outer edge of the grid, 0 elsewhere
    // (there the neighbouring cells are stale margin anyway).  bx, by = box origin; called by all NT threads.
    __device__ __forceinline__ void set_borders(const Geom& g, int bx, int by, const double* __restrict__ bE,
                                                const double* __restrict__ bN, const double* __restrict__ bS, int tid,
                                                int nthreads) {
        for (int r = tid; r < BH; r += nthreads) {
            exR[r * LS + 0] = 0.0;                                              // west of the box (cW = 0 on the axis)
            exL[r * LS + TXN + 1] = (bx + BW == g.nr) ? bE[by + r] : 0.0;       // east
            exL[r * LS + 0] = 0.0;
            exR[r * LS + TXN + 1] = 0.0;
        }
        for (int c = tid; c < BW; c += nthreads) {
            const int pos = (c & 1) * PW + plane_pos(c);
            exT[pos] = (by == 0 && g.symmetry == 0) ? bS[bx + c] : 0.0;         // south ghost (unused when mirrored)
            exB[(size_t)(TYN + 1) * BW + pos] = (by + BH == g.nz) ? bN[bx + c] : 0.0;   // north
            exB[pos] = 0.0;
            exT[(size_t)(TYN + 1) * BW + pos] = 0.0;
        }
    }

    __device__ __forceinline__ void load_patch(const double* __restrict__ src, int nr, int gi0, int gj0) {
#pragma unroll
        for (int q = 0; q < H; ++q) {
            const double2* s2 = reinterpret_cast<const double2*>(src + (size_t)(gj0 + q) * nr + gi0);
            const double2 v0 = __ldcg(s2), v1 = __ldcg(s2 + 1);
            phi[q][0] = v0.x; phi[q][1] = v0.y; phi[q][2] = v1.x; phi[q][3] = v1.y;
        }
    }
    __device__ __forceinline__ void store_patch(double* __restrict__ dst, int nr, int gi0, int gj0) const {
#pragma unroll
        for (int q = 0; q < H; ++q) {
            double2* d2 = reinterpret_cast<double2*>(dst + (size_t)(gj0 + q) * nr + gi0);
            __stcg(d2, make_double2(phi[q][0], phi[q][1]));
            __stcg(d2 + 1, make_double2(phi[q][2], phi[q][3]));
        }
    }
    // publish every edge value of the patch (both colours) to the exchange arrays
    __device__ __forceinline__ void publish_all() {
#pragma unroll
        for (int q = 0; q < H; ++q) {
            exL[(rowbase + q) * LS + a + 1] = phi[q][0];
            exR[(rowbase + q) * LS + a + 1] = phi[q][3];
        }
        double* bb = exB + (size_t)(b + 1) * BW + 2 * a;
        double* tt = exT + (size_t)(b + 1) * BW + 2 * a;
        *reinterpret_cast<double2*>(bb) = make_double2(phi[0][0], phi[0][2]);
        *reinterpret_cast<double2*>(bb + PW) = make_double2(phi[0][1], phi[0][3]);
        *reinterpret_cast<double2*>(tt) = make_double2(phi[H - 1][0], phi[H - 1][2]);
        *reinterpret_cast<double2*>(tt + PW) = make_double2(phi[H - 1][1], phi[H - 1][3]);
    }

    __device__ __forceinline__ void reset_maxima() {
        mres_k = 0ull; mphi_k = 0ull;
        mres_f = 0.0f; mphi_f = 0.0f;
    }

    template <int TRACK>
    __device__ __forceinline__ void track(double res, double pn) {
        if (TRACK == kTrackExact) {
            const unsigned long long kr = abs_key(res), kp = abs_key(pn);
            mres_k = kr > mres_k ? kr : mres_k;
            mphi_k = kp > mphi_k ? kp : mphi_k;
        } else if (TRACK == kTrackFast) {
            mres_f = fmaxf(mres_f, fabsf(__int_as_float(__double2hiint(res))));
            mphi_f = fmaxf(mphi_f, fabsf(__int_as_float(__double2hiint(pn))));
        }
    }

    // One half-sweep of colour COL over the patch, then publish the updated edge cells and __syncthreads().
    template <int COL, int TRACK>
    __device__ __forceinline__ void half_sweep() {
        // vertical outer neighbours of the bottom (q=0) and top (q=H-1) rows: other-colour cells of the rows outside
        constexpr int pb = COL & 1, pt = (H - 1 + COL) & 1;                 // column parity updated in those rows
        const double2 So = *reinterpret_cast<const double2*>(exT + (size_t)b * BW + pb * PW + 2 * a);
        const double2 No = *reinterpret_cast<const double2*>(exB + (size_t)(b + 2) * BW + pt * PW + 2 * a);
#pragma unroll
        for (int q = 0; q < H; ++q) {
            const int pq = (q + COL) & 1;                                   // compile-time after unrolling
            const double outer = pq == 0 ? exR[(rowbase + q) * LS + a] : exL[(rowbase + q) * LS + a + 2];
            const double2 fv = *reinterpret_cast<const double2*>(fs + (size_t)(rowbase + q) * BW + pq * PW + 2 * a);
            const double cS = q == 0 ? cS0 : iz2;
            const double dg = q == 0 ? diag0 : D;
            const double ww = q == 0 ? w0 : wD;
#pragma unroll
            for (int cc = 0; cc < 2; ++cc) {
                const int c = pq + 2 * cc;
                const double pW = c == 0 ? outer : phi[q][c == 0 ? 0 : c - 1];
                const double pE = c == 3 ? outer : phi[q][c == 3 ? 3 : c + 1];
                const double pN = q == H - 1 ? (cc == 0 ? No.x : No.y) : phi[q == H - 1 ? q : q + 1][c];
                const double pS = q == 0 ? (cc == 0 ? So.x : So.y) : phi[q == 0 ? 0 : q - 1][c];
                double res;
                const double pn = sor_update(cEr[c], cWr[c], iz2, cS, dg, ww, pE, pW, pN, pS, phi[q][c],
                                             cc == 0 ? fv.x : fv.y, res);
                phi[q][c] = pn;
                track<TRACK>(res, pn);
            }
        }
        // publish the updated edge cells of this colour
#pragma unroll
        for (int q = 0; q < H; ++q) {
            const int pq = (q + COL) & 1;
            if (pq == 0) exL[(rowbase + q) * LS + a + 1] = phi[q][0];
            else exR[(rowbase + q) * LS + a + 1] = phi[q][3];
        }
        *reinterpret_cast<double2*>(exB + (size_t)(b + 1) * BW + pb * PW + 2 * a) = make_double2(phi[0][pb], phi[0][pb + 2]);
        *reinterpret_cast<double2*>(exT + (size_t)(b + 1) * BW + pt * PW + 2 * a) =
            make_double2(phi[H - 1][pt], phi[H - 1][pt + 2]);
        __syncthreads();
    }

    template <int TRACK>
    __device__ __forceinline__ void sweep() {
        half_sweep<0, TRACK>();
        half_sweep<1, TRACK>();
    }

    // any non-finite value in the patch (NaN/Inf never relax away)
    __device__ __forceinline__ bool any_nonfinite() const {
        bool bad = false;
#pragma unroll
        for (int q = 0; q < H; ++q)
#pragma unroll
            for (int c = 0; c < 4; ++c) bad |= !(fabs(phi[q][c]) < INFINITY);
        return bad;
    }
};

// Exact max of order-preserving u64 keys across a warp with two 32-bit REDUX steps.
__device__ __forceinline__ unsigned long long warp_max_key(unsigned long long k) {
    const unsigned hi = (unsigned)(k >> 32), lo = (unsigned)k;
    const unsigned mh = __reduce_max_sync(0xffffffffu, hi);
    const unsigned ml = __reduce_max_sync(0xffffffffu, hi == mh ? lo : 0u);
    return ((unsigned long long)mh << 32) | ml;
}

}  // namespace snp
