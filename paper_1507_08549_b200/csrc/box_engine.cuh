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

constexpr int kMaxTB = 12;     // max sweeps per launch (blocked path) / per interval and exchange (resident path)

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
    // ring duty (halo mode): second-layer columns / rows + the ring threads' private copies of their two edge cells
    static constexpr size_t ring_doubles = (size_t)2 * (BH + BW);    // + the static stash, 2 (BH + BW)
    static constexpr size_t ring_ds_doubles = ring_doubles + (size_t)2 * (BH + BW);   // + the DSMEM landing zone
    static_assert(NT % 32 == 0 && H % 2 == 0, "shape");
};

// A double with a 32-bit tag in each 8-byte half: {lo, tag, hi, tag}.  ASSUMPTION (the NCCL "LL" idiom): a 16-byte
// vector store may become visible in two pieces, but each naturally aligned 8-byte half {payload word, tag} is
// single-copy atomic, so a reader that sees the expected tag in BOTH halves has the whole value; no fence and no
// separate flag are needed (the producer's tag is the step number, unique within a solve phase).
__device__ __forceinline__ void ll_store(uint4* p, double v, unsigned tag) {
    const unsigned lo = (unsigned)__double2loint(v), hi = (unsigned)__double2hiint(v);
    asm volatile("st.volatile.global.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(lo), "r"(tag), "r"(hi), "r"(tag)
                 : "memory");
}
// the same store without the compiler barrier (the payload comes from registers; nothing has to be ordered before it)
__device__ __forceinline__ void ll_store_early(uint4* p, double v, unsigned tag) {
    const unsigned lo = (unsigned)__double2loint(v), hi = (unsigned)__double2hiint(v);
    asm volatile("st.volatile.global.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(lo), "r"(tag), "r"(hi), "r"(tag));
}
__device__ __forceinline__ uint4 ll_load(const uint4* p) {
    uint4 v;
    asm volatile("ld.volatile.global.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                 : "l"(p)
                 : "memory");
    return v;
}
// Same load, but not a compiler barrier for ordinary memory accesses: used to put a poll IN FLIGHT early (its result
// is validated by the tags when it is consumed), so that the L2 round trip overlaps the patch update.
__device__ __forceinline__ uint4 ll_load_early(const uint4* p) {
    uint4 v;
    asm volatile("ld.volatile.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ bool ll_ready(const uint4& v, unsigned tag) { return v.y == tag && v.w == tag; }
__device__ __forceinline__ double ll_value(const uint4& v) { return __hiloint2double((int)v.z, (int)v.x); }

// Every wait on another CTA is bounded: a poll gives up when *quit becomes non-zero (the solve is leaving the phase)
// or when the watchdog trips (budget exceeded here, or tripped elsewhere: *g_panic non-zero).  A tripped watchdog
// makes every later wait fall through, so the kernel always terminates; the host then reports status -2.
struct PollCtx {
    const volatile int* quit;    // shared memory
    volatile int* s_panic;       // shared memory
    int* g_panic;                // Ctl::panic of this member
    int* g_info;                 // Ctl::panic_tile, panic_arg
    int tile;
};
// The bound has two stages.  A poll count alone is a poor clock (a poll is an L2 round trip on an idle GPU but can be
// far slower under a profiler's replay, a debugger or a time-sliced GPU), so the count only decides WHEN to start
// looking at the clock: after kPollBudget polls (~1 s on an idle GPU) the wait notes %globaltimer and from then on
// gives up only once kWatchdogMs more wall-clock milliseconds (2^20 ns units) have passed without the awaited word.
constexpr unsigned kPollBudget = 1u << 21;
constexpr unsigned kWatchdogMs = 20000;
constexpr unsigned kPollTimed = 0x80000000u;    // top bit of the poll counter: stage two, low 31 bits = start time

__device__ __forceinline__ unsigned watchdog_now() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return (unsigned)(t >> 20) & 0x7fffffffu;
}

__device__ __forceinline__ void trip_watchdog(const PollCtx& c, int code, int arg) {
    if (atomicCAS(c.g_panic, 0, code) == 0) {
        c.g_info[0] = c.tile;
        c.g_info[1] = arg;
    }
    *c.s_panic = 1;
}
// true: stop waiting
__device__ __forceinline__ bool poll_giveup(const PollCtx& c, unsigned& n, int code, int arg) {
    if (*c.quit || *c.s_panic) return true;
    if (n & kPollTimed) {                                    // stage two: bounded by the clock (rare, slow path)
        if (*(volatile int*)c.g_panic) { *c.s_panic = 1; return true; }
        if (((watchdog_now() - n) & 0x7fffffffu) > kWatchdogMs) { trip_watchdog(c, code, arg); return true; }
        return false;
    }
    if ((++n & 63u) == 0u) {
        if (*(volatile int*)c.g_panic) { *c.s_panic = 1; return true; }
        if (n > kPollBudget) n = kPollTimed | watchdog_now();
    }
    return false;
}

// BAR = 0: the engine's barrier is __syncthreads(); BAR > 0: named barrier BAR over the first NT threads of the CTA
// (the resident kernel runs an extra service warp that must not take part in it).
// Rows per update group (BoxEngine::update_cells) for a kernel of `threads` threads with `minb` CTAs per SM: every
// chain in flight needs ~6 registers of temporaries and operands on top of the 8 H registers of phi, so the group
// grows with the registers per thread the launch bounds leave (measured on B200: profiles/r02_ilp.md).
#ifndef SNP_GROUP_ROWS_ROOMY
#define SNP_GROUP_ROWS_ROOMY 4
#endif
__host__ __device__ constexpr int group_rows_for(int threads, int minb) {
    const int warps = (threads + 63) / 64 * 2;                   // registers are allocated per pair of warps
    const int regs = 65536 / (minb * warps * 32) > 255 ? 255 : 65536 / (minb * warps * 32);
    return regs >= 160 ? SNP_GROUP_ROWS_ROOMY : 2;
}

template <int H, int TXN, int TYN, int BAR = 0, int GR = 2>
struct BoxEngine {
    using S = BoxShape<H, TXN, TYN>;
    static constexpr int BW = S::BW, BH = S::BH, LS = S::LS, PW = S::PW;

    static __device__ __forceinline__ void sync() {
        if (BAR == 0) __syncthreads();
        else asm volatile("bar.sync %0, %1;" ::"n"(BAR), "n"(S::NT) : "memory");
    }

    // shared memory
    double* fs;     // [BH][2][PW]     f; plane p holds the columns with (c & 1) == p, thread a's pair at [2a, 2a+1]
    double* exL;    // [BH][LS]        column 0 of thread a at [row][a+1]
    double* exR;    // [BH][LS]        column 3 of thread a at [row][a+1]
    double* exB;    // [TYN+2][2][PW]  bottom row of thread-row b at [b+1]
    double* exT;    // [TYN+2][2][PW]  top row of thread-row b at [b+1]
    double *l2W = nullptr, *l2E = nullptr, *l2S = nullptr, *l2N = nullptr, *stash = nullptr, *land = nullptr;   // ring duty only

    // Inbox of one tile: tagged packets it receives from its four neighbours, [E: BH][W: BH][N: BW][S: BW], each edge
    // split by colour so that the packets of one half-sweep are contiguous: slot(i) = (i & 1) * n/2 + (i >> 1).
    // A slot is written once per sweep with a strictly increasing tag, and its reader consumes tag t before the
    // writer can produce t + 2, so one buffer is enough.
    static constexpr int kInboxE = 0, kInboxW = BH, kInboxN = 2 * BH, kInboxS = 2 * BH + BW, kInboxPackets = 2 * (BH + BW);

    // Which neighbours exist and where their inboxes are.
    struct HaloLinks {
        uint4* own;                  // this tile's inbox
        uint4 *w, *e, *s, *n;        // neighbours' inboxes (NULL: no neighbour on that side)
        int rows;                    // box rows inside the grid (== BH except in the ragged last tile row), even
    };

    // per-thread state
    int a, b, rowbase;
    bool active = true;         // false: the patch lies outside the grid (ragged last tile row of the halo mode);
                                // such a thread never updates and keeps publishing the north ghosts as its bottom row
    double phi[H][4];
    double cEr[4], cWr[4];
    double iz2, D, wD;          // interior rows (uniform: the compiler keeps them in the constant bank / uniform registers)
    double D0, wD0;             // reflecting-equator row (uniform)
    bool mirror0;               // row q = 0 of this patch is the reflecting equator row
    // running maxima of the current sweep
    unsigned long long mres_k, mphi_k;     // exact keys
    float mres_f, mphi_f;                  // fast: |upper word| compared as fp32 (same order for finite values)
    unsigned long long mres0_k;            // the same maxima of |res| over the reflecting-equator row alone (rule 1, R16)
    float mres0_f;

    __device__ __forceinline__ void carve(double* base) {
        fs = base;
        exL = fs + S::f_doubles;
        exR = exL + S::lat_doubles;
        exB = exR + S::lat_doubles;
        exT = exB + S::vert_doubles;
    }
    // ring-duty arrays; `base` = first double after everything else the kernel keeps in dynamic shared memory
    __device__ __forceinline__ void carve_ring(double* base) {
        l2W = base;            // [BH]        column 1 of the box (second layer behind the west edge)
        l2E = l2W + BH;        // [BH]        column BW-2
        l2S = l2E + BH;        // [2][PW]     row 1, parity planes like exB
        l2N = l2S + BW;        // [2][PW]     row BH-2
        land = l2N + BW;       // [2][BH+BW]  cluster mode only: where the neighbours' st.async land, per colour
    }
    // [2][BH+BW] per colour: the ring thread's own edge cell.  A static __shared__ array of the kernel (a distinct
    // object: its stores do not hold back the loads of the patch update that follows the ring duty).
    __device__ __forceinline__ void bind_stash(double* p) { stash = p; }
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
        iz2 = g.iz2; D = g.D; wD = g.wD; D0 = g.D0; wD0 = g.wD0;
        mirror0 = (g.symmetry == 1 && gj0 == 0);
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
            exL[r * LS + TXN + 1] = (bx + BW == g.nr && by + r < g.nz) ? bE[by + r] : 0.0;   // east (rows past nz: ragged halo tile)
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
    template <bool RING = false>
    __device__ __forceinline__ void publish_all() {
        if (RING) {
#pragma unroll
            for (int q = 0; q < H; ++q) {
                if (a == 0) l2W[rowbase + q] = phi[q][1];
                if (a == TXN - 1) l2E[rowbase + q] = phi[q][2];
            }
            if (b == 0) {
                *reinterpret_cast<double2*>(l2S + 2 * a) = make_double2(phi[1][0], phi[1][2]);
                *reinterpret_cast<double2*>(l2S + PW + 2 * a) = make_double2(phi[1][1], phi[1][3]);
            }
            if (b == TYN - 1) {
                *reinterpret_cast<double2*>(l2N + 2 * a) = make_double2(phi[H - 2][0], phi[H - 2][2]);
                *reinterpret_cast<double2*>(l2N + PW + 2 * a) = make_double2(phi[H - 2][1], phi[H - 2][3]);
            }
        }
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
        mres0_k = 0ull; mres0_f = 0.0f;
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

    // One half-sweep of colour COL over the patch, then publish the updated edge cells and (SYNC) the barrier.
    template <int COL, int TRACK, bool SYNC = true, bool RING = false>
    __device__ __forceinline__ void half_sweep() {
        if (active) {
            update_cells<COL, TRACK, 0>();
            publish_colour<COL, RING>();
        }
        if (SYNC) sync();
    }
    // ring variant: the packets of this half-sweep were sent by the neighbours' ring duty at its start, so the poll can
    // be put in flight in the middle of the patch update; returns what it fetched (tags 0 if nothing was fetched)
    template <int COL, int TRACK>
    __device__ __forceinline__ uint4 half_sweep_ring(const HaloLinks& L) {
        uint4 pf = make_uint4(0u, 0u, 0u, 0u);
        const uint4* src = h_edge >= 0 ? recv_src<COL>(L) : nullptr;
        if (active) {
            update_cells<COL, TRACK, 0, true>(src, &pf);
            publish_colour<COL, true>();
        } else if (src) {
            pf = ll_load_early(src);
        }
        return pf;
    }
    // All cells of colour COL of the patch.  The updates of one colour are mutually independent, so they are issued in
    // groups of kGroupRows rows (2 cells each) STAGE BY STAGE: all operands of the group are fetched first, then the
    // 7-deep fp64 chains of the group's cells advance in lock step, so that each warp has 2 kGroupRows independent
    // dependency chains in flight instead of one (a single chain issues one fp64 instruction per ~8.4 clocks; measured
    // in profiles/r02_ilp.md).  The expression tree of every cell is sor_update's (R10), only the issue order differs.
    // PF (ring duty): after the last row, put this thread's poll of the neighbour's packet in flight (pf_src may be
    // NULL: nothing to receive); halo_recv consumes *pf.
    // GR (template argument): rows per group the kernel can afford with its register budget (group_rows_for below).
    static constexpr int kGroupRows = H % GR == 0 ? GR : 2;
    template <int COL, int TRACK, int WHICH, bool PF = false>
    __device__ __forceinline__ void update_cells(const uint4* pf_src = nullptr, uint4* pf = nullptr) {
        static_assert(WHICH == 0 && H % kGroupRows == 0, "whole patch, whole groups");
        // vertical outer neighbours of the bottom (q=0) and top (q=H-1) rows: other-colour cells of the rows outside
        constexpr int pb = COL & 1, pt = (H - 1 + COL) & 1;                 // column parity updated in those rows
        const double2 So = *reinterpret_cast<const double2*>(exT + (size_t)b * BW + pb * PW + 2 * a);
        const double2 No = *reinterpret_cast<const double2*>(exB + (size_t)(b + 2) * BW + pt * PW + 2 * a);
        constexpr int G = kGroupRows, NC = 2 * G;
#pragma unroll
        for (int q0 = 0; q0 < H; q0 += G) {
            double pE[NC], pW[NC], pN[NC], pS[NC], pC[NC], ff[NC], t[NC];
            // ---- operands
#pragma unroll
            for (int gq = 0; gq < G; ++gq) {
                const int q = q0 + gq;
                const int pq = (q + COL) & 1;                               // compile-time after unrolling
                const double outer = pq == 0 ? exR[(rowbase + q) * LS + a] : exL[(rowbase + q) * LS + a + 2];
                const double2 fv = *reinterpret_cast<const double2*>(fs + (size_t)(rowbase + q) * BW + pq * PW + 2 * a);
#pragma unroll
                for (int cc = 0; cc < 2; ++cc) {
                    const int c = pq + 2 * cc, i = 2 * gq + cc;
                    pW[i] = c == 0 ? outer : phi[q][c == 0 ? 0 : c - 1];
                    pE[i] = c == 3 ? outer : phi[q][c == 3 ? 3 : c + 1];
                    pN[i] = q == H - 1 ? (cc == 0 ? No.x : No.y) : phi[q == H - 1 ? q : q + 1][c];
                    pS[i] = q == 0 ? (cc == 0 ? So.x : So.y) : phi[q == 0 ? 0 : q - 1][c];
                    pC[i] = phi[q][c];
                    ff[i] = cc == 0 ? fv.x : fv.y;
                }
            }
            // ---- the chains, stage by stage (sor_update's tree)
#pragma unroll
            for (int i = 0; i < NC; ++i) t[i] = __dmul_rn(cEr[((q0 + i / 2 + COL) & 1) + 2 * (i & 1)], pE[i]);
#pragma unroll
            for (int i = 0; i < NC; ++i) t[i] = __fma_rn(cWr[((q0 + i / 2 + COL) & 1) + 2 * (i & 1)], pW[i], t[i]);
#pragma unroll
            for (int i = 0; i < NC; ++i) t[i] = __fma_rn(iz2, pN[i], t[i]);
#pragma unroll
            for (int i = 0; i < NC; ++i) t[i] = __fma_rn((q0 + i / 2 == 0 && mirror0) ? 0.0 : iz2, pS[i], t[i]);
#pragma unroll
            for (int i = 0; i < NC; ++i) t[i] = __fma_rn(-((q0 + i / 2 == 0 && mirror0) ? D0 : D), pC[i], t[i]);
#pragma unroll
            for (int i = 0; i < NC; ++i) t[i] = __dsub_rn(ff[i], t[i]);                                   // res
#pragma unroll
            for (int i = 0; i < NC; ++i) pC[i] = __fma_rn(-((q0 + i / 2 == 0 && mirror0) ? wD0 : wD), t[i], pC[i]);
#pragma unroll
            for (int i = 0; i < NC; ++i) {
                const int q = q0 + i / 2, c = ((q + COL) & 1) + 2 * (i & 1);
                phi[q][c] = pC[i];
                track<TRACK>(t[i], pC[i]);
                if (q == 0 && mirror0) {             // q is a compile-time constant: two predicated maxima per half-sweep
                    if (TRACK == kTrackExact) { const unsigned long long kr = abs_key(t[i]); mres0_k = kr > mres0_k ? kr : mres0_k; }
                    else if (TRACK == kTrackFast) mres0_f = fmaxf(mres0_f, fabsf(__int_as_float(__double2hiint(t[i]))));
                }
            }
        }
        if (PF) { if (pf_src) *pf = ll_load_early(pf_src); }
    }
    // publish the updated patch-edge cells of colour COL to the exchange arrays of the CTA
    template <int COL, bool RING = false>
    __device__ __forceinline__ void publish_colour() {
        constexpr int pb = COL & 1, pt = (H - 1 + COL) & 1;
        if (RING) {            // second layer behind the box edges: what the ring duty of the NEXT half-sweep reads
            constexpr int p1 = (1 + COL) & 1, pn = (H - 2 + COL) & 1;
#pragma unroll
            for (int q = 0; q < H; ++q) {
                const int pq = (q + COL) & 1;
                if (pq == 1) { if (a == 0) l2W[rowbase + q] = phi[q][1]; }
                else { if (a == TXN - 1) l2E[rowbase + q] = phi[q][2]; }
            }
            if (b == 0) *reinterpret_cast<double2*>(l2S + p1 * PW + 2 * a) = make_double2(phi[1][p1], phi[1][p1 + 2]);
            if (b == TYN - 1) *reinterpret_cast<double2*>(l2N + pn * PW + 2 * a) = make_double2(phi[H - 2][pn], phi[H - 2][pn + 2]);
        }
#pragma unroll
        for (int q = 0; q < H; ++q) {
            const int pq = (q + COL) & 1;
            if (pq == 0) exL[(rowbase + q) * LS + a + 1] = phi[q][0];
            else exR[(rowbase + q) * LS + a + 1] = phi[q][3];
        }
        *reinterpret_cast<double2*>(exB + (size_t)(b + 1) * BW + pb * PW + 2 * a) = make_double2(phi[0][pb], phi[0][pb + 2]);
        *reinterpret_cast<double2*>(exT + (size_t)(b + 1) * BW + pt * PW + 2 * a) =
            make_double2(phi[H - 1][pt], phi[H - 1][pt + 2]);
    }

    template <int TRACK>
    __device__ __forceinline__ void sweep() {
        half_sweep<0, TRACK>();
        half_sweep<1, TRACK>();
    }

    // ---- halo mode (box == owned tile; the neighbours' edge cells arrive every half-sweep) ------------------------
    // Fill the border slots on the box edges that have a neighbouring tile from a full state array (both colours);
    // called after set_borders() whenever the box is (re)loaded.
    __device__ __forceinline__ void load_halo_borders(const double* __restrict__ src, int nr, int nz, int bx, int by) {
        const int gi0 = bx + 4 * a, gj0 = by + rowbase;
        if (!active) return;
        if (a == TXN - 1 && bx + BW < nr) {
#pragma unroll
            for (int q = 0; q < H; ++q) exL[(rowbase + q) * LS + TXN + 1] = __ldcg(src + (size_t)(gj0 + q) * nr + bx + BW);
        }
        if (a == 0 && bx > 0) {
#pragma unroll
            for (int q = 0; q < H; ++q) exR[(rowbase + q) * LS + 0] = __ldcg(src + (size_t)(gj0 + q) * nr + bx - 1);
        }
        if (b == TYN - 1 && by + BH < nz) {
            const double* row = src + (size_t)(gj0 + H) * nr + gi0;
            double* dst = exB + (size_t)(TYN + 1) * BW + 2 * a;
            *reinterpret_cast<double2*>(dst) = make_double2(__ldcg(row), __ldcg(row + 2));
            *reinterpret_cast<double2*>(dst + PW) = make_double2(__ldcg(row + 1), __ldcg(row + 3));
        }
        if (b == 0 && by > 0) {
            const double* row = src + (size_t)(gj0 - 1) * nr + gi0;
            double* dst = exT + 2 * a;
            *reinterpret_cast<double2*>(dst) = make_double2(__ldcg(row), __ldcg(row + 2));
            *reinterpret_cast<double2*>(dst + PW) = make_double2(__ldcg(row + 1), __ldcg(row + 3));
        }
    }

    // Per-thread halo state, computed once (halo_bind).  RECEIVE: thread (edge, j) fetches ONE packet per half-sweep
    // from this tile's inbox and drops it into the engine's border slot:
    //   E (j < BH/2): the east tile's column 0,  row 2j + COL      W: the west tile's column BW-1, row 2j + 1 - COL
    //   N (j < BW/2): the north tile's row 0,    plane COL, pos j  S: the south tile's row BH-1,   plane 1 - COL, pos j
    // (plane p, position j <-> box column 4 (j >> 1) + 2 (j & 1) + p).  Where the CTA has enough warps every edge gets
    // whole warps of its own (no divergence between the four cases), else the threads are packed E | W | N | S.
    // SEND, plain variant: the owners of the box-edge cells send after their patch update (h_scol / h_srow).
    // SEND, ring variant: see ring_duty().
    // (the first poll is issued after the last patch row: any earlier position in the source changes nothing, ptxas
    // sinks the load to its first use -- profiles/r02_ring.md)
    int h_edge = -1;                 // 0 E, 1 W, 2 N, 3 S; -1: this thread receives nothing
    int h_j = 0;
    uint4* h_scol = nullptr;         // column edge: west (h_west) or east
    uint4* h_srow = nullptr;         // row edge: south (h_south) or north
    bool h_west = false, h_south = false;

    static constexpr int kWE = (BH / 2 + 31) / 32, kWB = (BW / 2 + 31) / 32;       // warps per column / row edge
    static constexpr bool kWarpEdges = (2 * kWE + 2 * kWB) * 32 <= S::NT;

    template <bool RING>
    __device__ __forceinline__ void halo_bind(const HaloLinks& L, int tid) {
        static_assert(BH + BW <= S::NT && TXN >= 2 && TYN >= 2, "halo mode: one packet per thread, one edge per axis");
        int e = -1, j = 0;
        if (kWarpEdges) {
            const int w = tid >> 5, l = tid & 31;
            if (w < kWE) { e = 0; j = w * 32 + l; }
            else if (w < 2 * kWE) { e = 1; j = (w - kWE) * 32 + l; }
            else if (w < 2 * kWE + kWB) { e = 2; j = (w - 2 * kWE) * 32 + l; }
            else if (w < 2 * kWE + 2 * kWB) { e = 3; j = (w - 2 * kWE - kWB) * 32 + l; }
            if (e >= 0 && j >= (e < 2 ? BH / 2 : BW / 2)) e = -1;
        } else {
            if (tid < BH / 2) { e = 0; j = tid; }
            else if (tid < BH) { e = 1; j = tid - BH / 2; }
            else if (tid < BH + BW / 2) { e = 2; j = tid - BH; }
            else if (tid < BH + BW) { e = 3; j = tid - BH - BW / 2; }
        }
        const bool have = e == 0 ? (L.e != nullptr && 2 * j < L.rows) : e == 1 ? (L.w != nullptr && 2 * j < L.rows)
                        : e == 2 ? L.n != nullptr : e == 3 ? L.s != nullptr : false;
        h_edge = have ? e : -1;
        h_j = j;
        if (e == 0) { h_src0 = kInboxE + j; h_sdelta = BH / 2; h_dst0 = (int)(exL - fs) + 2 * j * LS + TXN + 1; h_ddelta = LS; }
        else if (e == 1) { h_src0 = kInboxW + BH / 2 + j; h_sdelta = -(BH / 2); h_dst0 = (int)(exR - fs) + (2 * j + 1) * LS; h_ddelta = -LS; }
        else if (e == 2) { h_src0 = kInboxN + j; h_sdelta = BW / 2; h_dst0 = (int)(exB - fs) + (TYN + 1) * BW + j; h_ddelta = PW; }
        else if (e == 3) { h_src0 = kInboxS + BW / 2 + j; h_sdelta = -(BW / 2); h_dst0 = (int)(exT - fs) + PW + j; h_ddelta = -PW; }
        if (!RING && active) {
            if (a == 0 && L.w) { h_scol = L.w + kInboxE + rowbase / 2; h_west = true; }
            else if (a == TXN - 1 && L.e) { h_scol = L.e + kInboxW + rowbase / 2; }
            if (b == 0 && L.s) { h_srow = L.s + kInboxN + 2 * a; h_south = true; }
            else if (b == TYN - 1 && L.n) { h_srow = L.n + kInboxS + 2 * a; }
        }
    }

    // After the half-sweep of colour COL: the owners of this box's edge cells send the values just updated ...
    template <int COL>
    __device__ __forceinline__ void halo_send(unsigned tag) const {
        constexpr int pb = COL & 1, pt = (H - 1 + COL) & 1;
        if (h_scol) {
            if (h_west) {                    // my column 0 (rows with (q + COL) even) -> the west tile's E edge
#pragma unroll
                for (int q = 0; q < H; ++q)
                    if (((q + COL) & 1) == 0) ll_store(h_scol + (q & 1) * (BH / 2) + (q >> 1), phi[q][0], tag);
            } else {                         // my column 3 (rows with (q + COL) odd) -> the east tile's W edge
#pragma unroll
                for (int q = 0; q < H; ++q)
                    if (((q + COL) & 1) == 1) ll_store(h_scol + (q & 1) * (BH / 2) + (q >> 1), phi[q][3], tag);
            }
        }
        if (h_srow) {
            if (h_south) {                   // my bottom row -> the south tile's N edge
                ll_store(h_srow + pb * (BW / 2), phi[0][pb], tag);
                ll_store(h_srow + pb * (BW / 2) + 1, phi[0][pb + 2], tag);
            } else {                         // my top row -> the north tile's S edge
                ll_store(h_srow + pt * (BW / 2), phi[H - 1][pt], tag);
                ll_store(h_srow + pt * (BW / 2) + 1, phi[H - 1][pt + 2], tag);
            }
        }
    }

    // ... and every receiving thread fetches its ONE packet (coalesced, all four sides in flight at once) into the
    // border slot.  The poll gives up when the context says so.
    // receive addressing, linear in the colour: packet index in the inbox and border slot (doubles from fs)
    int h_src0 = 0, h_sdelta = 0, h_dst0 = 0, h_ddelta = 0;
    template <int COL>
    __device__ __forceinline__ const uint4* recv_src(const HaloLinks& L) const { return L.own + (h_src0 + COL * h_sdelta); }
    template <int COL>
    __device__ __forceinline__ double* recv_dst() const { return fs + (h_dst0 + COL * h_ddelta); }
    // `first`: a poll already in flight (half_sweep_ring), consumed before any new load is issued
    template <int COL>
    __device__ __forceinline__ void halo_recv(const HaloLinks& L, unsigned tag, const PollCtx& pc,
                                              uint4 first = make_uint4(0u, 0u, 0u, 0u)) {
        if (h_edge < 0) return;
        double* dst = recv_dst<COL>();
        if (ll_ready(first, tag)) { *dst = ll_value(first); return; }       // tags start at 1: all-zero never matches
        const uint4* src = recv_src<COL>(L);
        unsigned spins = 0;
        for (;;) {
            const uint4 v = ll_load(src);
            if (ll_ready(v, tag)) { *dst = ll_value(v); break; }
            if (poll_giveup(pc, spins, 1, (int)tag)) break;
        }
    }

    // ---- ring duty (halo mode): the box-edge cells are ALSO updated, one per thread, by the thread that receives on
    // that edge, FIRST THING in the half-sweep and straight from shared memory, and sent at once.  The packets then
    // travel while the patch update runs, so the neighbours find them when their own patch update is done: the period
    // of a half-sweep becomes max(patch update, ring duty + packet flight) instead of their sum.  The patch owners
    // update the same cells again later in the half-sweep from the same inputs with the same expression tree: the two
    // results are the same bits (R10), the owners' copy is the one the maxima and the result come from.
    //   Thread (edge, j), colour COL:   E: cell (BW-1, 2j + 1 - COL)    W: cell (0, 2j + COL)
    //                                   N: cell (plane 1 - COL pos j, BH-1)    S: cell (plane COL pos j, 0)
    // Inputs: the border slot (the neighbour tile's cell, received in the previous half-sweep), the two other-colour
    // cells along the edge (published by their owners in the previous half-sweep; the corner's comes from the other
    // edge's border slot), the second-layer cell behind it (l2*: published by its owner), f, and the cell's own old
    // value from the thread's private stash (the owner overwrites the published copy DURING this half-sweep).
    // CTA-uniform ring constants, kept in shared memory by the kernel
    struct RingConst {
        double cE_e, cW_e;           // coefficients of the box's last column (east edge)
        double cE_w, cW_w;           // ... first column (west edge)
        const double *cE, *cW;       // g.cE + bx, g.cW + bx (row-edge threads index them with their column)
        int mirror_box;              // the box's row 0 is the reflecting equator row
        int tile, ntx;               // cluster mode: rank of this tile in the cluster, tiles per tile row
    };

    // stash <- the current values of this thread's two edge cells; call after publish_all() + sync, then sync again
    __device__ __forceinline__ void ring_init() {
        if (h_edge < 0) return;
        const int j = h_j;
#pragma unroll
        for (int col = 0; col < 2; ++col) {
            double v;
            if (h_edge == 0) v = exR[(2 * j + 1 - col) * LS + TXN];
            else if (h_edge == 1) v = exL[(2 * j + col) * LS + 1];
            else if (h_edge == 2) v = exT[(size_t)TYN * BW + (1 - col) * PW + j];
            else v = exB[(size_t)BW + col * PW + j];
            stash[col * (BH + BW) + ring_slot()] = v;
        }
    }
    __device__ __forceinline__ int ring_slot() const {
        return h_edge == 0 ? h_j : h_edge == 1 ? BH / 2 + h_j : h_edge == 2 ? BH + h_j : BH + BW / 2 + h_j;
    }

    // One specialised straight-line body per edge: every address is (compile-time constant) + (stride) * j.
    template <int COL, int EDGE, bool DSM = false>
    __device__ __forceinline__ void ring_cell(const HaloLinks& L, const RingConst& rc, unsigned tag) {
        const int j = h_j;
        double pE, pW, pN, pS, fv, cE, cW;
        double cS = iz2, dg = D, ww = wD;
        double* st;
        uint4* out;
        if (EDGE < 2) {
            constexpr bool east = EDGE == 0;
            constexpr int r0 = east ? 1 - COL : COL;                         // r = 2 j + r0
            const int r = 2 * j + r0;
            const double* own_col = east ? exR + TXN : exL + 1;              // this edge column as published by its owners
            constexpr int pc = east ? BW - 1 : 0;                            // position of the column in a row of f / exB / exT
            cE = east ? rc.cE_e : rc.cE_w;
            cW = east ? rc.cW_e : rc.cW_w;
            st = stash + COL * (BH + BW) + (east ? 0 : BH / 2) + j;
            fv = fs[(size_t)r * BW + pc];
            pE = east ? exL[r * LS + TXN + 1] : l2W[r];
            pW = east ? l2E[r] : exR[r * LS];
            // the corner cells take their vertical neighbour from the row border (the neighbouring tile / the ghosts)
            pN = own_col[(r + 1 < BH ? r + 1 : r) * LS];
            if (r0 == 1 && r + 1 == BH) pN = exB[(size_t)(TYN + 1) * BW + pc];
            pS = own_col[(r > 0 ? r - 1 : r) * LS];
            if (r0 == 0 && r == 0) {
                pS = exT[pc];
                if (rc.mirror_box) { cS = 0.0; dg = D0; ww = wD0; }
            }
            out = east ? L.e + kInboxW + (1 - COL) * (BH / 2) + j : L.w + kInboxE + COL * (BH / 2) + j;
        } else {
            constexpr bool north = EDGE == 2;
            constexpr int pl = north ? 1 - COL : COL;                        // parity plane of my cell; column c = 2 j + pl
            constexpr int r = north ? BH - 1 : 0;
            const int pp = pl * PW + j;
            const double* own_row = north ? exT + (size_t)TYN * BW : exB + BW;   // this edge row as published by its owners
            cE = __ldg(rc.cE + 2 * j + pl);
            cW = __ldg(rc.cW + 2 * j + pl);
            st = stash + COL * (BH + BW) + BH + (north ? 0 : BW / 2) + j;
            fv = fs[(size_t)r * BW + pp];
            pN = north ? exB[(size_t)(TYN + 1) * BW + pp] : l2S[pp];
            pS = north ? l2N[pp] : exT[pp];
            if (pl == 1) {           // odd column: west neighbour = plane 0 [j], east = plane 0 [j + 1] or the east border
                pW = own_row[j];
                pE = own_row[j + 1 < PW ? j + 1 : j];
                if (j + 1 == PW) pE = exL[r * LS + TXN + 1];
            } else {                 // even column: west = plane 1 [j - 1] or the west border, east = plane 1 [j]
                pE = own_row[PW + j];
                pW = own_row[PW + (j > 0 ? j - 1 : j)];
                if (j == 0) pW = exR[r * LS];
            }
            out = north ? L.n + kInboxS + (1 - COL) * (BW / 2) + j : L.s + kInboxN + COL * (BW / 2) + j;
        }
        double res;
        const double pn = sor_update(cE, cW, iz2, cS, dg, ww, pE, pW, pN, pS, *st, fv, res);
        if (DSM) {
            // cluster mode: straight into the neighbour's landing zone (the slot of ITS receiving thread on the
            // opposite edge, same j) through distributed shared memory; the bytes are credited to its mbarrier[COL].
            // A landing slot of colour COL is rewritten two half-sweeps later, after the neighbour's packets of the
            // half-sweep in between have arrived here, which it sends only after it has consumed this one.
            const int nslot = EDGE == 0 ? BH / 2 + j : EDGE == 1 ? j : EDGE == 2 ? BH + BW / 2 + j : BH + j;
            const unsigned rank = (unsigned)(EDGE == 0 ? rc.tile + 1 : EDGE == 1 ? rc.tile - 1 : EDGE == 2 ? rc.tile + rc.ntx : rc.tile - rc.ntx);
            ds_store(ds_mapa(smem_u32(land + COL * (BH + BW) + nslot), rank), pn, ds_mapa(ds_bar + 8u * COL, rank));
        } else {
            ll_store_early(out, pn, tag);
        }
        *st = pn;
    }

    template <int COL, bool DSM = false>
    __device__ __forceinline__ void ring_duty(const HaloLinks& L, const RingConst& rc, unsigned tag) {
        if (h_edge == 0) ring_cell<COL, 0, DSM>(L, rc, tag);
        else if (h_edge == 1) ring_cell<COL, 1, DSM>(L, rc, tag);
        else if (h_edge == 2) ring_cell<COL, 2, DSM>(L, rc, tag);
        else if (h_edge == 3) ring_cell<COL, 3, DSM>(L, rc, tag);
    }
    // cluster mode, after ds_recv<COL>: every receiving thread moves its value from the landing zone to the border slot
    template <int COL>
    __device__ __forceinline__ void ds_ring_copy() {
        if (h_edge >= 0) *recv_dst<COL>() = land[COL * (BH + BW) + ring_slot()];
    }

    // ---- halo mode inside ONE thread-block cluster: distributed shared memory instead of L2 packets ----------------
    // When all tiles of a member fit in one cluster (<= 16 CTAs), an edge value is written straight into the
    // neighbour's border slot with st.async, which also credits its bytes to an mbarrier in the neighbour's shared
    // memory; the neighbour waits on that mbarrier (one per colour; the bytes it expects per half-sweep are fixed).
    // One hop of ~250 clocks instead of an L2 round trip, no polling of memory.  Every CTA runs the same number of
    // half-sweeps and consumes every message right after its own half-sweep, so no message is ever left over.
    unsigned ds_col = 0, ds_row = 0;     // shared-window address of my first target slot in the (identical) layout
    unsigned ds_col_rank = 0, ds_row_rank = 0;
    unsigned ds_bar = 0;                 // shared-window address of mbar[0]; mbar[1] follows
    unsigned ds_phase = 0;               // bit c: parity of the phase of mbar[c] to wait for next

    static __device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
    static __device__ __forceinline__ unsigned ds_mapa(unsigned addr, unsigned rank) {
        unsigned r;
        asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
        return r;
    }
    static __device__ __forceinline__ void ds_store(unsigned raddr, double v, unsigned rbar) {
        asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b64 [%0], %1, [%2];" ::"r"(raddr),
                     "l"(__double_as_longlong(v)), "r"(rbar)
                     : "memory");
    }
    static __device__ __forceinline__ void ds_arm(unsigned bar, unsigned bytes) {
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
    }
    static __device__ __forceinline__ bool ds_test(unsigned bar, unsigned parity) {
        unsigned ok;
        asm volatile(
            "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok)
            : "r"(bar), "r"(parity)
            : "memory");
        return ok != 0u;
    }
    // bytes this tile receives per half-sweep (both colours alike: rows and BW are even)
    static __device__ __forceinline__ unsigned ds_expected_bytes(const HaloLinks& L) {
        return 8u * (unsigned)((L.e ? L.rows / 2 : 0) + (L.w ? L.rows / 2 : 0) + (L.n ? BW / 2 : 0) + (L.s ? BW / 2 : 0));
    }
    // mbar: two 8-byte mbarriers in shared memory, initialised (count 1) and armed by thread 0 before the cluster sync
    __device__ __forceinline__ void ds_bind(const HaloLinks& L, const unsigned long long* mbar, int tile, int ntx) {
        static_assert(TXN >= 2 && TYN >= 2, "halo mode: one edge per axis");
        ds_bar = smem_u32(mbar);
        if (!active) return;
        if (a == 0 && L.w) { ds_col = smem_u32(exL + rowbase * LS + TXN + 1); ds_col_rank = tile - 1; h_west = true; h_scol = L.own; }
        else if (a == TXN - 1 && L.e) { ds_col = smem_u32(exR + rowbase * LS); ds_col_rank = tile + 1; h_scol = L.own; }
        if (b == 0 && L.s) { ds_row = smem_u32(exB + (size_t)(TYN + 1) * BW + 2 * a); ds_row_rank = tile - ntx; h_south = true; h_srow = L.own; }
        else if (b == TYN - 1 && L.n) { ds_row = smem_u32(exT + 2 * a); ds_row_rank = tile + ntx; h_srow = L.own; }
    }
    template <int COL>
    __device__ __forceinline__ void ds_send() const {
        constexpr int pb = COL & 1, pt = (H - 1 + COL) & 1;
        if (h_scol) {
            const unsigned base = ds_mapa(ds_col, ds_col_rank), bar = ds_mapa(ds_bar + 8u * COL, ds_col_rank);
#pragma unroll
            for (int q = 0; q < H; ++q) {
                const int pq = (q + COL) & 1;
                if (h_west ? pq == 0 : pq == 1) ds_store(base + (unsigned)(q * LS * 8), h_west ? phi[q][0] : phi[q][3], bar);
            }
        }
        if (h_srow) {
            const unsigned bar = ds_mapa(ds_bar + 8u * COL, ds_row_rank);
            if (h_south) {                   // my bottom row -> the south tile's north border
                const unsigned base = ds_mapa(ds_row + (unsigned)(pb * PW * 8), ds_row_rank);
                ds_store(base, phi[0][pb], bar);
                ds_store(base + 8u, phi[0][pb + 2], bar);
            } else {                         // my top row -> the north tile's south border
                const unsigned base = ds_mapa(ds_row + (unsigned)(pt * PW * 8), ds_row_rank);
                ds_store(base, phi[H - 1][pt], bar);
                ds_store(base + 8u, phi[H - 1][pt + 2], bar);
            }
        }
    }
    // wait for the neighbours' edge cells of colour COL; thread `arm` re-arms the mbarrier for its next phase
    template <int COL>
    __device__ __forceinline__ void ds_recv(unsigned expect_bytes, bool arm, const PollCtx& pc) {
        const unsigned bar = ds_bar + 8u * COL, parity = (ds_phase >> COL) & 1u;
        unsigned spins = 0;
        while (!ds_test(bar, parity)) {
            if (poll_giveup(pc, spins, 6, (int)parity)) break;
        }
        ds_phase ^= 1u << COL;
        if (arm) ds_arm(bar, expect_bytes);
    }

    // ---- block mode, small tiles: the whole owned patch travels as tagged packets once per interval ---------------
    // (two buffers by interval parity: an owner writes interval r + 2 only after every neighbour has consumed r)
    __device__ __forceinline__ void ll_store_patch(uint4* __restrict__ mail, unsigned tag, int nr, int gi0, int gj0) const {
#pragma unroll
        for (int q = 0; q < H; ++q) {
            uint4* row = mail + (size_t)(gj0 + q) * nr + gi0;
#pragma unroll
            for (int c = 0; c < 4; ++c) ll_store(row + c, phi[q][c], tag);
        }
    }
    __device__ __forceinline__ void ll_wait_patch(const uint4* __restrict__ mail, unsigned tag, int nr, int gi0, int gj0,
                                                  const PollCtx& pc) {
        unsigned spins = 0;
        bool done;
        do {
            done = true;
#pragma unroll
            for (int q = 0; q < H; ++q) {
                const uint4* row = mail + (size_t)(gj0 + q) * nr + gi0;
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const uint4 v = ll_load(row + c);
                    if (ll_ready(v, tag)) phi[q][c] = ll_value(v);
                    else done = false;
                }
            }
        } while (!done && !poll_giveup(pc, spins, 5, (int)tag));
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
