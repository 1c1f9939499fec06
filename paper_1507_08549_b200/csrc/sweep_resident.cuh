// sweep_resident.cuh -- steps a-2 + a-3 as ONE persistent cooperative kernel with phi resident on chip.
//
// PAPER.md:99 "successive overrelaxation method with the Gauss-Seidel method"; PAPER.md:149 names the cost this
// design removes ("data migration, if not handled carefully, can take up even more time than using CPU solely").
// Discretisation / ordering / pinned arithmetic: DESIGN.md R1, R3, R7, R10.  Design: DESIGN.md section 6.
//
//  * The grid (of every batch member) is cut into tiles, one CTA per tile, all co-resident (cooperative launch).
//    Thread (a,b) of a CTA keeps a 4 x H patch of phi in REGISTERS for the whole solve, f = 4 pi rho sits in shared
//    memory (BoxEngine, box_engine.cuh).  Two ways of coupling the tiles:
//      - halo mode: box == owned tile.  After every half-sweep the edge cells of the colour just updated go to the
//        four neighbouring tiles and theirs come back into the border slots of the engine.  No redundant work;
//        where registers allow, the patch-edge cells are updated and sent first so that the packets travel while
//        the rest of the patch is updated.  For grids that fill the chip.
//      - block mode (temporal blocking): box = owned tile + a margin of 2m cells towards every neighbour; m full
//        sweeps run between two exchanges.  Every box cell is updated every half-sweep, cells closer than t to an
//        interior box edge are stale after t half-sweeps, so after 2m half-sweeps exactly the owned tile is still
//        exact; then the margins are refilled from the neighbours' tiles.  For grids that leave the chip idle.
//    In both modes a colour's updates are mutually independent, so tiling cannot change a bit of the result (R10).
//  * Exchange.  Halo mode: every edge value travels as a 16-byte packet carrying the half-sweep number in both
//    8-byte halves (ll_store / ll_load) into the neighbour's per-tile inbox; every receiving thread polls exactly
//    ONE packet (strong loads of one thread do not pipeline: measured ~+75 clocks per extra packet, profiles/
//    r01_microbench_b200.txt), so an exchange costs one L2 round trip and needs no fence and no flag.  Block mode:
//    the tile is stored to the checkpoint ring anyway; one release-store of a per-tile flag publishes it and the
//    neighbours refill their margins with ordinary (pipelined) loads after an acquire-poll of the flags of the tiles
//    their box overlaps.  Tiny tiles (H = 2, <= 256 cells) send their patches as tagged packets instead.
//    Halo mode with all tiles of a member in ONE thread-block cluster (DS): the edge values go straight into the
//    neighbour's border slots in distributed shared memory with st.async, which credits their bytes to an mbarrier
//    (one per colour) the neighbour waits on -- ~580 clocks per exchange instead of ~2300 through L2.
//  * a-3: per-sweep maxima of |res| and |phi_new| over the owned cells go warp -> CTA -> (service warp) atomicMax
//    into per-sweep global slots.  An extra SERVICE WARP per CTA does all of that and the stopping decision, so the
//    fences and L2 round trips of the reduction never stall the sweeps: the compute warps only hand it their maxima
//    at the end of every interval (Q sweeps) and run at most one interval ahead of its decisions.
//  * Main phase: FAST maxima (upper 32 bits of the doubles; one FMNMX per value).  They bound R_k from below within
//    2^-20, enough to know that the rule has NOT fired.  When it may have (interval r_c), every CTA stops, the
//    state at the start of r_c is reloaded from the checkpoint ring (each CTA stores its tile once per interval)
//    and the ENDGAME runs interval by interval with EXACT maxima until the first sweep k* with R_k <= tol; if k* is
//    inside an interval, its first sweeps are REPLAYED from the checkpoint.  The returned phi has exactly k* sweeps
//    applied and `residual` is the exact R_k*, like the oracle's (R_k is not monotone, so nothing may be skipped).
#pragma once
#include "box_engine.cuh"
#include "tiling.h"

namespace snp {

constexpr int kResRing = 3;          // checkpoint ring depth (main phase runs <= 1 interval ahead of the decision)
constexpr unsigned kTagEndgame = 1u << 28, kTagReplay = 2u << 28;

struct ResParams {
    Geom g;
    int halo;                  // 1: halo mode, 0: block mode (the kernel's HALO template argument)
    int ll;                    // block mode: 1 = margins travel as tagged packets (small tiles), 0 = tile flags + ring loads
    int ntx, nty;              // tiles in r and z
    int ow, oh;                // nominal owned tile size (halo mode: the box size)
    int m;                     // block mode: sweeps per exchange (== Q)
    int Q;                     // sweeps per interval (report / checkpoint / decision granularity)
    int max_sweeps;
    int force_exact;           // 1: exact maxima in every interval (exact history; every interval decided before the next)
    const double* rho;         // [nb][ncell]
    double* phi;               // [nb][ncell]  initial guess in, result out
    double* ring;              // [nb][kResRing][ncell]  checkpoints: state after interval r in ring[r % kResRing]
    uint4* mail;               // halo mode: [nb][ntiles][2(BH+BW)] inboxes of tagged packets; block mode with ll: [nb][2][ncell]
    unsigned int* flags;       // block mode: [nb][ntiles] last interval (phase tag + r) whose state the tile has published
    const double* bE;          // [nb][nz]
    const double* bN;          // [nb][nr]
    const double* bS;          // [nb][nr]
    unsigned int* slots_f;     // [nb][2*cap]  FAST maxima (upper words) per sweep
    unsigned long long* slots_x;   // [nb][2*cap]  EXACT maxima keys per sweep
    int slot_stride, hist_stride;
    unsigned int* arrived;     // [nb][2][nint+2]  CTAs that have reported interval r (main / endgame)
    int arr_stride;            // nint + 2
    unsigned int* gbar;        // [nb]  monotone grid-barrier counter
    Ctl* ctl;                  // [nb]
    double* hist;              // [nb][cap]
    long long* prof;           // optional [ctas][8] SM-clock counters of thread 0 of every CTA ("prof" option), else NULL
    double* gr;                // optional fused epilogue (NEXT-1, R15): [nb][ncell] g_r, g_z = -grad phi of the result, else NULL
    double* gz;
};

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned ld_relaxed_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u32(unsigned* p, unsigned v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void red_release_add_u32(unsigned* p, unsigned v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// One report of the compute warps to the service warp (shared memory, double-buffered by sequence parity).
struct ResReport {
    int r;          // interval (1-based)
    int k0;         // sweeps applied before it
    int n;          // sweeps in it
    int exact;      // 1: exact maxima (endgame), 0: FAST
    int bad;        // a non-finite owned value was seen
    int quit;       // 1: no more reports
};

// What the service warp hands back (shared memory).
struct ResDecision {
    volatile int seq;        // last report sequence number fully processed
    volatile int stop;       // main phase: a FAST candidate (or a non-finite value) was found in interval stop_r
    volatile int stop_r;
    volatile int stop_seq;   // ... by the decision of the report with this sequence number
    volatile int fire_k;     // endgame: first sweep whose exact ratio fires in the last decided interval (0: none)
    volatile int fire_bad;   // ... and whether it is non-finite
    volatile double R;       // exact ratio at fire_k, else of the last sweep of the interval
};

template <int H, int TXN, int TYN>
struct ResShape {
    using S = BoxShape<H, TXN, TYN>;
    static constexpr int NT = S::NT, NW = S::NW, NTHREADS = S::NT + 32;
    static constexpr size_t smax_entries = (size_t)2 * 2 * kMaxTB * NW;       // [parity][2Q][NW]
    static constexpr size_t smem_bytes = sizeof(double) * S::engine_doubles + sizeof(unsigned long long) * smax_entries;
    static constexpr size_t smem_bytes_ring = smem_bytes + sizeof(double) * S::ring_doubles;
    static constexpr size_t smem_bytes_ring_ds = smem_bytes + sizeof(double) * S::ring_ds_doubles;
};

// grid = (ntx*nty, nbatch), block = TXN*TYN + 32 threads (the last warp is the service warp), cooperative launch.
// RING (halo mode through L2 packets): ring duty -- every box-edge cell is also updated and sent by a receiving thread
// at the very start of the half-sweep, so that the packets travel during the patch update (BoxEngine::ring_duty).
// DS (halo mode, all tiles of a member in one thread-block cluster): edges travel through distributed shared memory.
template <int H, int TXN, int TYN, int MINB, bool HALO, bool RING, bool DS = false>
__global__ void __launch_bounds__(TXN* TYN + 32, MINB) k_sor_resident(const ResParams p) {
    static_assert(!RING || HALO, "ring duty belongs to the halo mode");
    using S = BoxShape<H, TXN, TYN>;
    using RS = ResShape<H, TXN, TYN>;
    constexpr int BW = S::BW, BH = S::BH, NT = S::NT, NW = S::NW;
    using Engine = BoxEngine<H, TXN, TYN, 1, group_rows_for(TXN * TYN + 32, MINB)>;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ ResReport s_rep[2];
    __shared__ ResDecision s_dec;
    __shared__ int s_bad;
    __shared__ int s_panic;        // watchdog tripped (here or in another CTA): every wait falls through
    __shared__ int s_zero;         // a quit word that never fires (endgame / replay polls)
    __shared__ __align__(8) unsigned long long s_mbar[2];   // DS: one mbarrier per colour, credited by the neighbours' st.async
    __shared__ long long s_pf[8];  // in-kernel profile of thread 0 ("prof" option)
    __shared__ typename Engine::HaloLinks s_links;   // halo mode: inboxes of this tile and its neighbours
    __shared__ typename Engine::RingConst s_ring;    // ring duty: CTA-uniform constants
    __shared__ double s_stash[RING ? 2 * (BoxShape<H, TXN, TYN>::BH + BoxShape<H, TXN, TYN>::BW) : 1];

    const Geom& g = p.g;
    const int member = blockIdx.y;
    const size_t ncell = (size_t)g.nr * g.nz;
    const int ntiles = p.ntx * p.nty;
    const int tile = blockIdx.x;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int Q = p.Q;
    const int R_last = (p.max_sweeps + Q - 1) / Q;          // number of intervals
    unsigned long long* smax =
        reinterpret_cast<unsigned long long*>(smem_raw + sizeof(double) * S::engine_doubles);   // [2][2*kMaxTB][NW]
    Ctl* ctl = p.ctl + member;
    unsigned int* arrived = p.arrived + (size_t)member * 2 * p.arr_stride;

    if (tid == 0) {
        s_dec.seq = 0; s_dec.stop = 0; s_dec.stop_r = 0; s_dec.stop_seq = 0; s_dec.fire_k = 0; s_dec.fire_bad = 0; s_dec.R = 0.0;
        s_bad = 0; s_panic = 0; s_zero = 0;
        for (int i = 0; i < 8; ++i) s_pf[i] = 0;
    }
    // DS: bytes this tile receives per half-sweep; thread 0 initialises and arms both mbarriers, and the whole cluster
    // (service warps included, once) synchronises before anybody sends
    unsigned ds_expect = 0;
    if (DS) {
        const int tx_ = tile % p.ntx, ty_ = tile / p.ntx;
        const int rows_ = min(BH, g.nz - ty_ * BH);
        ds_expect = 8u * (unsigned)((tx_ + 1 < p.ntx ? rows_ / 2 : 0) + (tx_ > 0 ? rows_ / 2 : 0) +
                                    (ty_ + 1 < p.nty ? BW / 2 : 0) + (ty_ > 0 ? BW / 2 : 0));
        if (tid == 0) {
            for (int c = 0; c < 2; ++c) {
                const unsigned bar = (unsigned)__cvta_generic_to_shared(&s_mbar[c]);
                asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(1u) : "memory");
            }
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            for (int c = 0; c < 2; ++c) Engine::ds_arm((unsigned)__cvta_generic_to_shared(&s_mbar[c]), ds_expect);
        }
    }
    __syncthreads();
    if (DS) asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");

    // =============================================================================================================
    // service warp
    // =============================================================================================================
    if (warp == NW) {
        unsigned int* slots_f = p.slots_f + (size_t)member * p.slot_stride;
        unsigned long long* slots_x = p.slots_x + (size_t)member * p.slot_stride;
        double* hist = p.hist + (size_t)member * p.hist_stride;
        bool stopped = false;
        const PollCtx pc_svc = {&s_zero, &s_panic, &ctl->panic, &ctl->panic_tile, tile};
        for (int seq = 1;; ++seq) {
            const int par = seq & 1;
            if (par) asm volatile("bar.sync 3, %0;" ::"n"(RS::NTHREADS) : "memory");
            else asm volatile("bar.sync 2, %0;" ::"n"(RS::NTHREADS) : "memory");
            const ResReport rep = s_rep[par];
            if (rep.quit) break;
            // ---- report: this CTA's maxima of the interval -> global slots, then arrive
            for (int idx = lane; idx < 2 * rep.n; idx += 32) {
                unsigned long long v = 0ull;
                for (int w = 0; w < NW; ++w) {
                    const unsigned long long t = smax[((size_t)par * 2 * kMaxTB + idx) * NW + w];
                    v = t > v ? t : v;
                }
                const size_t slot = 2 * (size_t)rep.k0 + idx;
                if (rep.exact) atomicMax(slots_x + slot, rep.bad ? 0x7ff8000000000000ull : v);
                else atomicMax(slots_f + slot, rep.bad ? 0x7ff80000u : (unsigned)v);
            }
            __syncwarp();
            unsigned int* arr = arrived + (size_t)rep.exact * p.arr_stride + rep.r;
            if (lane == 0) red_release_add_u32(arr, 1u);      // release: the warp's atomics above (ordered by __syncwarp)
            // ---- decide the interval (every CTA reads the same final slots -> the same answer)
            if (rep.exact || !stopped) {
                if (lane == 0) {
                    unsigned spins = 0;
                    while (ld_acquire_u32(arr) < (unsigned)ntiles && !poll_giveup(pc_svc, spins, 10 + rep.exact, rep.r))
                        __nanosleep(64);
                }
                __syncwarp();
                bool fire = false, bad = false;
                double R = 0.0;
                if (lane < rep.n) {
                    const size_t slot = 2 * (size_t)(rep.k0 + lane);
                    const size_t s0 = (size_t)member * g.slots0_stride + rep.k0 + lane;      // rule 1: equator-row maximum
                    if (rep.exact) {
                        const unsigned long long k0x = g.rule != 0 ? __ldcg(g.slots0_x + s0) : 0ull;
                        R = stop_value(g, __ldcg(slots_x + slot), __ldcg(slots_x + slot + 1), k0x, ctl->maxf);
                        bad = is_nonfinite(R);
                        fire = bad || (g.tol > 0.0 && R <= g.tol);
                    } else {
                        // upper words only: R_lo <= R_k (up to rounding, covered by the factor)
                        const unsigned long long kr = (unsigned long long)__ldcg(slots_f + slot) << 32;
                        const unsigned long long kp = ((unsigned long long)__ldcg(slots_f + slot + 1) << 32) | 0xffffffffull;
                        const unsigned long long k0f = g.rule != 0 ? (unsigned long long)__ldcg(g.slots0_f + s0) << 32 : 0ull;
                        R = stop_value(g, kr, kp, k0f, ctl->maxf);
                        bad = is_nonfinite(R);
                        fire = bad || (g.tol > 0.0 && R <= g.tol * 1.000000001);
                    }
                }
                const unsigned bal = __ballot_sync(0xffffffffu, fire);
                const int first = bal ? __ffs(bal) - 1 : -1;
                if (tile == 0 && lane < rep.n && (first < 0 || lane <= first || !rep.exact)) hist[rep.k0 + lane] = R;
                if (rep.exact) {
                    const int src = first < 0 ? rep.n - 1 : first;
                    const double Rsel = __shfl_sync(0xffffffffu, R, src);
                    const int badsel = __shfl_sync(0xffffffffu, (int)bad, src);
                    if (lane == 0) {
                        s_dec.fire_k = first < 0 ? 0 : rep.k0 + first + 1;
                        s_dec.fire_bad = badsel;
                        s_dec.R = Rsel;
                    }
                } else if (first >= 0) {
                    stopped = true;
                    if (lane == 0) {
                        s_dec.stop_r = rep.r;
                        s_dec.stop_seq = seq;
                        __threadfence_block();
                        s_dec.stop = 1;
                    }
                }
            }
            __syncwarp();
            if (lane == 0) {
                __threadfence_block();
                s_dec.seq = seq;
            }
        }
        return;
    }

    // =============================================================================================================
    // compute warps
    // =============================================================================================================
    Engine E;
    E.carve(reinterpret_cast<double*>(smem_raw));
    if (RING) {
        E.carve_ring(reinterpret_cast<double*>(smem_raw + RS::smem_bytes));
        E.bind_stash(s_stash);
    }
    E.bind_thread(tid);

    const int tx = tile % p.ntx, ty = tile / p.ntx;
    int x0, x1, y0, y1, bx, by;
    if (HALO) {
        x0 = bx = tx * BW; x1 = x0 + BW;
        y0 = by = ty * BH; y1 = min(g.nz, y0 + BH);
    } else {
        const int h = 2 * p.m;
        x0 = tx * p.ow; x1 = min(g.nr, x0 + p.ow);
        y0 = ty * p.oh; y1 = min(g.nz, y0 + p.oh);
        bx = box_origin(x0, h, 4, BW, g.nr);
        by = box_origin(y0, h, H, BH, g.nz);
    }
    const int gi0 = bx + 4 * E.a, gj0 = by + H * E.b;
    E.active = gj0 < g.nz;                                      // false only in the ragged last tile row (halo mode)
    const bool own = gi0 >= x0 && gi0 < x1 && gj0 >= y0 && gj0 < y1;
    const bool row0_warp = __any_sync(0xffffffffu, g.symmetry == 1 && gj0 == 0 && E.active);   // holds equator-row cells

    const double* rho = p.rho + (size_t)member * ncell;
    double* phi_io = p.phi + (size_t)member * ncell;
    double* ring = p.ring + (size_t)member * kResRing * ncell;
    // halo mode: inboxes of this tile and of its four neighbours
    const bool mirror_box = g.symmetry == 1 && by == 0;
    if constexpr (HALO) {
        typename Engine::HaloLinks links;
        uint4* mb = p.mail + (size_t)member * ntiles * Engine::kInboxPackets;
        auto inbox = [&](int t) { return mb + (size_t)t * Engine::kInboxPackets; };
        links.own = inbox(tile);
        links.w = (tx > 0) ? inbox(tile - 1) : nullptr;
        links.e = (tx + 1 < p.ntx) ? inbox(tile + 1) : nullptr;
        links.s = (ty > 0) ? inbox(tile - p.ntx) : nullptr;
        links.n = (ty + 1 < p.nty) ? inbox(tile + p.ntx) : nullptr;
        links.rows = min(BH, g.nz - by);
        if (DS) E.ds_bind(links, s_mbar, tile, p.ntx);
        if (!DS || RING) E.template halo_bind<RING>(links, tid);
        if (tid == 0) {                        // CTA-uniform: read from shared memory in the sweep loop, not kept in registers
            s_links = links;
            if (RING) {
                s_ring.cE_e = g.cE[bx + BW - 1]; s_ring.cW_e = g.cW[bx + BW - 1];
                s_ring.cE_w = g.cE[bx]; s_ring.cW_w = g.cW[bx];
                s_ring.cE = g.cE + bx; s_ring.cW = g.cW + bx;
                s_ring.mirror_box = mirror_box ? 1 : 0;
                s_ring.tile = tile; s_ring.ntx = p.ntx;
            }
        }
    }
    // block mode: the tiles whose owned cells this box overlaps (their flags gate the margin refill)
    unsigned int* flags = p.flags + (size_t)member * ntiles;
    const int nbx0 = bx / p.ow, nbx1 = (bx + BW - 1) / p.ow;
    const int nby0 = by / p.oh, nby1 = min(p.nty - 1, (by + BH - 1) / p.oh);
    const int nnb = (nbx1 - nbx0 + 1) * (nby1 - nby0 + 1);
    const double* bE = p.bE + (size_t)member * g.nz;
    const double* bN = p.bN + (size_t)member * g.nr;
    const double* bS = p.bS + (size_t)member * g.nr;
    unsigned int* gbar = p.gbar + member;
    const volatile int* stop = &s_dec.stop;
    const PollCtx pc_main = {&s_dec.stop, &s_panic, &ctl->panic, &ctl->panic_tile, tile};   // main phase: polls end at a stop
    const PollCtx pc_end = {&s_zero, &s_panic, &ctl->panic, &ctl->panic_tile, tile};        // endgame / replay

    // state after interval r (r = 0: the caller's initial guess, untouched until the very end)
    auto state_of = [&](int r) -> double* { return r == 0 ? phi_io : ring + (size_t)(r % kResRing) * ncell; };

    // (re)load the whole box from a full state array
    auto load_box = [&](const double* src) {
        if (E.active) {
            E.load_patch(src, g.nr, gi0, gj0);
        } else {
#pragma unroll
            for (int q = 0; q < H; ++q)
#pragma unroll
                for (int c = 0; c < 4; ++c) E.phi[q][c] = bN[gi0 + c];   // published as the north ghost row below
        }
        E.set_borders(g, bx, by, bE, bN, bS, tid, NT);
        Engine::sync();                                          // borders first: halo loads overwrite some of them
        if (HALO) E.load_halo_borders(src, g.nr, g.nz, bx, by);
        E.template publish_all<RING>();
        Engine::sync();
        if (RING) {                                              // the ring threads' private copies of their edge cells
            E.ring_init();
            Engine::sync();
        }
    };

    auto panicked = [&]() -> bool { return *(volatile int*)&s_panic != 0; };
    // The service warp (and the watchdog) write their words at any time, so two compute threads may read different
    // values; every branch that leads to a different sequence of barriers is taken on the OR over the compute warps.
    auto uniform_or = [&](bool v) -> bool {
        int out;
        asm volatile(
            "{\n\t.reg .pred p, q;\n\tsetp.ne.s32 q, %1, 0;\n\tbar.red.or.pred p, 1, %2, q;\n\tselp.s32 %0, 1, 0, p;\n\t}"
            : "=r"(out)
            : "r"((int)v), "n"(NT)
            : "memory");
        return out != 0;
    };
    // optional in-kernel profile (thread 0 of the CTA): 0 total, 1 half-sweep compute, 2 halo exchange, 3 barrier,
    // 4 end of interval, 5 margin refill, 6 wait for the decision, 7 half-sweeps
    const bool prof_on = p.prof != nullptr && tid == 0;
    auto tick = [&]() -> long long {          // asm volatile under the branch: never executed speculatively
        long long t = 0;
        if (prof_on) asm volatile("mov.u64 %0, %%clock64;" : "=l"(t));
        return t;
    };
    const long long t_begin = tick();
    unsigned gbar_gen = 0;
    auto grid_barrier = [&]() {
        ++gbar_gen;
        Engine::sync();
        if (tid == 0) {
            red_release_add_u32(gbar, 1u);
            unsigned spins = 0;
            while (ld_acquire_u32(gbar) < gbar_gen * (unsigned)ntiles && !poll_giveup(pc_end, spins, 20, (int)gbar_gen))
                __nanosleep(64);
        }
        Engine::sync();
    };

    // hand a report to the service warp: named barriers 2 / 3 alternate with the report's sequence parity
    auto report_arrive = [&](int par) {
        if (par) asm volatile("bar.arrive 3, %0;" ::"n"(RS::NTHREADS) : "memory");
        else asm volatile("bar.arrive 2, %0;" ::"n"(RS::NTHREADS) : "memory");
    };
    int seq = 0;                                                 // reports handed to the service warp so far
    auto wait_decided = [&](int want) {
        unsigned spins = 0;
        while (s_dec.seq < want && !poll_giveup(pc_end, spins, 30, want)) __nanosleep(32);
    };

    // n sweeps starting after k0 applied sweeps; maxima of sweep s of the interval go to smax[par][2s..2s+1][warp]
    auto run_sweeps = [&](auto trackTag, int k0, int n, unsigned tagbase, int par, const PollCtx& pc) {
        constexpr int TRACK = decltype(trackTag)::value;
        for (int s = 0; s < n; ++s) {
            E.reset_maxima();
            const long long t0 = tick();
            const unsigned tag0 = tagbase + 2u * (unsigned)(k0 + s) + 1u;
            uint4 pf = make_uint4(0u, 0u, 0u, 0u);
            if (RING && DS) {
                E.template ring_duty<0, true>(s_links, s_ring, tag0);
                if (prof_on) s_pf[5] += tick() - t0;                         // ring duty alone (slot 5: block mode's refill)
                E.template half_sweep<0, TRACK, false, true>();
            } else if (RING) {
                E.template ring_duty<0>(s_links, s_ring, tag0);
                if (prof_on) s_pf[5] += tick() - t0;
                pf = E.template half_sweep_ring<0, TRACK>(s_links);
            } else {
                E.template half_sweep<0, TRACK, false>();
                if (HALO && DS && !RING) E.template ds_send<0>();
                else if (HALO && !DS) E.template halo_send<0>(tag0);
            }
            const long long t1 = tick();
            if (HALO && DS) {
                E.template ds_recv<0>(ds_expect, tid == 0, pc_end);      // never abandoned: see box_engine.cuh
                if (RING) E.template ds_ring_copy<0>();
            }
            else if (HALO) {
                E.template halo_recv<0>(s_links, tag0, pc, pf);
            }
            const long long t2 = tick();
            Engine::sync();
            const long long t3 = tick();
            if (RING && DS) {
                E.template ring_duty<1, true>(s_links, s_ring, tag0 + 1u);
                if (prof_on) s_pf[5] += tick() - t3;
                E.template half_sweep<1, TRACK, false, true>();
            } else if (RING) {
                E.template ring_duty<1>(s_links, s_ring, tag0 + 1u);
                if (prof_on) s_pf[5] += tick() - t3;
                pf = E.template half_sweep_ring<1, TRACK>(s_links);
            } else {
                E.template half_sweep<1, TRACK, false>();
                if (HALO && DS && !RING) E.template ds_send<1>();
                else if (HALO && !DS) E.template halo_send<1>(tag0 + 1u);
            }
            const long long t4 = tick();
            // the sweep's maxima are complete: reduce them across the warp BEFORE the last wait / barrier of the sweep,
            // so that the REDUX latency (measured ~135 clocks per half-sweep when done after the barrier) hides in it
            // rule 1 (R16): the maximum over the reflecting-equator row goes straight to its own per-sweep slot from the
            // few warps that hold that row (ordered before the service warp's release by the barriers in between)
            if (g.rule != 0 && row0_warp && TRACK != kTrackNone) {
                if (TRACK == kTrackFast) {
                    const unsigned w0 = __reduce_max_sync(0xffffffffu, own ? __float_as_uint(E.mres0_f) : 0u);
                    if (lane == 0) atomicMax(g.slots0_f + (size_t)member * g.slots0_stride + k0 + s, w0);
                } else {
                    const unsigned long long w0 = warp_max_key(own ? E.mres0_k : 0ull);
                    if (lane == 0) atomicMax(g.slots0_x + (size_t)member * g.slots0_stride + k0 + s, w0);
                }
            }
            if (TRACK == kTrackFast) {
                const unsigned wr = __reduce_max_sync(0xffffffffu, own ? __float_as_uint(E.mres_f) : 0u);
                const unsigned wp = __reduce_max_sync(0xffffffffu, own ? __float_as_uint(E.mphi_f) : 0u);
                if (lane == 0) {
                    smax[((size_t)par * 2 * kMaxTB + 2 * s) * NW + warp] = wr;
                    smax[((size_t)par * 2 * kMaxTB + 2 * s + 1) * NW + warp] = wp;
                }
            } else if (TRACK == kTrackExact) {
                const unsigned long long wr = warp_max_key(own ? E.mres_k : 0ull);
                const unsigned long long wp = warp_max_key(own ? E.mphi_k : 0ull);
                if (lane == 0) {
                    smax[((size_t)par * 2 * kMaxTB + 2 * s) * NW + warp] = wr;
                    smax[((size_t)par * 2 * kMaxTB + 2 * s + 1) * NW + warp] = wp;
                }
            }
            if (HALO && DS) {
                E.template ds_recv<1>(ds_expect, tid == 0, pc_end);
                if (RING) E.template ds_ring_copy<1>();
            }
            else if (HALO) {
                E.template halo_recv<1>(s_links, tag0 + 1u, pc, pf);
            }
            const long long t5 = tick();
            Engine::sync();
            const long long t6 = tick();
            if (prof_on) {
                s_pf[1] += (t1 - t0) + (t4 - t3); s_pf[2] += (t2 - t1) + (t5 - t4); s_pf[3] += (t3 - t2) + (t6 - t5);
                s_pf[7] += 2;
            }
        }
    };

    // end of interval r (n sweeps after k0): checkpoint, block-mode exchange, report.  Returns the report's sequence
    // number.  The margins are NOT yet valid in block mode when this returns (see finish_exchange).
    auto end_interval = [&](int r, int k0, int n, int exact, unsigned tagbase) -> int {
        if (own) E.store_patch(state_of(r), g.nr, gi0, gj0);
        // FAST maxima drop NaN (FMNMX); any non-finite owned value persists (NaN/Inf never relax away), so one
        // check per interval is enough to poison its maxima and send the solve to the exact endgame
        if (!exact && own && E.any_nonfinite()) s_bad = 1;
        ++seq;
        const int par = seq & 1;
        Engine::sync();                                          // smax + s_bad complete
        if (tid == 0) {
            ResReport& rp = s_rep[par];
            rp.r = r; rp.k0 = k0; rp.n = n; rp.exact = exact; rp.quit = 0;
            rp.bad = exact ? 0 : s_bad;      // exact keys carry NaN/Inf themselves (abs_key sorts them highest)
        }
        report_arrive(par);
        // block mode: publish "state r of this tile is in the ring" (the barrier above ordered every thread's stores
        // before this thread's fence)
        if (!HALO && ntiles > 1) {
            if (p.ll) {
                if (own) E.ll_store_patch(p.mail + ((size_t)member * 2 + (r & 1)) * ncell, tagbase + (unsigned)r, g.nr, gi0, gj0);
            } else if (tid == 0) {
                st_release_u32(flags + tile, tagbase + (unsigned)r);
            }
        }
        return seq;
    };
    // block mode: refill the margins from the neighbours' tiles of interval r and republish the patch edges
    auto finish_exchange = [&](int r, unsigned tagbase, const PollCtx& pc) {
        if (HALO || ntiles == 1) return;
        if (p.ll) {
            if (!own) E.ll_wait_patch(p.mail + ((size_t)member * 2 + (r & 1)) * ncell, tagbase + (unsigned)r, g.nr, gi0, gj0, pc);
            E.publish_all();
            Engine::sync();
            return;
        }
        if (warp == NW - 1) {
            const unsigned want = tagbase + (unsigned)r;
            for (int i = lane; i < nnb; i += 32) {
                const int t = (nby0 + i / (nbx1 - nbx0 + 1)) * p.ntx + nbx0 + i % (nbx1 - nbx0 + 1);
                if (t == tile) continue;
                unsigned spins = 0;
                // relaxed polls (an acquire would invalidate L1 on every iteration)
                while (ld_relaxed_u32(flags + t) < want && !poll_giveup(pc, spins, 5, (int)want)) {}
            }
            // ONE acquire fence after the relaxed spin (not one per poll): relaxed load that observed the neighbour's
            // st.release + fence.acq_rel = acquire pattern of the PTX memory model, so the ring stores of every tile
            // polled above happen-before the margin loads of the whole CTA (ordered after this warp by the barrier).
            asm volatile("fence.acq_rel.gpu;" ::: "memory");
        }
        const long long tp0 = tick();
        Engine::sync();
        if (prof_on) s_pf[2] += tick() - tp0;                    // block mode: wait for the neighbours' flags
        if (!own) E.load_patch(state_of(r), g.nr, gi0, gj0);
        E.publish_all();
        Engine::sync();
    };

    // one-time set-up: f, coefficients, initial phi
    if (E.active) E.load_f(rho, g.nr, gi0, gj0);
    E.load_coeffs(g, gi0, E.active ? gj0 : 0);
    load_box(phi_io);
    if (DS) grid_barrier();      // DS: neighbours write straight into my border slots -- not before they are loaded

    // ---- main phase: FAST maxima, decisions one interval late -------------------------------------------------
    int r_c = 1;                 // interval the endgame starts with
    bool reload = false;         // endgame must reload the state before r_c (CTAs stopped at different intervals)
    if (!p.force_exact) {
        int r = 1;
        for (; r < R_last; ++r) {
            const int k0 = (r - 1) * Q;
            run_sweeps(std::integral_constant<int, kTrackFast>{}, k0, Q, 0u, (seq + 1) & 1, pc_main);
            const long long ta = tick();
            const int sq = end_interval(r, k0, Q, 0, 0u);
            const long long tb = tick();
            finish_exchange(r, 0u, pc_main);
            const long long tc = tick();
            wait_decided(sq - 1);
            if (prof_on) { s_pf[4] += tb - ta; s_pf[5] += tc - tb; s_pf[6] += tick() - tc; }
            // a stop decided by report sq (being processed right now) must not be seen by some threads only
            const bool stopped_now = *stop && s_dec.stop_seq <= sq - 1;
            if (uniform_or(stopped_now || panicked())) break;
        }
        if (r == R_last) {       // ran to the last interval: wait for every earlier decision
            wait_decided(seq);
        }
        if (uniform_or(*stop != 0)) {
            r_c = s_dec.stop_r;
            reload = true;
        } else {
            r_c = R_last;
        }
    }

    // ---- endgame: EXACT maxima, every interval decided before the next ------------------------------------------
    int sweeps = 0, status = 0;
    double Rfinal = 0.0;
    {
        unsigned tagbase = 0u;
        if (reload) {
            grid_barrier();
            load_box(state_of(r_c - 1));
            if (DS) grid_barrier();
            tagbase = kTagEndgame;
        }
        int r = r_c;
        for (;; ++r) {
            const int k0 = (r - 1) * Q;
            const int n = min(Q, p.max_sweeps - k0);
            if (n <= 0) {        // max_sweeps == 0
                sweeps = 0; status = g.tol > 0.0 ? 1 : 0; Rfinal = 0.0;
                break;
            }
            run_sweeps(std::integral_constant<int, kTrackExact>{}, k0, n, tagbase, (seq + 1) & 1, pc_end);
            const int sq = end_interval(r, k0, n, 1, tagbase);
            wait_decided(sq);
            if (uniform_or(panicked())) { sweeps = k0 + n; status = -2; break; }
            const int fk = s_dec.fire_k;
            if (fk) {
                sweeps = fk; status = s_dec.fire_bad ? -3 : 0; Rfinal = s_dec.R;
                if (fk != k0 + n) {                              // crossing inside the interval: replay from its start
                    grid_barrier();
                    load_box(state_of(r - 1));
                    if (DS) grid_barrier();
                    run_sweeps(std::integral_constant<int, kTrackNone>{}, k0, fk - k0, kTagReplay, 0, pc_end);
                }
                break;
            }
            if (k0 + n >= p.max_sweeps) {
                sweeps = p.max_sweeps; status = g.tol > 0.0 ? 1 : 0; Rfinal = s_dec.R;
                break;
            }
            finish_exchange(r, tagbase, pc_end);
        }
    }

    // ---- finish ---------------------------------------------------------------------------------------------------
    // Nobody may still be reading phi_io as "state 0": a reload from it is followed by a grid barrier-free run, so
    // make every CTA pass one more barrier before the result overwrites it.
    grid_barrier();
    if (own) E.store_patch(phi_io, g.nr, gi0, gj0);
    // ---- fused gravity epilogue (NEXT-1; eqs. 2-4; R15): g = -grad phi of the result while
    // phi is still in registers.  Neighbours inside the patch are registers; the ones outside come from the result
    // just stored (L2), after one more grid barrier -- the same in every tile mode, and exact: centred differences with
    // the pinned arithmetic (lo - hi) * (0.5 / d), reflecting axis / equator, ghosts elsewhere.
    if (p.gr != nullptr) {
        grid_barrier();
        if (own && E.active) {
            double* grm = p.gr + (size_t)member * ncell;
            double* gzm = p.gz + (size_t)member * ncell;
            const double hr = 0.5 / g.dr, hz = 0.5 / g.dz;
#pragma unroll
            for (int q = 0; q < H; ++q) {
                const int row = gj0 + q;
                const double* prow = phi_io + (size_t)row * g.nr;
                const double west = gi0 > 0 ? __ldcg(prow + gi0 - 1) : E.phi[q][0];                 // reflecting axis
                const double east = gi0 + 4 < g.nr ? __ldcg(prow + gi0 + 4) : bE[row];
                double r4[4], z4[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const double pW = c == 0 ? west : E.phi[q][c == 0 ? 0 : c - 1];
                    const double pE = c == 3 ? east : E.phi[q][c == 3 ? 3 : c + 1];
                    const double pN = q < H - 1 ? E.phi[q < H - 1 ? q + 1 : q][c]
                                                : (row + 1 < g.nz ? __ldcg(prow + g.nr + gi0 + c) : bN[gi0 + c]);
                    const double pS = q > 0 ? E.phi[q > 0 ? q - 1 : 0][c]
                                            : (row > 0 ? __ldcg(prow - g.nr + gi0 + c)
                                                       : (g.symmetry == 1 ? E.phi[q][c] : bS[gi0 + c]));
                    r4[c] = __dmul_rn(__dsub_rn(pW, pE), hr);
                    z4[c] = __dmul_rn(__dsub_rn(pS, pN), hz);
                }
                double2* o = reinterpret_cast<double2*>(grm + (size_t)row * g.nr + gi0);
                double2* z = reinterpret_cast<double2*>(gzm + (size_t)row * g.nr + gi0);
                __stcs(o, make_double2(r4[0], r4[1])); __stcs(o + 1, make_double2(r4[2], r4[3]));
                __stcs(z, make_double2(z4[0], z4[1])); __stcs(z + 1, make_double2(z4[2], z4[3]));
            }
        }
    }
    ++seq;
    Engine::sync();
    if (tid == 0) s_rep[seq & 1].quit = 1;
    report_arrive(seq & 1);
    if (prof_on) {
        s_pf[0] = clock64() - t_begin;
        long long* dst = p.prof + ((size_t)member * ntiles + tile) * 8;
        for (int i = 0; i < 8; ++i) dst[i] = s_pf[i];
    }
    if (tile == 0 && tid == 0) {
        ctl->sweeps = sweeps;
        ctl->status = status;
        ctl->residual = Rfinal;
        __threadfence();
        ctl->done = 1;
    }
}

}  // namespace snp
