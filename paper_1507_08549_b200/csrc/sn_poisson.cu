// sn_poisson.cu -- C-ABI host side of the B200-native Poisson solve (include/sn_poisson.h).
// Argument checks, workspace, launch sequencing; every step of the path runs in the kernels of
// moments.cuh / sweep_stream.cuh / sweep_resident.cuh.  No CPU fallback.
#include "../../include/sn_poisson.h"

#include <type_traits>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <algorithm>
#include <mutex>
#include <string>
#include <vector>

#include "common.cuh"
#include "moments.cuh"
#include "gravity.cuh"
#include "probe.cuh"
#include "sweep_stream.cuh"
#include "sweep_blocked.cuh"
#include "sweep_resident.cuh"
#include "shapes.cuh"
#include "mg.cuh"

using namespace snp;

namespace {

thread_local std::string g_err;

void set_err(const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
}

#define CU_TRY(expr)                                                                       \
    do {                                                                                   \
        cudaError_t e__ = (expr);                                                          \
        if (e__ != cudaSuccess) {                                                          \
            set_err("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
            return -2;                                                                     \
        }                                                                                  \
    } while (0)

template <typename T>
int dev_alloc(T** p, size_t n) {
    CU_TRY(cudaMalloc((void**)p, n * sizeof(T)));
    return 0;
}

}  // namespace

namespace {
struct BlkPlan {
    int shape = -1, m = 0, ntx = 0, nty = 0, ow = 0, oh = 0, ntiles = 0, occ = 0;
    double cost = 0;
};
struct ResPlan {
    int shape = -1, halo = 0, ds = 0, ring = 0, ll = 0, m = 0, Q = 0, ntx = 0, nty = 0, ow = 0, oh = 0, ntiles = 0;
    double cost = 0;
};
// Limits of the per-sweep bookkeeping (ensure_ws: d_slots 16 + d_slots_f 8 + d_slots0 8 + d_slots0_f 4 + d_hist 8 = 44 B
// per sweep and member).
constexpr int kMaxSweepsLimit = 1 << 22;                 // per solve
constexpr long long kMaxSweepSlots = 1ll << 26;          // max_sweeps x nbatch (2.75 GiB of bookkeeping)
}  // namespace

struct sn_poisson {
    int nr = 0, nz = 0, symmetry = 0, lmax = 0;
    double dr = 0, dz = 0;
    double omega = 0;
    bool omega_user = false;
    int device = 0, num_sms = 0;
    double L0 = 0;
    int NL = 0;                 // moment template width (lcap + 1)
    int mom_blocks = 0;

    // options
    int opt_path = 0, opt_chunk = 32, opt_tblock = 0, opt_shape = -1, opt_exact = 0, opt_halo = -1, opt_prof = 0, opt_ll = -1, opt_group = -1, opt_ds = -1, opt_ring = -1, opt_rule = 0;

    // device workspace (sized for `cap_batch` members)
    int cap_batch = 0, cap_sweeps = 0;
    double *d_cE = nullptr, *d_cW = nullptr;
    double *d_bE = nullptr, *d_bN = nullptr, *d_bS = nullptr, *d_M = nullptr, *d_partial = nullptr;
    unsigned long long* d_slots = nullptr;
    unsigned int* d_slots_f = nullptr;                       // blocked path: FAST maxima (upper words)
    unsigned long long* d_slots0 = nullptr;                  // rule 1: per-sweep maxima of |res| over the equator row
    unsigned int* d_slots0_f = nullptr;
    double* d_work = nullptr;                                // blocked path: second phi buffer, work_cap doubles
    size_t work_cap = 0;
    double* d_hist = nullptr;
    Ctl* d_ctl = nullptr;
    Ctl* h_ctl = nullptr;       // pinned, 2 * cap_batch (double-buffered polls)
    double *d_rho_stage = nullptr, *d_phi_stage = nullptr;   // solve_host staging
    double* d_ring = nullptr;                                // resident path: checkpoint ring, nb x kResRing x nr*nz
    void* d_mail = nullptr;                                  // resident path, halo mode: per-tile inboxes of 16-byte tagged packets
    unsigned int* d_sync = nullptr;                          // resident path: arrived counters | grid barriers | tile flags
    size_t ring_cap = 0, mail_cap = 0, sync_cap = 0;
    long long* d_prof = nullptr;                             // resident path: optional in-kernel profile, ctas x 8
    size_t prof_cap = 0, prof_ctas = 0;
    double prof_mean[8] = {0}, prof_max[8] = {0};
    bool user_boundary = false;
    int last_nbatch = 0;        // members whose ghost arrays are valid (last solve / set_boundary)
    cudaEvent_t ev_poll[2] = {nullptr, nullptr};
    cudaEvent_t ev_t[3] = {nullptr, nullptr, nullptr};
    // host-buffer entry points: staging (grown on demand, kept), a copy stream and its events
    size_t stage_cap = 0;       // doubles per staging array
    double* d_snap[2] = {nullptr, nullptr};                  // sequence: phi snapshots for the overlapped D2H
    size_t snap_cap = 0;
    cudaStream_t st_copy = nullptr;
    cudaEvent_t ev_io[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    // planner cache: the plan depends only on (nbatch, pointer alignment, options), not on the data
    struct {
        bool valid = false;
        int nbatch = 0, aligned = 0;
        ResPlan pl;
        BlkPlan bp;
        int group = 0;
    } plan_cache;

    // multigrid variant (NEXT-4): per-level coefficient tables, errors and right-hand sides (levels >= 1), the maxima slots
    struct MgWs {
        int nlev = 0;
        std::vector<int> nr, nz;
        std::vector<double*> cE, cW, phi, f;
        unsigned long long* slots = nullptr;
        MgPtrs* d_ptrs = nullptr;         // the caller's rho / phi of the current solve, read by the level-0 kernels
        bool tail_attr = false;
        int cap_batch = 0;                // members the per-level arrays hold
        int nb = 1;                       // members of the current solve
        // one V-cycle captured as a CUDA graph (the cycle is ~15-27 short launches): valid for one (tol, max_cycles,
        // options) key -- the caller's rho / phi reach the kernels through d_ptrs --, re-captured when the key changes
        cudaGraphExec_t exec = nullptr;
        cudaStream_t st = nullptr;        // runs the cycles when the caller hands in the (uncapturable) legacy stream
        double nodes = 0;                 // kernel nodes per captured cycle
        struct Key { double tol = 0; int max_cycles = -1, nu1 = 0, nu2 = 0, nc = 0, nb = 0, cap_sweeps = 0; } key;
        double* h_hist = nullptr;     // pinned: the last two ratios of every member, for the host's chunk prediction
        int hist_cap = 0;
    } mg;
    int opt_mg_nu1 = 1, opt_mg_nu2 = 1, opt_mg_nc = 12, opt_mg_graph = 1;

    // stats of the last solve
    double st_aux_launches = 0;   // launches that are not relaxation sweeps (moments, boundary, init, decide)
    double st_launches = 0, st_sweep_ms = 0, st_setup_ms = 0, st_path = 0;
    double st_ctas = 0, st_tile_w = 0, st_tile_h = 0, st_tblock = 0, st_shape = -1, st_halo = 0, st_group = 0, st_ds = 0, st_redund = 1, st_ring = 0;
    int last_sweeps0 = 0;
};

namespace {

// DESIGN.md R8: default relaxation factor, closed form with only + - * / sqrt (same expression order as stated there).
double default_omega(int nr, int nz, double dr, double dz, int symmetry) {
    const double j01 = 2.404825557695773;
    const double Lr = (nr + 0.5) * dr;
    const double kz = symmetry == 1 ? kPi / (2.0 * ((nz + 0.5) * dz)) : kPi / ((nz + 1.0) * dz);
    const double a = j01 / Lr;
    const double lambda = a * a + kz * kz;
    const double D = 2.0 / (dr * dr) + 2.0 / (dz * dz);
    const double mu = 1.0 - lambda / D;
    return 2.0 / (1.0 + std::sqrt(1.0 - mu * mu));
}

Geom make_geom(const sn_poisson* h, double tol) {
    Geom g;
    g.nr = h->nr; g.nz = h->nz; g.symmetry = h->symmetry; g.lmax = h->lmax;
    g.dr = h->dr; g.dz = h->dz;
    const double ir2 = 1.0 / (h->dr * h->dr);
    g.iz2 = 1.0 / (h->dz * h->dz);
    g.D = 2.0 * ir2 + 2.0 * g.iz2;
    g.D0 = g.D - g.iz2;
    g.wD = h->omega / g.D;
    g.wD0 = h->omega / g.D0;
    g.tol = tol;
    g.cE = h->d_cE;
    g.cW = h->d_cW;
    g.rule = h->opt_rule;
    g.slots0_stride = h->cap_sweeps;
    g.slots0_f = h->d_slots0_f;
    g.slots0_x = h->d_slots0;
    return g;
}

void free_batch_ws(sn_poisson* h) {
    if (h->mg.exec) { cudaGraphExecDestroy(h->mg.exec); h->mg.exec = nullptr; }      // the captured cycle holds these pointers
    cudaFree(h->d_bE); cudaFree(h->d_bN); cudaFree(h->d_bS); cudaFree(h->d_M); cudaFree(h->d_partial);
    cudaFree(h->d_slots); cudaFree(h->d_slots_f); cudaFree(h->d_hist); cudaFree(h->d_ctl);
    cudaFree(h->d_slots0); cudaFree(h->d_slots0_f);
    h->d_slots0 = nullptr; h->d_slots0_f = nullptr;
    if (h->h_ctl) cudaFreeHost(h->h_ctl);
    h->d_bE = h->d_bN = h->d_bS = h->d_M = h->d_partial = h->d_hist = nullptr;
    h->d_slots = nullptr; h->d_slots_f = nullptr; h->d_ctl = nullptr; h->h_ctl = nullptr;
    h->cap_batch = 0; h->cap_sweeps = 0;
    h->last_nbatch = 0;
}

// Grow the per-member workspace.  Keeps injected boundary arrays of member 0 across a regrow.
int ensure_ws(sn_poisson* h, int nbatch, int max_sweeps) {
    const int need_sw = max_sweeps < 1 ? 1 : max_sweeps;
    if (nbatch <= h->cap_batch && need_sw <= h->cap_sweeps) return 0;
    std::vector<double> kE, kN, kS;
    if (h->user_boundary && h->d_bE) {
        kE.resize(h->nz); kN.resize(h->nr); kS.resize(h->nr);
        CU_TRY(cudaMemcpy(kE.data(), h->d_bE, sizeof(double) * h->nz, cudaMemcpyDeviceToHost));
        CU_TRY(cudaMemcpy(kN.data(), h->d_bN, sizeof(double) * h->nr, cudaMemcpyDeviceToHost));
        CU_TRY(cudaMemcpy(kS.data(), h->d_bS, sizeof(double) * h->nr, cudaMemcpyDeviceToHost));
    }
    const int nb = nbatch > h->cap_batch ? nbatch : h->cap_batch;
    const int ns = need_sw > h->cap_sweeps ? need_sw : h->cap_sweeps;
    free_batch_ws(h);
    if (dev_alloc(&h->d_bE, (size_t)nb * h->nz) || dev_alloc(&h->d_bN, (size_t)nb * h->nr) ||
        dev_alloc(&h->d_bS, (size_t)nb * h->nr) || dev_alloc(&h->d_M, (size_t)nb * (kMaxL + 1)) ||
        dev_alloc(&h->d_partial, (size_t)nb * h->mom_blocks * h->NL) || dev_alloc(&h->d_slots, (size_t)nb * 2 * ns) || dev_alloc(&h->d_slots_f, (size_t)nb * 2 * ns) ||
        dev_alloc(&h->d_slots0, (size_t)nb * ns) || dev_alloc(&h->d_slots0_f, (size_t)nb * ns) ||
        dev_alloc(&h->d_hist, (size_t)nb * ns) || dev_alloc(&h->d_ctl, (size_t)nb))
        return -2;
    CU_TRY(cudaMallocHost((void**)&h->h_ctl, sizeof(Ctl) * 2 * nb));
    CU_TRY(cudaMemset(h->d_bS, 0, sizeof(double) * (size_t)nb * h->nr));
    CU_TRY(cudaMemset(h->d_M, 0, sizeof(double) * (size_t)nb * (kMaxL + 1)));
    h->cap_batch = nb;
    h->cap_sweeps = ns;
    if (!kE.empty()) {
        for (int b = 0; b < nb; ++b) {
            CU_TRY(cudaMemcpy(h->d_bE + (size_t)b * h->nz, kE.data(), sizeof(double) * h->nz, cudaMemcpyHostToDevice));
            CU_TRY(cudaMemcpy(h->d_bN + (size_t)b * h->nr, kN.data(), sizeof(double) * h->nr, cudaMemcpyHostToDevice));
            CU_TRY(cudaMemcpy(h->d_bS + (size_t)b * h->nr, kS.data(), sizeof(double) * h->nr, cudaMemcpyHostToDevice));
        }
    }
    return 0;
}

// blocks per member of the boundary fill: one ghost point per thread, at most 32 slices
inline int boundary_slices(const sn_poisson* h) {
    const int npts = h->nz + h->nr * (h->symmetry == 0 ? 2 : 1);
    return std::max(1, std::min(32, (npts + 255) / 256));
}

int launch_moments(sn_poisson* h, const Geom& g, int nbatch, const double* rho, cudaStream_t st) {
    dim3 grid(h->mom_blocks, nbatch);
    switch (h->NL) {
        case 9: k_moments<9><<<grid, kMomThreads, 0, st>>>(rho, g, h->L0, h->d_partial, h->d_ctl); break;
        case 17: k_moments<17><<<grid, kMomThreads, 0, st>>>(rho, g, h->L0, h->d_partial, h->d_ctl); break;
        case 33: k_moments<33><<<grid, kMomThreads, 0, st>>>(rho, g, h->L0, h->d_partial, h->d_ctl); break;
        default: k_moments<65><<<grid, kMomThreads, 0, st>>>(rho, g, h->L0, h->d_partial, h->d_ctl); break;
    }
    CU_TRY(cudaGetLastError());
    return 0;
}

// Streaming path: two launches per sweep, decision folded into the next sweep's launches, host polls per chunk.
int run_stream(sn_poisson* h, const Geom& g, int nbatch, const double* rho, double* phi, int max_sweeps,
               cudaStream_t st) {
    dim3 grid((h->nr + kStreamTileW - 1) / kStreamTileW, (h->nz + kStreamTileH - 1) / kStreamTileH, nbatch);
    const int slot_stride = 2 * h->cap_sweeps, hist_stride = h->cap_sweeps;
    const int chunk = h->opt_chunk < 1 ? 1 : h->opt_chunk;
    int k = 1, poll = 0;
    bool have_poll[2] = {false, false};
    bool all_done = false;
    while (k <= max_sweeps && !all_done) {
        const int kend = (max_sweeps - k + 1 < chunk) ? max_sweeps : k + chunk - 1;
        for (; k <= kend; ++k) {
            for (int colour = 0; colour < 2; ++colour) {
                k_halfsweep<<<grid, kStreamWarps * 32, 0, st>>>(g, colour, k, slot_stride, hist_stride, rho, phi,
                                                                h->d_bE, h->d_bN, h->d_bS, h->d_slots, h->d_ctl,
                                                                h->d_hist);
                h->st_launches += 1;
            }
        }
        CU_TRY(cudaGetLastError());
        if (g.tol > 0.0 && k <= max_sweeps) {
            // poll the device-side decision one chunk behind, so the queue never drains
            CU_TRY(cudaMemcpyAsync(h->h_ctl + (size_t)poll * h->cap_batch, h->d_ctl, sizeof(Ctl) * nbatch,
                                   cudaMemcpyDeviceToHost, st));
            CU_TRY(cudaEventRecord(h->ev_poll[poll], st));
            have_poll[poll] = true;
            const int prev = poll ^ 1;
            if (have_poll[prev]) {
                CU_TRY(cudaEventSynchronize(h->ev_poll[prev]));
                all_done = true;
                for (int b = 0; b < nbatch; ++b) all_done = all_done && h->h_ctl[(size_t)prev * h->cap_batch + b].done;
            }
            poll ^= 1;
        }
    }
    k_decide_last<<<nbatch, 32, 0, st>>>(g, k - 1, slot_stride, hist_stride, h->d_slots, h->d_ctl, h->d_hist);
    h->st_launches += 1;
    h->st_aux_launches += 1;
    CU_TRY(cudaGetLastError());
    return 0;
}


// ---- blocked path: shapes, planner, launcher -------------------------------------------------------------------
const std::vector<BlkShapeInfo>& blk_shapes() {
    static const std::vector<BlkShapeInfo> v = [] {
        std::vector<BlkShapeInfo> t;
        for (int i = 0; i < kNumBlkShapes; ++i) t.push_back(blk_shape(i));      // shape_tu.cu
        return t;
    }();
    return v;
}


// Pick (shape, m) minimising modelled clocks per sweep; honours the "shape"/"tblock" overrides.
BlkPlan plan_blocked(sn_poisson* h, int nbatch, const double* rho, const double* phi) {
    BlkPlan best;
    if (((uintptr_t)rho | (uintptr_t)phi) & 15) return best;
    const auto& sh = blk_shapes();
    for (int si = 0; si < (int)sh.size(); ++si) {
        if (h->opt_shape >= 0 && si != h->opt_shape) continue;
        const BlkShapeInfo& S = sh[si];
        int occ = 0;
        if (cudaFuncSetAttribute(S.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S.smem) != cudaSuccess ||
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, S.fn, S.NT(), S.smem) != cudaSuccess || occ < 1) {
            cudaGetLastError();
            continue;
        }
        if (occ > S.minb) occ = S.minb;
        for (int m = 1; m <= kMaxTB; ++m) {
            if (h->opt_tblock > 0 && m != h->opt_tblock) continue;
            BlkPlan p;
            if (!plan_axis(h->nr, S.BW(), 2 * m, 4, &p.ntx, &p.ow)) continue;
            if (!plan_axis(h->nz, S.BH(), 2 * m, S.H, &p.nty, &p.oh)) continue;
            bool ok = true;                      // the property the kernel relies on, checked for every tile
            for (int t = 0; t < p.ntx && ok; ++t) ok = box_covers(t, p.ow, 2 * m, 4, S.BW(), h->nr);
            for (int t = 0; t < p.nty && ok; ++t) ok = box_covers(t, p.oh, 2 * m, S.H, S.BH(), h->nz);
            if (!ok) continue;
            p.ntiles = p.ntx * p.nty;
            p.shape = si;
            p.m = m;
            p.occ = occ;
            // cost model (SM clocks per sweep): waves of CTAs; each CTA loads its box (16 B / cell at a share of the
            // L2 / HBM bandwidth), runs 2m half-sweeps and stores its tile; plus the launch gap.
            const double ctas = (double)p.ntiles * nbatch;
            const double slots = (double)h->num_sms * occ;
            const double waves = std::ceil(ctas / slots);
            const double bytes = 16.0 * S.BW() * S.BH() + 8.0 * p.ow * p.oh;
            const bool in_l2 = 16.0 * h->nr * h->nz * nbatch < 100e6;
            const double bw_per_sm = (in_l2 ? 40.0 : 18.0) / occ;          // bytes per clock per CTA
            const double t_cta = bytes / bw_per_sm * (occ > 1 ? 0.5 : 1.0) + 2.0 * m * S.hs_clk + 1500.0;
            p.cost = (waves * t_cta + 4000.0) / m;
            if (best.shape < 0 || p.cost < best.cost) best = p;
        }
    }
    return best;
}

int run_blocked(sn_poisson* h, const Geom& g, const BlkPlan& pl, int nbatch, const double* rho, double* phi,
                int max_sweeps, cudaStream_t st) {
    const BlkShapeInfo& S = blk_shapes()[pl.shape];
    const size_t ncell = (size_t)h->nr * h->nz;
    if (h->work_cap < ncell * nbatch) {
        cudaFree(h->d_work);
        h->d_work = nullptr;
        h->work_cap = 0;
        CU_TRY(cudaMalloc((void**)&h->d_work, sizeof(double) * ncell * nbatch));
        h->work_cap = ncell * nbatch;
    }
    CU_TRY(cudaMemset2DAsync(h->d_slots_f, sizeof(unsigned int) * 2 * (size_t)h->cap_sweeps, 0,
                             sizeof(unsigned int) * 2 * (size_t)std::max(1, max_sweeps), nbatch, st));
    BlkParams P;
    P.g = g;
    P.ntx = pl.ntx; P.nty = pl.nty; P.ow = pl.ow; P.oh = pl.oh; P.m = pl.m; P.max_sweeps = max_sweeps;
    P.force_exact = h->opt_exact;
    P.nbatch = nbatch;
    P.rho = rho; P.buf[0] = phi; P.buf[1] = h->d_work;
    P.bE = h->d_bE; P.bN = h->d_bN; P.bS = h->d_bS;
    P.slots_f = h->d_slots_f; P.slots_x = h->d_slots;
    P.slot_stride = 2 * h->cap_sweeps; P.hist_stride = h->cap_sweeps;
    P.ctl = h->d_ctl; P.hist = h->d_hist;
    k_blocked_init<<<nbatch, 32, 0, st>>>(h->d_ctl, pl.m, max_sweeps, h->opt_exact);
    h->st_launches += 1;
    h->st_aux_launches += 1;
    void* args[] = {&P};
    const dim3 grid(pl.ntiles, nbatch), block(S.NT());
    // every advance may be followed by one exact re-run; plus replay and copy
    const long long bound = 2ll * ((max_sweeps + pl.m - 1) / pl.m) + 4;
    const int chunk = h->opt_chunk < 1 ? 1 : h->opt_chunk;
    long long launched = 0;
    int poll = 0;
    bool have_poll[2] = {false, false};
    bool all_done = false;
    while (launched < bound && !all_done) {
        for (int i = 0; i < chunk && launched < bound; ++i, ++launched) {
            CU_TRY(cudaLaunchKernel(S.fn, grid, block, args, S.smem, st));
            h->st_launches += 1;
        }
        // poll the device-side decision one chunk behind, so the queue never drains
        CU_TRY(cudaMemcpyAsync(h->h_ctl + (size_t)poll * h->cap_batch, h->d_ctl, sizeof(Ctl) * nbatch,
                               cudaMemcpyDeviceToHost, st));
        CU_TRY(cudaEventRecord(h->ev_poll[poll], st));
        have_poll[poll] = true;
        const int prev = poll ^ 1;
        if (have_poll[prev]) {
            CU_TRY(cudaEventSynchronize(h->ev_poll[prev]));
            all_done = true;
            for (int b = 0; b < nbatch; ++b) all_done = all_done && h->h_ctl[(size_t)prev * h->cap_batch + b].done;
        }
        poll ^= 1;
    }
    h->st_path = 3;
    h->st_ctas = (double)pl.ntiles * nbatch; h->st_tile_w = pl.ow; h->st_tile_h = pl.oh; h->st_tblock = pl.m;
    h->st_shape = pl.shape;
    h->st_redund = (double)pl.ntiles * S.BW() * S.BH() / ((double)h->nr * h->nz);
    return 0;
}


// ---- resident path: shapes, planner, launcher ------------------------------------------------------------------
const std::vector<ShapeInfo>& shapes() {
    static const std::vector<ShapeInfo> v = [] {
        std::vector<ShapeInfo> t;
        for (int i = 0; i < kNumResShapes; ++i) t.push_back(res_shape(i));      // shape_tu.cu: one translation unit per shape
        return t;
    }();
    return v;
}

// Modelled SM clocks of one half-sweep of a box when `k` CTAs of that shape share an SM, calibrated with the
// in-kernel profile ("prof" option; profiles/r01c_resident_inkernel.md): a warp needs `lat` clocks for its 2H cell
// updates (7 dependent fp64 instructions each, little ILP left once 4 x H values of phi live in registers), and the
// fp64 pipe issues one warp instruction per 2 clocks per SM sub-partition at ~62 % efficiency.
double model_half_sweep(const ShapeInfo& S, int k) {
    const double dpw = 2.0 * S.H * 7.0;                          // fp64 instructions per warp and half-sweep
    const double lat = S.H <= 2 ? 215.0 : S.H <= 4 ? 420.0 : S.H <= 6 ? 480.0 : 545.0;
    const double warps_per_smsp = std::ceil(k * (S.NT() / 32.0) / 4.0);
    // CTAs sharing an SM also share its latency-bound phases (measured: ~ +50 % per extra CTA)
    // ... and every half-sweep costs each warp ~70 + 22 H issue slots (SASS of the sweep loops: 102 instructions per
    // half-sweep at H = 2, ~250 at H = 8), one per clock and sub-partition: the limit of the many-warp small-patch shapes
    const double issue = warps_per_smsp * (70.0 + 22.0 * S.H);
    double t = std::max(std::max(lat * (1.0 + 0.5 * (k - 1)), warps_per_smsp * dpw * 2.0 / 0.62 + 100.0), issue);
    if (S.threads() * S.minb > 448 && k == 1 && S.H == 8 && S.NT() < 448) t = std::max(t, 1400.0);   // 128-register cap
    return t;
}

// Can `nclusters` clusters of `csize` CTAs of this shape be resident at once?
bool cluster_fits(sn_poisson* h, const ShapeInfo& S, int fi, int csize, int nclusters) {
    const void* fn = S.fn[fi];
    if (cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S.smem_of(fi)) != cudaSuccess ||
        (csize > 8 && cudaFuncSetAttribute(fn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess)) {
        cudaGetLastError();
        return false;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(csize, nclusters);
    cfg.blockDim = dim3(S.threads());
    cfg.dynamicSmemBytes = S.smem_of(fi);
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = csize; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, fn, &cfg) != cudaSuccess) { cudaGetLastError(); return false; }
    (void)h;
    return n >= nclusters;
}

// Pick (shape, mode, m) minimising modelled clocks per sweep; honours the "shape" / "tblock" / "halo" overrides.
ResPlan plan_resident(sn_poisson* h, int nbatch, const double* rho, const double* phi) {
    ResPlan best;
    if (((uintptr_t)rho | (uintptr_t)phi) & 15) return best;
    const auto& sh = shapes();
    for (int si = 0; si < (int)sh.size(); ++si) {
        if (h->opt_shape >= 0 && si != h->opt_shape) continue;
        const ShapeInfo& S = sh[si];
        const int halo_fn = h->opt_ring != 0 ? 3 : 1;      // halo mode through L2 packets: ring duty unless switched off
        long long max_ctas_mode[2] = {0, 0};
        for (int md = 0; md < 2; ++md) {
            const int f = md == 0 ? 0 : halo_fn;
            int occ = 0;
            if (!S.fn[f]) { max_ctas_mode[md] = 0; continue; }       // shape without this mode
            if (cudaFuncSetAttribute(S.fn[f], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S.smem_of(f)) != cudaSuccess ||
                cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, S.fn[f], S.threads(), S.smem_of(f)) != cudaSuccess) {
                cudaGetLastError();
                occ = 0;
            }
            max_ctas_mode[md] = (long long)occ * h->num_sms;
        }
        // halo mode: box == tile on a regular lattice, ragged last tile row allowed
        if (h->opt_halo != 0 && S.fn[halo_fn] && h->nr % S.BW() == 0 && h->nz % S.H == 0) {
            ResPlan p;
            p.shape = si; p.halo = 1; p.ring = halo_fn == 3;
            p.ntx = h->nr / S.BW(); p.nty = (h->nz + S.BH() - 1) / S.BH();
            p.ow = S.BW(); p.oh = S.BH();
            p.ntiles = p.ntx * p.nty;
            p.Q = h->opt_tblock > 0 ? h->opt_tblock : kMaxTB;
            p.m = p.Q;
            if ((long long)p.ntiles * nbatch <= max_ctas_mode[1] && (p.ntiles > 1 || h->opt_halo == 1)) {
                const int k = (int)((p.ntiles * (long long)nbatch + h->num_sms - 1) / h->num_sms);
                // per half-sweep: compute + the exposed part of the edge exchange (poll round trips, barrier, the
                // neighbour's slowest warp) + the checkpoint / report of the interval
                // (ring duty: the packet flight overlaps the patch update; what stays exposed is the ring duty itself, one
                // L2 round trip of the poll and the barrier skew -- calibrated on profiles/r02_ring.md)
                p.cost = 2.0 * (model_half_sweep(S, k) + (p.ring ? 1350.0 + 0.05 * S.BW() * S.BH() : 1500.0 + 0.1 * S.BW() * S.BH()));
                if (best.shape < 0 || p.cost < best.cost) best = p;
            }
        }
        // halo mode with all tiles of a member in ONE thread-block cluster: edges through distributed shared memory
        if (h->opt_halo != 0 && h->opt_ds != 0 && S.fn[2] && h->nr % S.BW() == 0 && h->nz % S.H == 0) {
            ResPlan p;
            // ring duty in cluster mode only on request: a DSMEM st.async needs ~550 clocks until the mbarrier fires,
            // more than the patch update of the small boxes this mode serves, so sending first gains nothing there
            p.shape = si; p.halo = 1; p.ds = 1; p.ring = h->opt_ring == 1;
            p.ntx = h->nr / S.BW(); p.nty = (h->nz + S.BH() - 1) / S.BH();
            p.ow = S.BW(); p.oh = S.BH();
            p.ntiles = p.ntx * p.nty;
            p.Q = h->opt_tblock > 0 ? h->opt_tblock : kMaxTB;
            p.m = p.Q;
            // members are independent and a cluster is gang-scheduled, so the clusters of a batch need not be
            // co-resident with each other: any batch size runs, in waves of clusters if it has to
            if (p.ntiles > 1 && p.ntiles <= 16 && cluster_fits(h, S, p.ring ? 4 : 2, p.ntiles, 1)) {
                // per half-sweep: compute + the edge threads' st.async (~250 clocks) + one DSMEM hop and the mbarrier
                // wake-up (~300); 420 puts the model where the measurements are (128^2: wins; 64^2, 256^2: block mode)
                p.cost = 2.0 * (model_half_sweep(S, 1) + 420.0);
                if (best.shape < 0 || p.cost < best.cost || h->opt_ds == 1) best = p;
            }
        }
        if (h->opt_ds == 1 && best.ds) continue;
        if (h->opt_halo == 1) continue;
        // block mode: temporal blocking with margins of 2m cells
        for (int m = 1; m <= kMaxTB; ++m) {
            if (h->opt_tblock > 0 && m != h->opt_tblock) continue;
            ResPlan p;
            if (!plan_axis(h->nr, S.BW(), 2 * m, 4, &p.ntx, &p.ow)) continue;
            if (!plan_axis(h->nz, S.BH(), 2 * m, S.H, &p.nty, &p.oh)) continue;
            p.ntiles = p.ntx * p.nty;
            if ((long long)p.ntiles * nbatch > max_ctas_mode[0]) continue;
            bool ok = true;                      // the property the kernel relies on, checked for every tile
            for (int t = 0; t < p.ntx && ok; ++t) ok = box_covers(t, p.ow, 2 * m, 4, S.BW(), h->nr);
            for (int t = 0; t < p.nty && ok; ++t) ok = box_covers(t, p.oh, 2 * m, S.H, S.BH(), h->nz);
            if (!ok) continue;
            p.shape = si; p.halo = 0; p.m = m; p.Q = m;
            p.ll = h->opt_ll >= 0 ? h->opt_ll : (S.H == 2 && p.ow * p.oh <= 256 ? 1 : 0);   // tiny tiles: packets beat flags
            const int k = (int)((p.ntiles * (long long)nbatch + h->num_sms - 1) / h->num_sms);
            // per exchange: checkpoint store, release of the tile flag, the neighbours' acquire, margin refill
            // (tagged packets: every non-owned cell of the box is polled -- measured 5.5 k clocks for a 32 x 32 box, 13 k
            // for 64 x 64)
            const double exchange = p.ntiles == 1 ? 2000.0 : p.ll ? 2500.0 + 2.6 * S.BW() * S.BH() : 4200.0 + 0.7 * S.BW() * S.BH();
            // CTAs sharing an SM overlap one's flag wait with the other's sweeps; polling packets instead competes
            // for issue slots (measured)
            p.cost = 2.0 * model_half_sweep(S, k) + exchange * (p.ll ? 1.0 + 0.5 * (k - 1) : 1.0) / m;
            if (best.shape < 0 || p.cost < best.cost) best = p;
        }
    }
    return best;
}

// Members member0 .. member0 + nbatch - 1 of the caller's batch (rho, phi point at member 0 of the batch).
int run_resident(sn_poisson* h, const Geom& g, const ResPlan& pl, int nbatch, const double* rho, double* phi,
                 int max_sweeps, cudaStream_t st, int member0 = 0, double* gr = nullptr, double* gz = nullptr) {
    const ShapeInfo& S = shapes()[pl.shape];
    const size_t ncell = (size_t)h->nr * h->nz;
    const size_t nint = (size_t)(max_sweeps + pl.Q - 1) / pl.Q;
    const size_t need_ring = (size_t)nbatch * kResRing * ncell;
    const size_t need_mail = pl.halo ? (size_t)nbatch * pl.ntiles * 2 * (S.BW() + S.BH())
                                     : pl.ll ? (size_t)nbatch * 2 * ncell : 1;                       // 16-byte packets
    const size_t need_sync = (size_t)nbatch * (2 * (nint + 2) + 1 + pl.ntiles);
    if (h->ring_cap < need_ring) {
        cudaFree(h->d_ring); h->d_ring = nullptr; h->ring_cap = 0;
        CU_TRY(cudaMalloc((void**)&h->d_ring, sizeof(double) * need_ring));
        h->ring_cap = need_ring;
    }
    if (h->mail_cap < need_mail) {
        cudaFree(h->d_mail); h->d_mail = nullptr; h->mail_cap = 0;
        CU_TRY(cudaMalloc((void**)&h->d_mail, 16 * need_mail));
        h->mail_cap = need_mail;
    }
    if (h->sync_cap < need_sync) {
        cudaFree(h->d_sync); h->d_sync = nullptr; h->sync_cap = 0;
        CU_TRY(cudaMalloc((void**)&h->d_sync, sizeof(unsigned int) * need_sync));
        h->sync_cap = need_sync;
    }
    CU_TRY(cudaMemsetAsync(h->d_sync, 0, sizeof(unsigned int) * need_sync, st));
    CU_TRY(cudaMemset2DAsync(h->d_slots_f + (size_t)member0 * 2 * h->cap_sweeps, sizeof(unsigned int) * 2 * (size_t)h->cap_sweeps,
                             0, sizeof(unsigned int) * 2 * (size_t)std::max(1, max_sweeps), nbatch, st));
    if ((pl.halo && !pl.ds) || pl.ll) CU_TRY(cudaMemsetAsync(h->d_mail, 0, 16 * need_mail, st));   // packet tags start at 1
    ResParams P;
    P.g = g;
    P.g.slots0_f += (size_t)member0 * h->cap_sweeps;         // the kernel indexes members from 0
    P.g.slots0_x += (size_t)member0 * h->cap_sweeps;
    P.halo = pl.halo;
    P.ll = pl.ll;
    P.ntx = pl.ntx; P.nty = pl.nty; P.ow = pl.ow; P.oh = pl.oh; P.m = pl.m; P.Q = pl.Q;
    P.max_sweeps = max_sweeps;
    P.force_exact = h->opt_exact;
    P.rho = rho + (size_t)member0 * ncell; P.phi = phi + (size_t)member0 * ncell;
    P.ring = h->d_ring;
    P.mail = reinterpret_cast<uint4*>(h->d_mail);
    P.bE = h->d_bE + (size_t)member0 * h->nz; P.bN = h->d_bN + (size_t)member0 * h->nr;
    P.bS = h->d_bS + (size_t)member0 * h->nr;
    P.slots_f = h->d_slots_f + (size_t)member0 * 2 * h->cap_sweeps;
    P.slots_x = h->d_slots + (size_t)member0 * 2 * h->cap_sweeps;
    P.slot_stride = 2 * h->cap_sweeps; P.hist_stride = h->cap_sweeps;
    P.arrived = h->d_sync;
    P.arr_stride = (int)(nint + 2);
    P.gbar = h->d_sync + (size_t)nbatch * 2 * (nint + 2);
    P.flags = P.gbar + nbatch;
    P.ctl = h->d_ctl + member0; P.hist = h->d_hist + (size_t)member0 * h->cap_sweeps;
    P.prof = nullptr;
    P.gr = gr ? gr + (size_t)member0 * ncell : nullptr;
    P.gz = gz ? gz + (size_t)member0 * ncell : nullptr;
    h->prof_ctas = 0;
    if (h->opt_prof) {
        const size_t need = (size_t)pl.ntiles * nbatch * 8;
        if (h->prof_cap < need) {
            cudaFree(h->d_prof); h->d_prof = nullptr; h->prof_cap = 0;
            CU_TRY(cudaMalloc((void**)&h->d_prof, sizeof(long long) * need));
            h->prof_cap = need;
        }
        CU_TRY(cudaMemsetAsync(h->d_prof, 0, sizeof(long long) * need, st));
        P.prof = h->d_prof;
        h->prof_ctas = (size_t)pl.ntiles * nbatch;
    }
    void* args[] = {&P};
    const int fi = pl.ds ? (pl.ring ? 4 : 2) : pl.halo ? (pl.ring ? 3 : 1) : 0;
    const void* fn = S.fn[fi];
    const size_t smem = S.smem_of(fi);
    // (the planner has already set the kernel's shared-memory attribute; plans are cached on the handle)
    if (pl.ds) {
        // one cluster per member (gang-scheduled, so its CTAs are co-resident by construction; the clusters of a batch
        // were checked against cudaOccupancyMaxActiveClusters by the planner)
        if (pl.ntiles > 8) CU_TRY(cudaFuncSetAttribute(fn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(pl.ntiles, nbatch);
        cfg.blockDim = dim3(S.threads());
        cfg.dynamicSmemBytes = smem;
        cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = pl.ntiles; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        CU_TRY(cudaLaunchKernelExC(&cfg, fn, args));
    } else {
        CU_TRY(cudaLaunchCooperativeKernel(fn, dim3(pl.ntiles, nbatch), dim3(S.threads()), args, smem, st));
    }
    h->st_launches += 1;
    h->st_path = 2;
    h->st_ctas = (double)pl.ntiles * nbatch; h->st_tile_w = pl.ow; h->st_tile_h = pl.oh; h->st_tblock = pl.Q;
    h->st_shape = pl.shape; h->st_halo = pl.halo; h->st_group = nbatch; h->st_ds = pl.ds; h->st_ring = pl.ring;
    h->st_redund = pl.halo ? 1.0 : (double)pl.ntiles * S.BW() * S.BH() / ((double)h->nr * h->nz);
    return 0;
}

// Hooks of the host-buffer entry points into one solve: an event the relaxation must wait for (phi's H2D on the copy
// stream) and a device -> host copy enqueued right after the relaxation, before the call's single synchronisation.
struct HostIO {
    double* gr = nullptr;        // fused gravity epilogue: DEVICE outputs [nbatch][ncell] (NULL: none)
    double* gz = nullptr;
    cudaEvent_t wait_before_relax = nullptr;
    double* d2h_dst = nullptr;
    const double* d2h_src = nullptr;
    size_t d2h_bytes = 0;
};

// The plan of a solve depends only on (nbatch, pointer alignment, options): planned once, cached on the handle
// (set_option invalidates).  The planners also set the kernels' shared-memory attributes, once.
void plan_solve(sn_poisson* h, int nbatch, const double* rho, const double* phi, ResPlan* pl_out, BlkPlan* bp_out,
                int* group_out) {
    const int aligned = ((((uintptr_t)rho | (uintptr_t)phi) & 15) == 0) ? 1 : 0;
    auto& pc = h->plan_cache;
    if (pc.valid && pc.nbatch == nbatch && pc.aligned == aligned) {
        *pl_out = pc.pl; *bp_out = pc.bp; *group_out = pc.group;
        return;
    }
    ResPlan pl;
    BlkPlan bp;
    int group = nbatch;          // members per resident launch
    if (h->opt_path == 0 || h->opt_path == 2) {
        pl = plan_resident(h, nbatch, rho, phi);
        // A batch whose tiles cannot all be co-resident: solve it in groups of G members, one resident launch after
        // the other, if a group fills the chip (otherwise the blocked path streams the whole batch).  "group"
        // option: 0 never, G > 0 exactly G, -1 this rule.
        const bool forced = h->opt_group > 0 && h->opt_group < nbatch;
        if (forced) pl = ResPlan();
        if (pl.shape < 0 && nbatch > 1 && h->opt_group != 0) {
            double best_total = 0;
            for (int G = std::min(nbatch - 1, h->opt_group > 0 ? h->opt_group : nbatch - 1); G >= 1; --G) {
                if (h->opt_group > 0 && G != h->opt_group) break;
                const ResPlan cand = plan_resident(h, G, rho, phi);
                if (cand.shape < 0) continue;
                const double total = cand.cost * ((nbatch + G - 1) / G);
                if (pl.shape < 0 || total < best_total) { pl = cand; best_total = total; group = G; }
            }
            const int occ_ctas = pl.shape >= 0 ? pl.ntiles * group : 0;
            if (pl.shape >= 0 && !forced && (occ_ctas < 1.7 * h->num_sms || !pl.halo)) pl = ResPlan();
            if (pl.shape < 0) group = nbatch;
        }
    }
    if ((h->opt_path == 0 || h->opt_path == 3) && pl.shape < 0) bp = plan_blocked(h, nbatch, rho, phi);
    pc.valid = true; pc.nbatch = nbatch; pc.aligned = aligned; pc.pl = pl; pc.bp = bp; pc.group = group;
    *pl_out = pl; *bp_out = bp; *group_out = group;
}

int launch_gravity(sn_poisson* h, const Geom& g, int nbatch, const double* phi, double* gr, double* gz, cudaStream_t st) {
    const bool vec = h->nr % 4 == 0 && ((((uintptr_t)phi | (uintptr_t)gr | (uintptr_t)gz) & 15) == 0);
    if (vec) {
        const unsigned qx = (h->nr / 4 + 127) / 128;                       // rows folded into grid.x: no 65535 limit on nz
        const dim3 grid(qx * (unsigned)h->nz, 1, nbatch);
        k_gravity4<<<grid, 128, 0, st>>>(g, (int)qx, phi, h->d_bE, h->d_bN, h->d_bS, gr, gz);
    } else {
        const unsigned qx = (h->nr + 127) / 128;
        const dim3 grid(qx * (unsigned)h->nz, 1, nbatch);
        k_gravity1<<<grid, 128, 0, st>>>(g, (int)qx, phi, h->d_bE, h->d_bN, h->d_bS, gr, gz);
    }
    CU_TRY(cudaGetLastError());
    return 0;
}

int solve_impl(sn_poisson* h, int nbatch, const double* rho, double* phi, double tol, int max_sweeps,
               cudaStream_t st, sn_poisson_result* out, const HostIO* io = nullptr) {
    CU_TRY(cudaSetDevice(h->device));
    if (int rc = ensure_ws(h, nbatch, max_sweeps)) return rc;
    if (!h->omega_user) h->omega = default_omega(h->nr, h->nz, h->dr, h->dz, h->symmetry);
    const Geom g = make_geom(h, tol);
    h->st_launches = 0;
    h->st_aux_launches = 0;
    h->st_path = 1;
    h->st_halo = 0;
    h->st_ds = 0;
    h->st_ring = 0;
    h->st_redund = 1;

    CU_TRY(cudaEventRecord(h->ev_t[0], st));
    CU_TRY(cudaMemsetAsync(h->d_ctl, 0, sizeof(Ctl) * nbatch, st));
    CU_TRY(cudaMemset2DAsync(h->d_slots, sizeof(unsigned long long) * 2 * (size_t)h->cap_sweeps, 0,
                             sizeof(unsigned long long) * 2 * (size_t)std::max(1, max_sweeps), nbatch, st));
    if (h->opt_rule != 0 && h->symmetry == 1) {
        CU_TRY(cudaMemset2DAsync(h->d_slots0, sizeof(unsigned long long) * (size_t)h->cap_sweeps, 0,
                                 sizeof(unsigned long long) * (size_t)std::max(1, max_sweeps), nbatch, st));
        CU_TRY(cudaMemset2DAsync(h->d_slots0_f, sizeof(unsigned int) * (size_t)h->cap_sweeps, 0,
                                 sizeof(unsigned int) * (size_t)std::max(1, max_sweeps), nbatch, st));
    }
    // a-1: moments (+ max|4 pi rho|), a-1b: boundary fill (skipped when ghosts were injected by the test hook)
    if (int rc = launch_moments(h, g, nbatch, rho, st)) return rc;
    h->st_launches += 1;
    h->st_aux_launches += 1;
    if (!h->user_boundary) {
        k_boundary<<<dim3(nbatch, boundary_slices(h)), 256, 0, st>>>(g, h->L0, h->NL, h->mom_blocks, h->d_partial, h->d_M, h->d_bE, h->d_bN,
                                           h->d_bS, 0);
        CU_TRY(cudaGetLastError());
        h->st_launches += 1;
        h->st_aux_launches += 1;
    }
    h->last_nbatch = h->user_boundary ? h->cap_batch : nbatch;
    CU_TRY(cudaEventRecord(h->ev_t[1], st));
    if (io && io->wait_before_relax) CU_TRY(cudaStreamWaitEvent(st, io->wait_before_relax, 0));
    // a-2 + a-3
    ResPlan pl;
    BlkPlan bp;
    int group = nbatch;
    if (max_sweeps > 0) plan_solve(h, nbatch, rho, phi, &pl, &bp, &group);
    if (h->opt_path == 2 && pl.shape < 0 && max_sweeps > 0) {
        set_err("resident path requested but not eligible (needs nr%%4==0, nz%%H==0, grid >= one box, 16-byte aligned "
                "pointers, tiles x batch <= co-resident CTAs)");
        return -1;
    }
    if (h->opt_path == 3 && bp.shape < 0 && max_sweeps > 0) {
        set_err("blocked path requested but not eligible (needs nr%%4==0, nz%%H==0, grid >= one box, 16-byte aligned "
                "pointers)");
        return -1;
    }
    if (pl.shape >= 0) {
        // the fused epilogue stores gr / gz as double2: it needs them 16-byte aligned (rho / phi are, or the resident path
        // would not have been planned).  Output arrays that are only 8-byte aligned get the standalone kernel instead,
        // which picks its scalar variant -- same values, bit for bit.
        const bool fused = io && io->gr && ((((uintptr_t)io->gr | (uintptr_t)io->gz) & 15) == 0);
        for (int m0 = 0; m0 < nbatch; m0 += group)
            if (int rc = run_resident(h, g, pl, std::min(group, nbatch - m0), rho, phi, max_sweeps, st, m0,
                                      fused ? io->gr : nullptr, fused ? io->gz : nullptr)) return rc;
        h->st_group = group;
        h->st_ctas = (double)pl.ntiles * group;
        if (io && io->gr && !fused)
            if (int rc = launch_gravity(h, g, nbatch, phi, io->gr, io->gz, st)) return rc;
    } else {
        if (bp.shape >= 0) {
            if (int rc = run_blocked(h, g, bp, nbatch, rho, phi, max_sweeps, st)) return rc;
        } else {
            if (int rc = run_stream(h, g, nbatch, rho, phi, max_sweeps, st)) return rc;
        }
        // the streamed / blocked paths have no phi on chip at the end: the epilogue is the standalone kernel, enqueued
        // right behind the last sweep (phi is still L2-resident for grids that fit)
        if (io && io->gr)
            if (int rc = launch_gravity(h, g, nbatch, phi, io->gr, io->gz, st)) return rc;
    }
    CU_TRY(cudaEventRecord(h->ev_t[2], st));
    if (io && io->d2h_dst)
        CU_TRY(cudaMemcpyAsync(io->d2h_dst, io->d2h_src, io->d2h_bytes, cudaMemcpyDeviceToHost, st));
    CU_TRY(cudaMemcpyAsync(h->h_ctl, h->d_ctl, sizeof(Ctl) * nbatch, cudaMemcpyDeviceToHost, st));
    CU_TRY(cudaStreamSynchronize(st));
    float ms = 0;
    CU_TRY(cudaEventElapsedTime(&ms, h->ev_t[0], h->ev_t[1]));
    h->st_setup_ms = ms;
    CU_TRY(cudaEventElapsedTime(&ms, h->ev_t[1], h->ev_t[2]));
    h->st_sweep_ms = ms;
    for (int b = 0; b < nbatch; ++b) {
        if (h->h_ctl[b].panic) {
            set_err("resident kernel watchdog: a wait exceeded its budget (member %d, code %d, tile %d, arg %d)", b,
                    h->h_ctl[b].panic, h->h_ctl[b].panic_tile, h->h_ctl[b].panic_arg);
            return -2;
        }
        if (!h->h_ctl[b].done) {
            set_err("internal error: member %d not finished after the enqueued launches", b);
            return -2;
        }
        out[b].sweeps = h->h_ctl[b].sweeps;
        out[b].status = h->h_ctl[b].status;
        out[b].residual = h->h_ctl[b].residual;
    }
    h->last_sweeps0 = out[0].sweeps;
    if (h->prof_ctas) {                         // in-kernel profile of the resident kernel: mean / max over its CTAs
        std::vector<long long> pf(h->prof_ctas * 8);
        CU_TRY(cudaMemcpy(pf.data(), h->d_prof, sizeof(long long) * pf.size(), cudaMemcpyDeviceToHost));
        for (int i = 0; i < 8; ++i) {
            double sum = 0, mx = 0;
            for (size_t c = 0; c < h->prof_ctas; ++c) {
                sum += (double)pf[c * 8 + i];
                mx = std::max(mx, (double)pf[c * 8 + i]);
            }
            h->prof_mean[i] = sum / h->prof_ctas;
            h->prof_max[i] = mx;
        }
    }
    return 0;
}

bool check_solve_args(sn_poisson* h, const void* rho, const void* phi, double tol, int max_sweeps, int nbatch = 1) {
    if (!h) { set_err("NULL handle"); return false; }
    if (!rho || !phi) { set_err("NULL rho / phi pointer"); return false; }
    if (max_sweeps < 0) { set_err("max_sweeps < 0"); return false; }
    if (max_sweeps > kMaxSweepsLimit || (long long)max_sweeps * nbatch > kMaxSweepSlots) {
        set_err("max_sweeps too large: the per-sweep bookkeeping allows max_sweeps <= %d and max_sweeps x nbatch <= %lld",
                kMaxSweepsLimit, kMaxSweepSlots);
        return false;
    }
    if (tol != tol) { set_err("tol is NaN"); return false; }
    return true;
}

// Device staging of the host-buffer entry points: `n` doubles each for rho and phi, grown on demand and kept.
int ensure_stage(sn_poisson* h, size_t n) {
    if (!h->st_copy) {
        CU_TRY(cudaStreamCreateWithFlags(&h->st_copy, cudaStreamNonBlocking));
        for (auto& e : h->ev_io) CU_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    }
    if (h->stage_cap >= n) return 0;
    cudaFree(h->d_rho_stage); cudaFree(h->d_phi_stage);
    h->d_rho_stage = h->d_phi_stage = nullptr;
    h->stage_cap = 0;
    CU_TRY(cudaMalloc((void**)&h->d_rho_stage, sizeof(double) * n));
    CU_TRY(cudaMalloc((void**)&h->d_phi_stage, sizeof(double) * n));
    h->stage_cap = n;
    return 0;
}

}  // namespace

namespace {

// ---- multigrid variant (NEXT-4; mg.cuh, readings M1..M8) ---------------------------------------------------------
int mg_num_levels(int nr, int nz) {                                  // M1
    int n = 1;
    while (nr % 2 == 0 && nz % 2 == 0 && nr / 2 >= 4 && nz / 2 >= 4) { nr /= 2; nz /= 2; ++n; }
    return n;
}

// Releases the level arrays of the multigrid workspace and marks it as not built (the stream and the pinned history
// buffer are independent of the level layout and stay).
void free_mg_levels(sn_poisson* h) {
    auto& W = h->mg;
    if (W.exec) { cudaGraphExecDestroy(W.exec); W.exec = nullptr; }
    for (auto* v : {&W.cE, &W.cW, &W.phi, &W.f}) {
        for (double* p : *v) cudaFree(p);
        v->clear();
    }
    cudaFree(W.slots); W.slots = nullptr;
    cudaFree(W.d_ptrs); W.d_ptrs = nullptr;
    W.nlev = 0;
    W.cap_batch = 0;
    W.key = {};
}

int ensure_mg_levels(sn_poisson* h, int nbatch);

// Builds / grows the multigrid workspace.  A failure half way (out of memory while growing for a larger batch, or
// during the first build) would leave level pointers NULL under a non-zero nlev / cap_batch, or leak the levels already
// allocated: on any failure everything is released and the next call rebuilds from scratch.
int ensure_mg(sn_poisson* h, int nbatch) {
    const int rc = ensure_mg_levels(h, nbatch);
    if (rc) free_mg_levels(h);
    return rc;
}

int ensure_mg_levels(sn_poisson* h, int nbatch) {
    auto& W = h->mg;
    if (W.nlev && nbatch > W.cap_batch) {        // grow the per-member arrays (the captured cycle holds their addresses)
        if (W.exec) { cudaGraphExecDestroy(W.exec); W.exec = nullptr; }
        for (int l = 1; l < W.nlev; ++l) {
            cudaFree(W.phi[l]); cudaFree(W.f[l]);
            W.phi[l] = W.f[l] = nullptr;
            if (int rc = dev_alloc(&W.phi[l], (size_t)nbatch * W.nr[l] * W.nz[l])) return rc;
            if (int rc = dev_alloc(&W.f[l], (size_t)nbatch * W.nr[l] * W.nz[l])) return rc;
        }
        cudaFree(W.slots); W.slots = nullptr;
        if (int rc = dev_alloc(&W.slots, (size_t)2 * nbatch)) return rc;
        W.cap_batch = nbatch;
    }
    if (W.nlev) return 0;
    const int nlev = std::min(mg_num_levels(h->nr, h->nz), kMgMaxLevels);
    W.nr.resize(nlev); W.nz.resize(nlev);
    W.cE.assign(nlev, nullptr); W.cW.assign(nlev, nullptr); W.phi.assign(nlev, nullptr); W.f.assign(nlev, nullptr);
    for (int l = 0; l < nlev; ++l) {
        const int nr = h->nr >> l, nz = h->nz >> l;
        W.nr[l] = nr; W.nz[l] = nz;
        const double dr = std::ldexp(h->dr, l);
        const double ir2 = 1.0 / (dr * dr);
        std::vector<double> cE(nr), cW(nr);
        for (int i = 0; i < nr; ++i) {
            cE[i] = ((i + 1.0) / (i + 0.5)) * ir2;
            cW[i] = (i / (i + 0.5)) * ir2;
        }
        if (int rc = dev_alloc(&W.cE[l], (size_t)nr)) return rc;
        if (int rc = dev_alloc(&W.cW[l], (size_t)nr)) return rc;
        CU_TRY(cudaMemcpy(W.cE[l], cE.data(), sizeof(double) * nr, cudaMemcpyHostToDevice));
        CU_TRY(cudaMemcpy(W.cW[l], cW.data(), sizeof(double) * nr, cudaMemcpyHostToDevice));
        if (l > 0) {
            if (int rc = dev_alloc(&W.phi[l], (size_t)nbatch * nr * nz)) return rc;
            if (int rc = dev_alloc(&W.f[l], (size_t)nbatch * nr * nz)) return rc;
        }
    }
    if (int rc = dev_alloc(&W.slots, (size_t)2 * nbatch)) return rc;
    W.cap_batch = nbatch;
    if (int rc = dev_alloc(&W.d_ptrs, (size_t)1)) return rc;
    CU_TRY(cudaFuncSetAttribute(k_mg_tail, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
    W.tail_attr = true;
    W.nlev = nlev;
    return 0;
}

MgLevel mg_level(const sn_poisson* h, int l, const double* rho, double* phi) {
    const auto& W = h->mg;
    MgLevel L;
    L.nr = W.nr[l]; L.nz = W.nz[l]; L.symmetry = h->symmetry;
    const double dr = std::ldexp(h->dr, l), dz = std::ldexp(h->dz, l);
    const double ir2 = 1.0 / (dr * dr);
    L.iz2 = 1.0 / (dz * dz);
    L.D = 2.0 * ir2 + 2.0 * L.iz2;
    L.D0 = L.D - L.iz2;
    L.wD = 1.0 / L.D;
    L.wD0 = 1.0 / L.D0;
    const double s = std::ldexp(1.0, -l);
    L.beta = (1.0 - s) / (1.0 + s);
    L.scale = l == 0 ? kFourPi : 1.0;
    L.cE = W.cE[l]; L.cW = W.cW[l];
    L.phi = l == 0 ? nullptr : W.phi[l];          // level 0: resolved on the device through MgPtrs (mg.cuh)
    L.src = l == 0 ? nullptr : W.f[l];
    (void)rho; (void)phi;
    L.bE = l == 0 ? h->d_bE : nullptr;
    L.bN = l == 0 ? h->d_bN : nullptr;
    L.bS = l == 0 ? h->d_bS : nullptr;
    return L;
}

// blocks per member: one thread per unit, at most 16 CTAs per SM over the whole batch
inline int mg_blocks(size_t n, int num_sms, int nb = 1) {
    return (int)std::max<size_t>(1, std::min<size_t>((n + 255) / 256, std::max<size_t>(1, (size_t)num_sms * 16 / nb)));
}

// 32-bit cell indices (a 64-bit division per cell is a third of these kernels' instructions) where they suffice
inline bool mg_small(int nr, int nz) { return (long long)nr * nz < (1ll << 30); }

int mg_smooth(sn_poisson* h, const MgLevel& L, int nsweeps, cudaStream_t st) {
    const dim3 blocks(mg_blocks((size_t)((L.nr + 1) / 2) * L.nz, h->num_sms, h->mg.nb), h->mg.nb);
    const bool small = mg_small(L.nr, L.nz);
    for (int k = 0; k < nsweeps; ++k) {
        if (small) {
            k_mg_halfsweep<0, unsigned><<<blocks, 256, 0, st>>>(L, h->d_ctl, h->mg.d_ptrs);
            k_mg_halfsweep<1, unsigned><<<blocks, 256, 0, st>>>(L, h->d_ctl, h->mg.d_ptrs);
        } else {
            k_mg_halfsweep<0, size_t><<<blocks, 256, 0, st>>>(L, h->d_ctl, h->mg.d_ptrs);
            k_mg_halfsweep<1, size_t><<<blocks, 256, 0, st>>>(L, h->d_ctl, h->mg.d_ptrs);
        }
        h->st_launches += 2;
    }
    CU_TRY(cudaGetLastError());
    return 0;
}

// one V-cycle from level 0, then the true residual's maxima and the decision of the cycle (M8)
int mg_cycle(sn_poisson* h, const double* rho, double* phi, double tol, int max_cycles, cudaStream_t st) {
    const auto& W = h->mg;
    const int nu1 = h->opt_mg_nu1, nu2 = h->opt_mg_nu2;
    std::vector<MgLevel> Ls;
    for (int l = 0; l < W.nlev; ++l) Ls.push_back(mg_level(h, l, rho, phi));
    // levels 0 .. top-1 run as separate launches; the tail (every level of <= kMgTailCells cells) is ONE launch
    int k = W.nlev;
    for (int l = 0; l < W.nlev; ++l)
        if ((long long)W.nr[l] * W.nz[l] <= kMgTailCells) { k = l; break; }
    const int top = k < W.nlev ? k : W.nlev - 1;
    for (int l = 0; l < top; ++l) {                                  // down
        if (int rc = mg_smooth(h, Ls[l], nu1, st)) return rc;
        const size_t nc = (size_t)W.nr[l + 1] * W.nz[l + 1];
        if (mg_small(W.nr[l], W.nz[l]))
            k_mg_residual<true, false, unsigned><<<dim3(mg_blocks(nc, h->num_sms, W.nb), W.nb), 256, 0, st>>>(Ls[l], W.f[l + 1], W.phi[l + 1], nullptr, h->d_ctl, W.d_ptrs);
        else
            k_mg_residual<true, false, size_t><<<dim3(mg_blocks(nc, h->num_sms, W.nb), W.nb), 256, 0, st>>>(Ls[l], W.f[l + 1], W.phi[l + 1], nullptr, h->d_ctl, W.d_ptrs);
        h->st_launches += 1;
    }
    if (k < W.nlev) {
        MgTail T;
        T.n = W.nlev - k; T.nu1 = nu1; T.nu2 = nu2; T.nc = h->opt_mg_nc;
        for (int l = k; l < W.nlev; ++l) T.L[l - k] = Ls[l];
        const size_t smem = sizeof(double) * mg_tail_smem_doubles(T);
        k_mg_tail<<<W.nb, 1024, smem, st>>>(T, h->d_ctl, W.d_ptrs);
        h->st_launches += 1;
    } else {                                                         // a coarsest level too large for one CTA
        if (int rc = mg_smooth(h, Ls[W.nlev - 1], W.nlev == 1 ? nu1 + nu2 : h->opt_mg_nc, st)) return rc;
    }
    for (int l = top - 1; l >= 0; --l) {                             // up
        const size_t nf = (size_t)W.nr[l] * W.nz[l];
        if (mg_small(W.nr[l], W.nz[l]))
            k_mg_prolong_add<unsigned><<<dim3(mg_blocks(nf, h->num_sms, W.nb), W.nb), 256, 0, st>>>(Ls[l + 1], Ls[l].phi, W.nr[l], W.nz[l], h->d_ctl, W.d_ptrs);
        else
            k_mg_prolong_add<size_t><<<dim3(mg_blocks(nf, h->num_sms, W.nb), W.nb), 256, 0, st>>>(Ls[l + 1], Ls[l].phi, W.nr[l], W.nz[l], h->d_ctl, W.d_ptrs);
        h->st_launches += 1;
        if (int rc = mg_smooth(h, Ls[l], nu2, st)) return rc;
    }
    const size_t nb = (size_t)W.nr[0] * W.nz[0];
    if (mg_small(W.nr[0], W.nz[0])) k_mg_resmax<unsigned><<<dim3(mg_blocks(nb, h->num_sms, W.nb), W.nb), 256, 0, st>>>(Ls[0], W.slots, h->d_ctl, W.d_ptrs);
    else k_mg_resmax<size_t><<<dim3(mg_blocks(nb, h->num_sms, W.nb), W.nb), 256, 0, st>>>(Ls[0], W.slots, h->d_ctl, W.d_ptrs);
    k_mg_decide<<<W.nb, 32, 0, st>>>(h->d_ctl, W.slots, Ls[0].D, tol, max_cycles, h->d_hist, h->cap_sweeps);
    h->st_launches += 2;
    CU_TRY(cudaGetLastError());
    return 0;
}

// One cycle through the cached graph ("mg_graph" option, default on; the legacy default stream cannot be captured
// and takes the plain launches).
int mg_launch_cycle(sn_poisson* h, const double* rho, double* phi, double tol, int max_cycles, cudaStream_t st) {
    auto& W = h->mg;
    if (!h->opt_mg_graph || st == nullptr || st == cudaStreamLegacy) return mg_cycle(h, rho, phi, tol, max_cycles, st);
    const auto& k = W.key;
    const bool same = W.exec && k.tol == tol && k.max_cycles == max_cycles &&
                      k.nu1 == h->opt_mg_nu1 && k.nu2 == h->opt_mg_nu2 && k.nc == h->opt_mg_nc && k.nb == W.nb &&
                      k.cap_sweeps == h->cap_sweeps;
    if (!same) {
        if (W.exec) { cudaGraphExecDestroy(W.exec); W.exec = nullptr; }
        const double launches_before = h->st_launches;
        if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
            cudaGetLastError();
            return mg_cycle(h, rho, phi, tol, max_cycles, st);
        }
        const int rc = mg_cycle(h, rho, phi, tol, max_cycles, st);
        cudaGraph_t graph = nullptr;
        const cudaError_t e = cudaStreamEndCapture(st, &graph);
        W.nodes = h->st_launches - launches_before;
        h->st_launches = launches_before;
        if (rc || e != cudaSuccess || !graph) {
            cudaGetLastError();
            if (graph) cudaGraphDestroy(graph);
            if (rc) return rc;
            return mg_cycle(h, rho, phi, tol, max_cycles, st);
        }
        const cudaError_t ei = cudaGraphInstantiate(&W.exec, graph, 0);
        cudaGraphDestroy(graph);
        if (ei != cudaSuccess) {
            cudaGetLastError();
            W.exec = nullptr;
            return mg_cycle(h, rho, phi, tol, max_cycles, st);
        }
        W.key.tol = tol; W.key.max_cycles = max_cycles;
        W.key.nu1 = h->opt_mg_nu1; W.key.nu2 = h->opt_mg_nu2; W.key.nc = h->opt_mg_nc; W.key.nb = W.nb;
        W.key.cap_sweeps = h->cap_sweeps;
    }
    CU_TRY(cudaGraphLaunch(W.exec, st));
    h->st_launches += W.nodes;            // kernels of mine that run inside the graph
    return 0;
}

int solve_mg_impl(sn_poisson* h, int nbatch, const double* rho, double* phi, double tol, int max_cycles, cudaStream_t st,
                  sn_poisson_result* out, const HostIO* io = nullptr) {
    CU_TRY(cudaSetDevice(h->device));
    if (int rc = ensure_ws(h, nbatch, max_cycles)) return rc;
    if (int rc = ensure_mg(h, nbatch)) return rc;
    h->mg.nb = nbatch;
    const Geom g = make_geom(h, tol);
    h->st_launches = 0; h->st_aux_launches = 0;
    h->st_path = 4; h->st_halo = 0; h->st_ds = 0; h->st_ring = 0; h->st_redund = 1;
    h->st_ctas = 0; h->st_tile_w = h->nr; h->st_tile_h = h->nz; h->st_tblock = 0; h->st_shape = -1; h->st_group = nbatch;
    CU_TRY(cudaEventRecord(h->ev_t[0], st));
    CU_TRY(cudaMemsetAsync(h->d_ctl, 0, sizeof(Ctl) * nbatch, st));
    CU_TRY(cudaMemsetAsync(h->mg.slots, 0, 2 * sizeof(unsigned long long) * nbatch, st));
    {
        const MgPtrs hp = {rho, phi};
        CU_TRY(cudaMemcpyAsync(h->mg.d_ptrs, &hp, sizeof hp, cudaMemcpyHostToDevice, st));     // pageable: staged before return
    }
    if (int rc = launch_moments(h, g, nbatch, rho, st)) return rc;    // a-1 (+ max|4 pi rho|), a-1b as in the SOR path
    h->st_launches += 1; h->st_aux_launches += 1;
    if (!h->user_boundary) {
        k_boundary<<<dim3(nbatch, boundary_slices(h)), 256, 0, st>>>(g, h->L0, h->NL, h->mom_blocks, h->d_partial, h->d_M, h->d_bE, h->d_bN, h->d_bS, 0);
        CU_TRY(cudaGetLastError());
        h->st_launches += 1; h->st_aux_launches += 1;
    }
    h->last_nbatch = h->user_boundary ? h->cap_batch : nbatch;
    CU_TRY(cudaEventRecord(h->ev_t[1], st));
    if (io && io->wait_before_relax) CU_TRY(cudaStreamWaitEvent(st, io->wait_before_relax, 0));
    if (max_cycles == 0) {
        for (int b = 0; b < nbatch; ++b) {
            h->h_ctl[b] = Ctl();
            h->h_ctl[b].done = 1; h->h_ctl[b].status = tol > 0.0 ? 1 : 0;
        }
    }
    // The decision of a cycle is taken on the device (k_mg_decide, M8), per member; once `done` is set every later
    // kernel of the variant returns at once for that member, so cycles enqueued ahead neither touch its phi nor cost more
    // than their launches.  A host round trip costs about as much as a whole cycle of a small grid, so the host enqueues
    // cycles in chunks: two first, then as many as the measured contraction per cycle predicts the slowest member
    // still needs (a V-cycle contracts at a nearly constant rate), and looks at the decisions only between chunks.
    // tol <= 0: all cycles at once.
    if (max_cycles > 0) {
        if (h->mg.hist_cap < nbatch) {
            if (h->mg.h_hist) cudaFreeHost(h->mg.h_hist);
            h->mg.h_hist = nullptr; h->mg.hist_cap = 0;
            CU_TRY(cudaMallocHost((void**)&h->mg.h_hist, 2 * sizeof(double) * nbatch));
            h->mg.hist_cap = nbatch;
        }
        // The legacy default stream cannot be captured: the cycles then run on a stream of the handle, ordered after
        // the caller's stream here and before it again below.
        cudaStream_t caller = st;
        if (h->opt_mg_graph && (st == nullptr || st == cudaStreamLegacy)) {
            if (!h->mg.st) CU_TRY(cudaStreamCreateWithFlags(&h->mg.st, cudaStreamNonBlocking));
            CU_TRY(cudaEventRecord(h->ev_poll[0], caller));
            CU_TRY(cudaStreamWaitEvent(h->mg.st, h->ev_poll[0], 0));
            st = h->mg.st;
        }
        int enq = 0;
        int chunk = tol > 0.0 ? std::min(2, max_cycles) : max_cycles;
        for (;;) {
            for (int c = 0; c < chunk; ++c)
                if (int rc = mg_launch_cycle(h, rho, phi, tol, max_cycles, st)) return rc;
            enq += chunk;
            CU_TRY(cudaMemcpyAsync(h->h_ctl, h->d_ctl, sizeof(Ctl) * nbatch, cudaMemcpyDeviceToHost, st));
            if (enq >= 2)
                CU_TRY(cudaMemcpy2DAsync(h->mg.h_hist, 2 * sizeof(double), h->d_hist + (enq - 2), sizeof(double) * h->cap_sweeps,
                                         2 * sizeof(double), nbatch, cudaMemcpyDeviceToHost, st));
            CU_TRY(cudaStreamSynchronize(st));
            bool all_done = true;
            for (int b = 0; b < nbatch; ++b) all_done = all_done && h->h_ctl[b].done;
            if (all_done || enq >= max_cycles) break;
            chunk = 1;
            if (enq >= 2) {
                double need = 1.0;
                for (int b = 0; b < nbatch; ++b) {
                    const double r0 = h->mg.h_hist[2 * b], r1 = h->mg.h_hist[2 * b + 1];
                    if (h->h_ctl[b].done || !(r0 > 0.0) || !(r1 > 0.0)) continue;      // (a finished member's slots hold older cycles)
                    const double rate = std::min(0.5, std::max(0.02, r1 / r0));
                    need = std::max(need, std::ceil(std::log(tol / r1) / std::log(rate)));
                }
                chunk = (int)std::min(16.0, std::max(1.0, need));
            }
            chunk = std::min(chunk, max_cycles - enq);
        }
        if (st != caller) {                  // the loop above ended with st synchronised: the caller's stream may go on
            CU_TRY(cudaEventRecord(h->ev_poll[1], st));
            CU_TRY(cudaStreamWaitEvent(caller, h->ev_poll[1], 0));
            st = caller;
        }
    }
    CU_TRY(cudaEventRecord(h->ev_t[2], st));
    if (io && io->d2h_dst) CU_TRY(cudaMemcpyAsync(io->d2h_dst, io->d2h_src, io->d2h_bytes, cudaMemcpyDeviceToHost, st));
    CU_TRY(cudaStreamSynchronize(st));
    float ms = 0;
    CU_TRY(cudaEventElapsedTime(&ms, h->ev_t[0], h->ev_t[1]));
    h->st_setup_ms = ms;
    CU_TRY(cudaEventElapsedTime(&ms, h->ev_t[1], h->ev_t[2]));
    h->st_sweep_ms = ms;
    for (int b = 0; b < nbatch; ++b) {
        out[b].sweeps = h->h_ctl[b].sweeps;
        out[b].status = h->h_ctl[b].status;
        out[b].residual = h->h_ctl[b].residual;
    }
    h->last_sweeps0 = out[0].sweeps;
    return 0;
}

// Failure tail of the host-buffer entry points: wait for the caller's stream and the handle's copy stream, so that no
// copy enqueued by the failed call still reads or writes the caller's host memory after it returns.  Keeps the message
// of the original failure.
void drain_host_io(sn_poisson* h, cudaStream_t st) {
    cudaStreamSynchronize(st);
    if (h->st_copy) cudaStreamSynchronize(h->st_copy);
}

}  // namespace

extern "C" {

const char* sn_poisson_last_error(void) { return g_err.c_str(); }
const char* sn_poisson_version(void) { return "sn_poisson 0.1 (sm_100a)"; }

sn_poisson* sn_poisson_create(int nr, int nz, double dr, double dz, int symmetry, int lmax) {
    g_err.clear();
    if (nr < 2 || nz < 2) { set_err("nr, nz must be >= 2"); return nullptr; }
    if (!(dr > 0) || !(dz > 0) || !std::isfinite(dr) || !std::isfinite(dz)) {
        set_err("dr, dz must be finite and > 0");
        return nullptr;
    }
    if (symmetry != 0 && symmetry != 1) { set_err("symmetry must be 0 or 1"); return nullptr; }
    if (lmax < 0 || lmax > kMaxL) { set_err("lmax must be in [0, %d]", kMaxL); return nullptr; }
    if ((long long)nr * nz > (1ll << 31) - 1) { set_err("grid too large"); return nullptr; }
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { set_err("no CUDA device: %s", cudaGetErrorString(cudaGetLastError())); return nullptr; }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) { set_err("cudaGetDeviceProperties failed"); return nullptr; }
    if (prop.major != 10) {
        set_err("device %d is sm_%d%d; this library is built for sm_100a only (no fallback)", dev, prop.major, prop.minor);
        return nullptr;
    }
    sn_poisson* h = new (std::nothrow) sn_poisson();
    if (!h) { set_err("out of host memory"); return nullptr; }
    h->nr = nr; h->nz = nz; h->dr = dr; h->dz = dz; h->symmetry = symmetry; h->lmax = lmax;
    h->device = dev;
    h->num_sms = prop.multiProcessorCount;
    h->L0 = nr * dr;
    h->NL = lmax <= 8 ? 9 : lmax <= 16 ? 17 : lmax <= 32 ? 33 : 65;
    const size_t ncell = (size_t)nr * nz;
    size_t blocks = (ncell + kMomThreads * 4 - 1) / (kMomThreads * 4);
    const size_t cap = (size_t)h->num_sms * 4;
    h->mom_blocks = (int)(blocks < 1 ? 1 : blocks > cap ? cap : blocks);
    h->omega = default_omega(nr, nz, dr, dz, symmetry);
    // coefficient tables (R10): cE_i = ((i+1)/(i+1/2))/dr^2, cW_i = (i/(i+1/2))/dr^2
    std::vector<double> cE(nr), cW(nr);
    const double ir2 = 1.0 / (dr * dr);
    for (int i = 0; i < nr; ++i) {
        cE[i] = ((i + 1.0) / (i + 0.5)) * ir2;
        cW[i] = (i / (i + 0.5)) * ir2;
    }
    bool ok = cudaMalloc((void**)&h->d_cE, sizeof(double) * nr) == cudaSuccess &&
              cudaMalloc((void**)&h->d_cW, sizeof(double) * nr) == cudaSuccess &&
              cudaMemcpy(h->d_cE, cE.data(), sizeof(double) * nr, cudaMemcpyHostToDevice) == cudaSuccess &&
              cudaMemcpy(h->d_cW, cW.data(), sizeof(double) * nr, cudaMemcpyHostToDevice) == cudaSuccess;
    for (int i = 0; i < 2 && ok; ++i) ok = cudaEventCreateWithFlags(&h->ev_poll[i], cudaEventDisableTiming) == cudaSuccess;
    for (int i = 0; i < 3 && ok; ++i) ok = cudaEventCreate(&h->ev_t[i]) == cudaSuccess;
    if (!ok) {
        set_err("CUDA allocation failed: %s", cudaGetErrorString(cudaGetLastError()));
        sn_poisson_destroy(h);
        return nullptr;
    }
    return h;
}

void sn_poisson_destroy(sn_poisson* h) {
    if (!h) return;
    for (auto& v : {&h->mg.cE, &h->mg.cW, &h->mg.phi, &h->mg.f})
        for (double* p : *v) cudaFree(p);
    cudaFree(h->mg.slots);
    cudaFree(h->mg.d_ptrs);
    if (h->mg.exec) { cudaGraphExecDestroy(h->mg.exec); h->mg.exec = nullptr; }
    if (h->mg.st) cudaStreamDestroy(h->mg.st);
    if (h->mg.h_hist) cudaFreeHost(h->mg.h_hist);
    free_batch_ws(h);
    cudaFree(h->d_cE); cudaFree(h->d_cW);
    cudaFree(h->d_rho_stage); cudaFree(h->d_phi_stage); cudaFree(h->d_snap[0]); cudaFree(h->d_snap[1]);
    if (h->st_copy) cudaStreamDestroy(h->st_copy);
    for (auto& e : h->ev_io) if (e) cudaEventDestroy(e);
    cudaFree(h->d_prof); cudaFree(h->d_ring); cudaFree(h->d_mail); cudaFree(h->d_sync); cudaFree(h->d_work);
    for (auto& e : h->ev_poll) if (e) cudaEventDestroy(e);
    for (auto& e : h->ev_t) if (e) cudaEventDestroy(e);
    delete h;
}

sn_poisson_result sn_poisson_solve(sn_poisson* h, const double* rho, double* phi_inout, double tol, int max_sweeps,
                                   void* stream) {
    g_err.clear();
    sn_poisson_result r = {0, -1, 0.0};
    if (!check_solve_args(h, rho, phi_inout, tol, max_sweeps)) return r;
    const int rc = solve_impl(h, 1, rho, phi_inout, tol, max_sweeps, (cudaStream_t)stream, &r);
    if (rc) { r.sweeps = 0; r.status = rc; r.residual = 0.0; }
    return r;
}

int sn_poisson_solve_batch(sn_poisson* h, int nbatch, const double* rho, double* phi_inout, double tol,
                           int max_sweeps, void* stream, sn_poisson_result* out) {
    g_err.clear();
    if (nbatch < 1 || !out) { set_err("nbatch < 1 or NULL out"); return -1; }
    if (nbatch > 65535) { set_err("nbatch > 65535"); return -1; }
    if (!check_solve_args(h, rho, phi_inout, tol, max_sweeps, nbatch)) return -1;
    return solve_impl(h, nbatch, rho, phi_inout, tol, max_sweeps, (cudaStream_t)stream, out);
}

sn_poisson_result sn_poisson_solve_host(sn_poisson* h, const double* rho_host, double* phi_inout_host, double tol,
                                        int max_sweeps, void* stream) {
    g_err.clear();
    sn_poisson_result r = {0, -1, 0.0};
    if (!check_solve_args(h, rho_host, phi_inout_host, tol, max_sweeps)) return r;
    sn_poisson_result out;
    const int rc = sn_poisson_solve_batch_host(h, 1, rho_host, phi_inout_host, tol, max_sweeps, stream, &out);
    if (rc) { r.sweeps = 0; r.status = rc; r.residual = 0.0; return r; }
    return out;
}

sn_poisson_result sn_poisson_solve_mg(sn_poisson* h, const double* rho, double* phi_inout, double tol, int max_cycles,
                                      void* stream) {
    g_err.clear();
    sn_poisson_result r = {0, -1, 0.0};
    if (!check_solve_args(h, rho, phi_inout, tol, max_cycles)) return r;
    sn_poisson_result out = {0, 0, 0.0};
    const int rc = solve_mg_impl(h, 1, rho, phi_inout, tol, max_cycles, (cudaStream_t)stream, &out);
    if (rc) { r.status = rc; return r; }
    return out;
}

int sn_poisson_solve_mg_batch(sn_poisson* h, int nbatch, const double* rho, double* phi_inout, double tol, int max_cycles,
                              void* stream, sn_poisson_result* out) {
    g_err.clear();
    if (nbatch < 1 || !out) { set_err("nbatch < 1 or NULL out"); return -1; }
    if (nbatch > 65535) { set_err("nbatch > 65535"); return -1; }
    if (!check_solve_args(h, rho, phi_inout, tol, max_cycles, nbatch)) return -1;
    return solve_mg_impl(h, nbatch, rho, phi_inout, tol, max_cycles, (cudaStream_t)stream, out);
}

int sn_poisson_solve_mg_batch_host(sn_poisson* h, int nbatch, const double* rho_host, double* phi_inout_host, double tol,
                                   int max_cycles, void* stream, sn_poisson_result* out) {
    g_err.clear();
    if (nbatch < 1 || !out) { set_err("nbatch < 1 or NULL out"); return -1; }
    if (nbatch > 65535) { set_err("nbatch > 65535"); return -1; }
    if (!check_solve_args(h, rho_host, phi_inout_host, tol, max_cycles, nbatch)) return -1;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)h->nr * h->nz * nbatch, bytes = sizeof(double) * n;
    CU_TRY(cudaSetDevice(h->device));
    if (int rc = ensure_stage(h, n)) return rc;
    // rho on the caller's stream (the moments need it first), phi on the copy stream behind the moment / boundary
    // kernels, waited for just before the first cycle; phi's download behind the last cycle, before the one sync
    auto upload = [&]() -> int {
        CU_TRY(cudaEventRecord(h->ev_io[0], st));
        CU_TRY(cudaStreamWaitEvent(h->st_copy, h->ev_io[0], 0));
        CU_TRY(cudaMemcpyAsync(h->d_rho_stage, rho_host, bytes, cudaMemcpyHostToDevice, st));
        CU_TRY(cudaMemcpyAsync(h->d_phi_stage, phi_inout_host, bytes, cudaMemcpyHostToDevice, h->st_copy));
        CU_TRY(cudaEventRecord(h->ev_io[1], h->st_copy));
        return 0;
    };
    int rc = upload();
    if (rc == 0) {
        HostIO io;
        io.wait_before_relax = h->ev_io[1];
        io.d2h_dst = phi_inout_host; io.d2h_src = h->d_phi_stage; io.d2h_bytes = bytes;
        rc = solve_mg_impl(h, nbatch, h->d_rho_stage, h->d_phi_stage, tol, max_cycles, st, out, &io);
    }
    if (rc) drain_host_io(h, st);        // a failed call may have left the uploads in flight: not past the return
    return rc;
}

sn_poisson_result sn_poisson_solve_mg_host(sn_poisson* h, const double* rho_host, double* phi_inout_host, double tol,
                                           int max_cycles, void* stream) {
    g_err.clear();
    sn_poisson_result r = {0, -1, 0.0};
    if (!check_solve_args(h, rho_host, phi_inout_host, tol, max_cycles)) return r;
    sn_poisson_result out = {0, 0, 0.0};
    const int rc = sn_poisson_solve_mg_batch_host(h, 1, rho_host, phi_inout_host, tol, max_cycles, stream, &out);
    if (rc) { r.status = rc; return r; }
    return out;
}

int sn_poisson_solve_batch_host(sn_poisson* h, int nbatch, const double* rho_host, double* phi_inout_host, double tol,
                                int max_sweeps, void* stream, sn_poisson_result* out) {
    g_err.clear();
    if (nbatch < 1 || !out) { set_err("nbatch < 1 or NULL out"); return -1; }
    if (nbatch > 65535) { set_err("nbatch > 65535"); return -1; }
    if (!check_solve_args(h, rho_host, phi_inout_host, tol, max_sweeps, nbatch)) return -1;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)h->nr * h->nz * nbatch, bytes = sizeof(double) * n;
    CU_TRY(cudaSetDevice(h->device));
    if (int rc = ensure_stage(h, n)) return rc;
    // rho goes first on the caller's stream (the moments need it); phi's upload rides on the copy stream behind the
    // moments / boundary kernels and is waited for just before the relaxation; phi's download is enqueued right
    // after the relaxation, before the call's single synchronisation.
    CU_TRY(cudaEventRecord(h->ev_io[0], st));                          // order the copy stream after the caller's work
    CU_TRY(cudaStreamWaitEvent(h->st_copy, h->ev_io[0], 0));
    CU_TRY(cudaMemcpyAsync(h->d_rho_stage, rho_host, bytes, cudaMemcpyHostToDevice, st));
    CU_TRY(cudaMemcpyAsync(h->d_phi_stage, phi_inout_host, bytes, cudaMemcpyHostToDevice, h->st_copy));
    CU_TRY(cudaEventRecord(h->ev_io[1], h->st_copy));
    HostIO io;
    io.wait_before_relax = h->ev_io[1];
    io.d2h_dst = phi_inout_host; io.d2h_src = h->d_phi_stage; io.d2h_bytes = bytes;
    const int rc = solve_impl(h, nbatch, h->d_rho_stage, h->d_phi_stage, tol, max_sweeps, st, out, &io);
    if (rc) drain_host_io(h, st);        // a failed call may have left the uploads in flight: not past the return
    return rc;
}

int sn_poisson_solve_sequence_host(sn_poisson* h, int nsteps, const double* rho_seq_host, double* phi_inout_host,
                                   double* phi_seq_host, double tol, int max_sweeps, void* stream,
                                   sn_poisson_result* out) {
    g_err.clear();
    if (nsteps < 1 || !out) { set_err("nsteps < 1 or NULL out"); return -1; }
    if (!check_solve_args(h, rho_seq_host, phi_inout_host, tol, max_sweeps)) return -1;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)h->nr * h->nz, bytes = sizeof(double) * n;
    CU_TRY(cudaSetDevice(h->device));
    if (int rc = ensure_stage(h, 2 * n)) return rc;                    // rho double-buffered in d_rho_stage[2][n]
    if (phi_seq_host && h->snap_cap < n) {
        for (auto& d : h->d_snap) { cudaFree(d); d = nullptr; }
        h->snap_cap = 0;
        for (auto& d : h->d_snap) CU_TRY(cudaMalloc((void**)&d, bytes));
        h->snap_cap = n;
    }
    cudaEvent_t ev_h2d[2] = {h->ev_io[0], h->ev_io[1]}, ev_snap[2] = {h->ev_io[2], h->ev_io[3]},
                ev_d2h[2] = {h->ev_io[4], h->ev_io[5]};
    // Everything that touches the caller's host buffers is enqueued inside `run`; whatever way it ends (all steps, a
    // failed step, a CUDA error), the tail below drains both streams before the call returns, so no DMA is still
    // reading rho_seq_host or writing phi_seq_host / phi_inout_host when the caller gets control back.
    auto run = [&]() -> int {
    CU_TRY(cudaMemcpyAsync(h->d_rho_stage, rho_seq_host, bytes, cudaMemcpyHostToDevice, st));
    CU_TRY(cudaMemcpyAsync(h->d_phi_stage, phi_inout_host, bytes, cudaMemcpyHostToDevice, st));
    CU_TRY(cudaEventRecord(ev_h2d[0], st));
    CU_TRY(cudaStreamWaitEvent(h->st_copy, ev_h2d[0], 0));             // the copy stream starts behind the caller's work
    bool d2h_pending[2] = {false, false};
    for (int t = 0; t < nsteps; ++t) {
        const int cur = t & 1, nxt = cur ^ 1;
        // upload rho_{t+1} on the copy stream while solve t runs (its buffer was last read by solve t-1: complete,
        // every solve ends with a stream synchronisation)
        if (t + 1 < nsteps) {
            CU_TRY(cudaMemcpyAsync(h->d_rho_stage + (size_t)nxt * n, rho_seq_host + (size_t)(t + 1) * n, bytes,
                                   cudaMemcpyHostToDevice, h->st_copy));
            CU_TRY(cudaEventRecord(ev_h2d[nxt], h->st_copy));
        }
        if (t > 0) CU_TRY(cudaStreamWaitEvent(st, ev_h2d[cur], 0));
        if (int rc = solve_impl(h, 1, h->d_rho_stage + (size_t)cur * n, h->d_phi_stage, tol, max_sweeps, st, out + t)) return rc;
        if (out[t].status < 0) break;                                   // the caller sees which step failed
        if (phi_seq_host) {
            // snapshot on the caller's stream (the next solve updates phi in place), download on the copy stream
            // while solve t+1 runs
            if (d2h_pending[cur]) CU_TRY(cudaStreamWaitEvent(st, ev_d2h[cur], 0));
            CU_TRY(cudaMemcpyAsync(h->d_snap[cur], h->d_phi_stage, bytes, cudaMemcpyDeviceToDevice, st));
            CU_TRY(cudaEventRecord(ev_snap[cur], st));
            CU_TRY(cudaStreamWaitEvent(h->st_copy, ev_snap[cur], 0));
            CU_TRY(cudaMemcpyAsync(phi_seq_host + (size_t)t * n, h->d_snap[cur], bytes, cudaMemcpyDeviceToHost, h->st_copy));
            CU_TRY(cudaEventRecord(ev_d2h[cur], h->st_copy));
            d2h_pending[cur] = true;
        }
    }
    // after the last step -- or after a failed one: phi as the device holds it, like sn_poisson_solve leaves it
    CU_TRY(cudaMemcpyAsync(phi_inout_host, h->d_phi_stage, bytes, cudaMemcpyDeviceToHost, st));
    return 0;
    };
    int rc = run();
    const cudaError_t e1 = cudaStreamSynchronize(st), e2 = cudaStreamSynchronize(h->st_copy);
    if (rc == 0 && (e1 != cudaSuccess || e2 != cudaSuccess)) {
        set_err("stream synchronisation failed: %s", cudaGetErrorString(e1 != cudaSuccess ? e1 : e2));
        rc = -2;
    }
    return rc;
}

int sn_poisson_solve_gravity(sn_poisson* h, int nbatch, const double* rho, double* phi_inout, double* gr, double* gz,
                             double tol, int max_sweeps, void* stream, sn_poisson_result* out) {
    g_err.clear();
    if (nbatch < 1 || !out) { set_err("nbatch < 1 or NULL out"); return -1; }
    if (nbatch > 65535) { set_err("nbatch > 65535"); return -1; }
    if (!gr || !gz) { set_err("NULL gr / gz pointer"); return -1; }
    if (gr == phi_inout || gz == phi_inout || gr == gz) { set_err("gr, gz and phi must not alias"); return -1; }
    if (!check_solve_args(h, rho, phi_inout, tol, max_sweeps, nbatch)) return -1;
    HostIO io;
    io.gr = gr; io.gz = gz;
    return solve_impl(h, nbatch, rho, phi_inout, tol, max_sweeps, (cudaStream_t)stream, out, &io);
}

int sn_poisson_gravity(sn_poisson* h, int nbatch, const double* phi, double* gr, double* gz, void* stream) {
    g_err.clear();
    if (!h || !phi || !gr || !gz) { set_err("NULL argument"); return -1; }
    if (nbatch < 1 || nbatch > 65535) { set_err("nbatch must be in [1, 65535]"); return -1; }
    if (!h->d_bE || nbatch > h->last_nbatch) {
        set_err("no ghost values for %d member(s): the last solve / set_boundary on this handle covered %d", nbatch,
                h->d_bE ? h->last_nbatch : 0);
        return -1;
    }
    CU_TRY(cudaSetDevice(h->device));
    const Geom g = make_geom(h, 0.0);
    cudaStream_t st = (cudaStream_t)stream;
    return launch_gravity(h, g, nbatch, phi, gr, gz, st);
}

int sn_poisson_probe_l2(int mib, double* copy_gbs, double* read_gbs, void* stream) {
    g_err.clear();
    if (mib < 1 || mib > 1024 || !copy_gbs || !read_gbs) { set_err("bad argument"); return -1; }
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    CU_TRY(cudaGetDevice(&dev));
    CU_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const size_t n2 = (size_t)mib * (1u << 20) / 16;                   // double2 elements per array
    const int grid = 2 * sms, reps = 20;
    double2 *a = nullptr, *b = nullptr;
    double* sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = 0;
    auto body = [&]() -> int {
        CU_TRY(cudaMalloc((void**)&a, 16 * n2));
        CU_TRY(cudaMalloc((void**)&b, 16 * n2));
        CU_TRY(cudaMalloc((void**)&sink, sizeof(double) * grid * kProbeThreads));
        CU_TRY(cudaMemsetAsync(a, 0, 16 * n2, st));
        CU_TRY(cudaEventCreate(&e0));
        CU_TRY(cudaEventCreate(&e1));
        double best_c = 0, best_r = 0;
        for (int it = 0; it < 6; ++it) {                               // first pass of each kind warms L2 and clocks
            float ms = 0;
            CU_TRY(cudaEventRecord(e0, st));
            k_probe_l2_copy<<<grid, kProbeThreads, 0, st>>>(a, b, n2, reps);
            CU_TRY(cudaEventRecord(e1, st));
            CU_TRY(cudaEventSynchronize(e1));
            CU_TRY(cudaEventElapsedTime(&ms, e0, e1));
            if (it > 0) best_c = std::max(best_c, 2.0 * 16.0 * n2 * reps / (ms * 1e-3) / 1e9);
            CU_TRY(cudaEventRecord(e0, st));
            k_probe_l2_read<<<grid, kProbeThreads, 0, st>>>(a, n2, reps, sink);
            CU_TRY(cudaEventRecord(e1, st));
            CU_TRY(cudaEventSynchronize(e1));
            CU_TRY(cudaEventElapsedTime(&ms, e0, e1));
            if (it > 0) best_r = std::max(best_r, 16.0 * n2 * reps / (ms * 1e-3) / 1e9);
        }
        CU_TRY(cudaGetLastError());
        *copy_gbs = best_c;
        *read_gbs = best_r;
        return 0;
    };
    rc = body();
    cudaFree(a); cudaFree(b); cudaFree(sink);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    return rc;
}

int sn_poisson_set_stop_rule(sn_poisson* h, int rule) {
    g_err.clear();
    if (!h) { set_err("NULL handle"); return -1; }
    if (rule != 0 && rule != 1) { set_err("rule must be 0 (residual ratio) or 1 (relative change)"); return -1; }
    h->opt_rule = rule;
    return 0;
}

int sn_poisson_set_omega(sn_poisson* h, double omega) {
    g_err.clear();
    if (!h) { set_err("NULL handle"); return -1; }
    if (!(omega > 0)) {
        h->omega_user = false;
        h->omega = default_omega(h->nr, h->nz, h->dr, h->dz, h->symmetry);
        return 0;
    }
    if (!(omega < 2.0)) { set_err("omega must be in (0, 2)"); return -1; }
    h->omega = omega;
    h->omega_user = true;
    return 0;
}

double sn_poisson_get_omega(const sn_poisson* h) { return h ? h->omega : 0.0; }

int sn_poisson_get_moments(sn_poisson* h, double* M) {
    g_err.clear();
    if (!h || !M) { set_err("NULL argument"); return -1; }
    if (!h->d_M) { set_err("no solve has run yet"); return -1; }
    CU_TRY(cudaMemcpy(M, h->d_M, sizeof(double) * (h->lmax + 1), cudaMemcpyDeviceToHost));
    return 0;
}

int sn_poisson_set_boundary(sn_poisson* h, const double* bE, const double* bN, const double* bS) {
    g_err.clear();
    if (!h) { set_err("NULL handle"); return -1; }
    if (!bE && !bN && !bS) { h->user_boundary = false; return 0; }
    if (!bE || !bN || (h->symmetry == 0 && !bS)) { set_err("NULL boundary array"); return -1; }
    if (int rc = ensure_ws(h, 1, 1)) return rc;
    for (int b = 0; b < h->cap_batch; ++b) {
        CU_TRY(cudaMemcpy(h->d_bE + (size_t)b * h->nz, bE, sizeof(double) * h->nz, cudaMemcpyHostToDevice));
        CU_TRY(cudaMemcpy(h->d_bN + (size_t)b * h->nr, bN, sizeof(double) * h->nr, cudaMemcpyHostToDevice));
        if (h->symmetry == 0)
            CU_TRY(cudaMemcpy(h->d_bS + (size_t)b * h->nr, bS, sizeof(double) * h->nr, cudaMemcpyHostToDevice));
    }
    h->user_boundary = true;
    h->last_nbatch = h->cap_batch;
    return 0;
}

int sn_poisson_get_boundary(sn_poisson* h, double* bE, double* bN, double* bS) {
    g_err.clear();
    if (!h || !bE || !bN) { set_err("NULL argument"); return -1; }
    if (!h->d_bE) { set_err("no solve has run yet"); return -1; }
    CU_TRY(cudaMemcpy(bE, h->d_bE, sizeof(double) * h->nz, cudaMemcpyDeviceToHost));
    CU_TRY(cudaMemcpy(bN, h->d_bN, sizeof(double) * h->nr, cudaMemcpyDeviceToHost));
    if (bS && h->symmetry == 0) CU_TRY(cudaMemcpy(bS, h->d_bS, sizeof(double) * h->nr, cudaMemcpyDeviceToHost));
    return 0;
}

int sn_poisson_get_history(sn_poisson* h, double* R, int n) {
    g_err.clear();
    if (!h || !R || n < 0) { set_err("bad argument"); return -1; }
    if (!h->d_hist) { set_err("no solve has run yet"); return -1; }
    const int m = n < h->last_sweeps0 ? n : h->last_sweeps0;
    if (m > 0) CU_TRY(cudaMemcpy(R, h->d_hist, sizeof(double) * m, cudaMemcpyDeviceToHost));
    return m;
}

int sn_poisson_set_option(sn_poisson* h, const char* key, int64_t value) {
    g_err.clear();
    if (!h || !key) { set_err("NULL argument"); return -1; }
    h->plan_cache.valid = false;
    if (!strcmp(key, "path")) { if (value < 0 || value > 3) { set_err("path must be 0..3"); return -1; } h->opt_path = (int)value; return 0; }
    if (!strcmp(key, "chunk")) { if (value < 1) { set_err("chunk must be >= 1"); return -1; } h->opt_chunk = (int)value; return 0; }
    if (!strcmp(key, "exact")) { h->opt_exact = value ? 1 : 0; return 0; }
    if (!strcmp(key, "prof")) { h->opt_prof = value ? 1 : 0; return 0; }
    if (!strcmp(key, "ring")) { if (value < -1 || value > 1) { set_err("ring must be -1, 0 or 1"); return -1; } h->opt_ring = (int)value; return 0; }
    if (!strcmp(key, "ds")) { if (value < -1 || value > 1) { set_err("ds must be -1, 0 or 1"); return -1; } h->opt_ds = (int)value; return 0; }
    if (!strcmp(key, "group")) { if (value < -1 || value > 65535) { set_err("group must be -1, 0 or a member count"); return -1; } h->opt_group = (int)value; return 0; }
    if (!strcmp(key, "ll")) { if (value < -1 || value > 1) { set_err("ll must be -1, 0 or 1"); return -1; } h->opt_ll = (int)value; return 0; }
    if (!strcmp(key, "halo")) { if (value < -1 || value > 1) { set_err("halo must be -1, 0 or 1"); return -1; } h->opt_halo = (int)value; return 0; }
    if (!strcmp(key, "shape")) { if (value < -1 || value >= (int64_t)std::max(shapes().size(), blk_shapes().size())) { set_err("bad shape"); return -1; } h->opt_shape = (int)value; return 0; }
    if (!strcmp(key, "mg_nu1")) { if (value < 0 || value > 8) { set_err("mg_nu1 must be 0..8"); return -1; } h->opt_mg_nu1 = (int)value; return 0; }
    if (!strcmp(key, "mg_nu2")) { if (value < 0 || value > 8) { set_err("mg_nu2 must be 0..8"); return -1; } h->opt_mg_nu2 = (int)value; return 0; }
    if (!strcmp(key, "mg_graph")) { h->opt_mg_graph = value ? 1 : 0; return 0; }
    if (!strcmp(key, "mg_nc")) { if (value < 1 || value > 1000) { set_err("mg_nc must be 1..1000"); return -1; } h->opt_mg_nc = (int)value; return 0; }
    if (!strcmp(key, "tblock")) { if (value < 0 || value > kMaxTB) { set_err("tblock must be 0..%d", kMaxTB); return -1; } h->opt_tblock = (int)value; return 0; }
    set_err("unknown option '%s'", key);
    return -1;
}

int sn_poisson_get_stat(sn_poisson* h, const char* key, double* out) {
    g_err.clear();
    if (!h || !key || !out) { set_err("NULL argument"); return -1; }
    if (!strcmp(key, "launches")) { *out = h->st_launches; return 0; }
    if (!strcmp(key, "sweep_launches")) { *out = h->st_launches - h->st_aux_launches; return 0; }
    if (!strcmp(key, "sweep_ms")) { *out = h->st_sweep_ms; return 0; }
    if (!strcmp(key, "setup_ms")) { *out = h->st_setup_ms; return 0; }
    if (!strcmp(key, "path")) { *out = h->st_path; return 0; }
    if (!strcmp(key, "ctas")) { *out = h->st_ctas; return 0; }
    if (!strcmp(key, "tile_w")) { *out = h->st_tile_w; return 0; }
    if (!strcmp(key, "tile_h")) { *out = h->st_tile_h; return 0; }
    if (!strcmp(key, "tblock")) { *out = h->st_tblock; return 0; }
    if (!strcmp(key, "shape")) { *out = h->st_shape; return 0; }
    if (!strcmp(key, "halo")) { *out = h->st_halo; return 0; }
    if (!strcmp(key, "ds")) { *out = h->st_ds; return 0; }
    if (!strcmp(key, "ring")) { *out = h->st_ring; return 0; }
    if (!strcmp(key, "group")) { *out = h->st_group; return 0; }
    if (!strcmp(key, "redundancy")) { *out = h->st_redund; return 0; }
    if (!strcmp(key, "mg_levels")) { *out = h->mg.nlev; return 0; }
    if (!strncmp(key, "prof_mean", 9) && key[9] >= '0' && key[9] <= '7' && !key[10]) { *out = h->prof_mean[key[9] - '0']; return 0; }
    if (!strncmp(key, "prof_max", 8) && key[8] >= '0' && key[8] <= '7' && !key[9]) { *out = h->prof_max[key[8] - '0']; return 0; }
    set_err("unknown stat '%s'", key);
    return -1;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// sn_poisson_moments_static: the multipole moments (step a-1) for callers that must not allocate device memory.
//
// k_moments reduces in two stages and needs global scratch between them: one row of NL partial sums per block, plus a
// per-member Ctl block whose `maxf` word collects max|4 pi rho| by atomicMax.  Everywhere else in this library that
// scratch comes from cudaMalloc inside a handle.  Here it is a fixed array that is part of the loaded module instead,
// so the entry point below needs no handle and makes no allocating call of any kind.
//
// The array exists once per GPU that loads this library and stays until the process exits (kStaticBytes = 520 KiB each).
// All calls on one GPU share it.  Layout: [0, kStaticCtlBytes) = Ctl[kStaticMaxBatch]; then kStaticPartialDoubles doubles.
// ---------------------------------------------------------------------------------------------------------------------
namespace {

constexpr int kStaticMaxBatch = SN_POISSON_STATIC_MAX_BATCH;
constexpr size_t kStaticCtlBytes = 8192;
constexpr size_t kStaticPartialDoubles = SN_POISSON_STATIC_MAX_DOUBLES;
constexpr size_t kStaticBytes = kStaticCtlBytes + kStaticPartialDoubles * sizeof(double);
static_assert(sizeof(Ctl) * kStaticMaxBatch <= kStaticCtlBytes, "Ctl area of the static scratch too small");
static_assert(kStaticCtlBytes % 256 == 0, "partials must stay 256-byte aligned");

static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];

// In host code `g_static_scratch` is only a stand-in the runtime uses to look the array up; it is NOT a device address
// and must never be handed to a kernel or a memset.  The real address differs per GPU and is fetched once per device,
// with that device current, by cudaGetSymbolAddress below.
constexpr int kStaticMaxDevices = 64;
struct StaticDev {
    bool ready = false;
    unsigned char* base = nullptr;   // device address of g_static_scratch on this GPU
    int num_sms = 0;
};
std::mutex g_static_mu;
StaticDev g_static_dev[kStaticMaxDevices];

// Second stage: fixed-order sum of the block partials (the order k_boundary uses, so the bits agree with the handle
// path when the block count is the same), symmetry rule, result straight into the caller's arrays.  grid = nbatch.
__global__ void __launch_bounds__(128) k_moments_static_finish(int lmax, int symmetry, int NL, int nblocks,
                                                               const double* __restrict__ partial,
                                                               const Ctl* __restrict__ ctl, double* __restrict__ M_out,
                                                               double* __restrict__ maxf_out) {
    const int b = blockIdx.x;
    for (int l = threadIdx.x; l <= lmax; l += blockDim.x) {
        double v = 0.0;
        for (int k = 0; k < nblocks; ++k) v += partial[((size_t)b * nblocks + k) * NL + l];
        if (symmetry == 1) v = (l & 1) ? 0.0 : 2.0 * v;
        M_out[(size_t)b * (lmax + 1) + l] = v;
    }
    if (maxf_out && threadIdx.x == 0) maxf_out[b] = ctl[b].maxf;
}

// One-time set-up of the current device: architecture check, SM count, device address of the scratch array.
int static_setup(StaticDev** out) {
    int dev = 0;
    CU_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) { set_err("device ordinal %d outside [0, %d)", dev, kStaticMaxDevices); return -1; }
    std::lock_guard<std::mutex> lock(g_static_mu);
    StaticDev& d = g_static_dev[dev];
    if (!d.ready) {
        int major = 0, sms = 0;
        CU_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        CU_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        if (major != 10) { set_err("device %d is not sm_10x; this library is built for sm_100a only (no fallback)", dev); return -1; }
        unsigned char* base = nullptr;
        CU_TRY(cudaGetSymbolAddress((void**)&base, g_static_scratch));
        if (!base) { set_err("cudaGetSymbolAddress returned a NULL address"); return -2; }
        d.base = base;
        d.num_sms = sms;
        d.ready = true;
    }
    *out = &d;
    return 0;
}

}  // namespace

extern "C" int sn_poisson_moments_static(const double* rho, int nbatch, int nr, int nz, double dr, double dz,
                                         int symmetry, int lmax, double* M_out, double* maxf_out, void* stream) {
    g_err.clear();
    if (!rho || !M_out) { set_err("NULL argument"); return -1; }
    if (nr < 2 || nz < 2) { set_err("nr, nz must be >= 2"); return -1; }
    if (!(dr > 0) || !(dz > 0) || !std::isfinite(dr) || !std::isfinite(dz)) { set_err("dr, dz must be finite and > 0"); return -1; }
    if (symmetry != 0 && symmetry != 1) { set_err("symmetry must be 0 or 1"); return -1; }
    if (lmax < 0 || lmax > kMaxL) { set_err("lmax must be in [0, %d]", kMaxL); return -1; }
    if ((long long)nr * nz > (1ll << 31) - 1) { set_err("grid too large"); return -1; }
    if (nbatch < 1 || nbatch > kStaticMaxBatch) {
        set_err("nbatch = %d: the static scratch holds control blocks for 1..%d members", nbatch, kStaticMaxBatch);
        return -1;
    }
    StaticDev* d = nullptr;
    if (int rc = static_setup(&d)) return rc;
    // same template choice and block count as a handle makes in sn_poisson_create, so both paths sum in the same order
    const int NL = lmax <= 8 ? 9 : lmax <= 16 ? 17 : lmax <= 32 ? 33 : 65;
    const size_t ncell = (size_t)nr * nz;
    size_t blocks = (ncell + kMomThreads * 4 - 1) / (kMomThreads * 4);
    const size_t cap = (size_t)d->num_sms * 4;
    blocks = blocks < 1 ? 1 : blocks > cap ? cap : blocks;
    const size_t need = (size_t)nbatch * blocks * NL;
    if (need > kStaticPartialDoubles) {
        set_err("this call needs %zu doubles of scratch (nbatch %d x %zu blocks x %d sums); the static area holds %zu -- "
                "use fewer members per call, or a handle (sn_poisson_create), which allocates what it needs",
                need, nbatch, blocks, NL, kStaticPartialDoubles);
        return -1;
    }
    cudaStream_t st = (cudaStream_t)stream;
    Ctl* ctl = reinterpret_cast<Ctl*>(d->base);
    double* partial = reinterpret_cast<double*>(d->base + kStaticCtlBytes);
    // The array keeps whatever the previous call left.  The partials are overwritten in full by every launch (each
    // block stores all NL of its sums), but `maxf` is accumulated with atomicMax and has to start from zero.
    CU_TRY(cudaMemsetAsync(ctl, 0, sizeof(Ctl) * nbatch, st));
    Geom g{};
    g.nr = nr; g.nz = nz; g.symmetry = symmetry; g.lmax = lmax; g.dr = dr; g.dz = dz;
    const double L0 = nr * dr;
    dim3 grid((unsigned)blocks, nbatch);
    switch (NL) {
        case 9: k_moments<9><<<grid, kMomThreads, 0, st>>>(rho, g, L0, partial, ctl); break;
        case 17: k_moments<17><<<grid, kMomThreads, 0, st>>>(rho, g, L0, partial, ctl); break;
        case 33: k_moments<33><<<grid, kMomThreads, 0, st>>>(rho, g, L0, partial, ctl); break;
        default: k_moments<65><<<grid, kMomThreads, 0, st>>>(rho, g, L0, partial, ctl); break;
    }
    CU_TRY(cudaGetLastError());
    k_moments_static_finish<<<nbatch, 128, 0, st>>>(lmax, symmetry, NL, (int)blocks, partial, ctl, M_out, maxf_out);
    CU_TRY(cudaGetLastError());
    return 0;
}
