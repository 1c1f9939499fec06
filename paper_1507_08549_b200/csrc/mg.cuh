// mg.cuh -- red-black-smoothed geometric multigrid variant of the Poisson solve (not in
// the paper, which relaxes the same equation by SOR).  Same discretisation, ghosts and fixed point as the
// SOR path; the iteration is the textbook V-cycle on cell-centred grids, readings M1..M8 of
// rediscretised coarse operators whose outer Dirichlet ghost is -beta_l x (adjacent value) so
// that the zero of the error stays at the level-0 ghost centre (M2), red-black Gauss-Seidel smoothing with the pinned
// update of R10 at omega = 1 (M3), volume-weighted restriction (M5), bilinear prolongation (M7), the ratio of R9 on
// the true residual after every cycle (M8).  Every kernel is a plain streaming kernel (the coarse levels are tiny and
// launch bound; the fine levels are L2 / HBM bound at 24-40 B per cell and pass); the coarsest level is solved by one
// CTA.  All arithmetic is pinned like the SOR path, so the iterates are reproducible bit for bit by any implementation of M1-M8 that keeps the expression trees.
#pragma once
#include "box_engine.cuh"      // warp_max_key
#include "common.cuh"

namespace snp {

struct MgLevel {
    int nr, nz, symmetry;
    double iz2, D, D0, wD, wD0;     // wD = 1 / D, wD0 = 1 / D0  (omega = 1)
    double beta;                    // M2: outer ghost = -beta * adjacent value (0 on level 0, which has real ghosts)
    double scale;                   // f = scale * src: 4 pi on level 0 (src = rho), 1 on coarse levels (src = restricted residual)
    const double* cE;               // [nr]
    const double* cW;               // [nr]
    double* phi;                    // level 0: the caller's phi; coarse: the error
    const double* src;
    const double *bE, *bN, *bS;     // level 0: multipole ghosts; coarse: NULL
};

// The caller's arrays of the current solve.  Level 0 reaches them through this device-side record (phi == NULL in its
// MgLevel), so that a captured cycle (CUDA graph) stays valid when the next solve brings other pointers.
struct MgPtrs {
    const double* rho;
    double* phi;
};
// Batches: member m of a batch works on the m-th slice of every array (the members' slices are contiguous).
__device__ __forceinline__ MgLevel mg_resolve(MgLevel L, const MgPtrs* __restrict__ pp, int member = 0) {
    if (L.phi == nullptr) { L.phi = pp->phi; L.src = pp->rho; }
    const size_t off = (size_t)member * L.nr * L.nz;
    L.phi += off;
    L.src += off;
    if (L.bE) {
        L.bE += (size_t)member * L.nz;
        L.bN += (size_t)member * L.nr;
        if (L.bS) L.bS += (size_t)member * L.nr;
    }
    return L;
}

// t = (A phi)(i, j) with the pinned tree (R10); ghosts per M2.  Also returns the row's diagonal and omega / diag.
__device__ __forceinline__ double mg_apply_at(const MgLevel& L, int i, int j, double pC, double& diag, double& w) {
    const size_t c = (size_t)j * L.nr + i;
    const bool mirror_row = L.symmetry == 1 && j == 0;
    const double cS = mirror_row ? 0.0 : L.iz2;
    diag = mirror_row ? L.D0 : L.D;
    w = mirror_row ? L.wD0 : L.wD;
    const double ghost = -__dmul_rn(L.beta, pC);
    // the four neighbours are fetched UNCONDITIONALLY from clamped (always valid) positions and selected afterwards: as
    // conditional loads the lanes of a boundary warp -- every warp of the small levels -- take them one branch after the
    // other, each with its own load latency (measured: a warp-wide update of a 4 x 4 level took 720 clocks)
    const int ie = i + 1 < L.nr ? 1 : 0, iw = i > 0 ? 1 : 0;
    const int jn = j + 1 < L.nz ? L.nr : 0, js = j > 0 ? L.nr : 0;
    const double vE = L.phi[c + ie], vW = L.phi[c - iw], vN = L.phi[c + jn], vS = L.phi[c - js];
    double gE = ghost, gN = ghost, gS = ghost;
    if (L.bE) {                                   // level 0: the multipole ghosts (uniform branch)
        if (!ie) gE = L.bE[j];
        if (!jn) gN = L.bN[i];
        if (!js && L.bS) gS = L.bS[i];
    }
    const double pE = ie ? vE : gE;
    const double pW = iw ? vW : 0.0;
    const double pN = jn ? vN : gN;
    const double pS = js ? vS : (L.symmetry == 1 ? 0.0 : gS);
    double t = __dmul_rn(L.cE[i], pE);
    t = __fma_rn(L.cW[i], pW, t);
    t = __fma_rn(L.iz2, pN, t);
    t = __fma_rn(cS, pS, t);
    t = __fma_rn(-diag, pC, t);
    return t;
}

// M3: the Gauss-Seidel update of the idx-th cell of colour col (cells of one colour are numbered row by row)
// (IDX: size_t in the streaming kernels, unsigned in the one-CTA tail, where a 64-bit division per cell would dominate)
template <typename IDX>
__device__ __forceinline__ void mg_update_cell(const MgLevel& L, IDX idx, int col) {
    const IDX half = (IDX)((L.nr + 1) / 2);
    const int j = (int)(idx / half), i = 2 * (int)(idx - (IDX)j * half) + ((j + col) & 1);
    if (i >= L.nr) return;
    const size_t c = (size_t)j * L.nr + i;
    const double pC = L.phi[c];
    double diag, w;
    const double t = mg_apply_at(L, i, j, pC, diag, w);
    const double res = __dsub_rn(__dmul_rn(L.scale, L.src[c]), t);
    L.phi[c] = __fma_rn(-w, res, pC);
}

// M3: one half-sweep of colour COL; one thread per cell of that colour
template <int COL, typename IDX>
__global__ void __launch_bounds__(256) k_mg_halfsweep(const MgLevel Larg, const Ctl* __restrict__ ctl,
                                                      const MgPtrs* __restrict__ pp) {
    if (ctl[blockIdx.y].done) return;    // a finished solve: cycles enqueued ahead of the host's poll do nothing
    const MgLevel L = mg_resolve(Larg, pp, blockIdx.y);
    const IDX n = (IDX)((L.nr + 1) / 2) * (IDX)L.nz;
    for (IDX idx = (IDX)blockIdx.x * blockDim.x + threadIdx.x; idx < n; idx += (IDX)gridDim.x * blockDim.x)
        mg_update_cell<IDX>(L, idx, COL);
}

// M4 + M5 + M8: one thread per 2 x 2 block of the level.  RESTRICT: the volume-weighted average of the four residuals
// becomes the right-hand side of the next coarser level, whose error is zeroed.  MAXIMA: max|res| and max|phi| of the
// level as order-preserving keys (warp REDUX, one atomicMax per warp) for the stopping ratio.
template <bool RESTRICT, bool MAXIMA, typename IDX>
__device__ __forceinline__ void mg_residual_block(const MgLevel& L, IDX idx, double* __restrict__ fc,
                                                  double* __restrict__ ec, unsigned long long& kr, unsigned long long& kp) {
    const IDX nrc = (IDX)((L.nr + 1) / 2);
    {
        const int J = (int)(idx / nrc), I = (int)(idx - (IDX)J * nrc);
        double r[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
#pragma unroll
        for (int b = 0; b < 2; ++b)
#pragma unroll
            for (int a = 0; a < 2; ++a) {
                const int i = 2 * I + a, j = 2 * J + b;
                if (i >= L.nr || j >= L.nz) continue;
                const size_t c = (size_t)j * L.nr + i;
                const double pC = L.phi[c];
                double diag, w;
                const double t = mg_apply_at(L, i, j, pC, diag, w);
                r[b][a] = __dsub_rn(__dmul_rn(L.scale, L.src[c]), t);
                if (MAXIMA) {
                    const unsigned long long a1 = abs_key(r[b][a]), a2 = abs_key(pC);
                    kr = a1 > kr ? a1 : kr;
                    kp = a2 > kp ? a2 : kp;
                }
            }
        if (RESTRICT) {
            const double ra = (2 * I) + 0.5, rb = (2 * I + 1) + 0.5;
            const double num = __dadd_rn(__dadd_rn(__dmul_rn(ra, r[0][0]), __dmul_rn(rb, r[0][1])),
                                         __dadd_rn(__dmul_rn(ra, r[1][0]), __dmul_rn(rb, r[1][1])));
            fc[idx] = __ddiv_rn(num, __dmul_rn(2.0, __dadd_rn(ra, rb)));
            ec[idx] = 0.0;
        }
    }
}

template <bool RESTRICT, bool MAXIMA, typename IDX>
__global__ void __launch_bounds__(256) k_mg_residual(const MgLevel Larg, double* __restrict__ fc, double* __restrict__ ec,
                                                     unsigned long long* __restrict__ slots, const Ctl* __restrict__ ctl,
                                                     const MgPtrs* __restrict__ pp) {
    if (ctl[blockIdx.y].done) return;
    const MgLevel L = mg_resolve(Larg, pp, blockIdx.y);
    const IDX n = (IDX)((L.nr + 1) / 2) * (IDX)((L.nz + 1) / 2);
    if (RESTRICT) { fc += (size_t)blockIdx.y * n; ec += (size_t)blockIdx.y * n; }
    if (MAXIMA) slots += 2 * blockIdx.y;
    unsigned long long kr = 0ull, kp = 0ull;
    for (IDX idx = (IDX)blockIdx.x * blockDim.x + threadIdx.x; idx < n; idx += (IDX)gridDim.x * blockDim.x)
        mg_residual_block<RESTRICT, MAXIMA, IDX>(L, idx, fc, ec, kr, kp);
    if (MAXIMA) {
        kr = warp_max_key(kr);
        kp = warp_max_key(kp);
        if ((threadIdx.x & 31) == 0) {
            atomicMax(slots, kr);
            atomicMax(slots + 1, kp);
        }
    }
}

// M8: max|res| and max|phi| of a level, one thread per CELL (coalesced rows; the 2 x 2 mapping above is only needed
// where the restriction wants the four residuals in one thread)
template <typename IDX>
__global__ void __launch_bounds__(256) k_mg_resmax(const MgLevel Larg, unsigned long long* __restrict__ slots,
                                                   const Ctl* __restrict__ ctl, const MgPtrs* __restrict__ pp) {
    if (ctl[blockIdx.y].done) return;
    const MgLevel L = mg_resolve(Larg, pp, blockIdx.y);
    const IDX n = (IDX)L.nr * (IDX)L.nz;
    slots += 2 * blockIdx.y;
    unsigned long long kr = 0ull, kp = 0ull;
    for (IDX idx = (IDX)blockIdx.x * blockDim.x + threadIdx.x; idx < n; idx += (IDX)gridDim.x * blockDim.x) {
        const int j = (int)(idx / (IDX)L.nr), i = (int)(idx - (IDX)j * (IDX)L.nr);
        const double pC = L.phi[idx];
        double diag, w;
        const double t = mg_apply_at(L, i, j, pC, diag, w);
        const double r = __dsub_rn(__dmul_rn(L.scale, L.src[idx]), t);
        const unsigned long long a1 = abs_key(r), a2 = abs_key(pC);
        kr = a1 > kr ? a1 : kr;
        kp = a2 > kp ? a2 : kp;
    }
    // warp -> CTA -> ONE atomic pair per CTA (thousands of warps hitting the same two words serialise in L2)
    __shared__ unsigned long long sk[2][8];
    kr = warp_max_key(kr);
    kp = warp_max_key(kp);
    if ((threadIdx.x & 31) == 0) { sk[0][threadIdx.x >> 5] = kr; sk[1][threadIdx.x >> 5] = kp; }
    __syncthreads();
    if (threadIdx.x < 32) {
        const unsigned nw = blockDim.x >> 5;
        kr = warp_max_key(threadIdx.x < nw ? sk[0][threadIdx.x] : 0ull);
        kp = warp_max_key(threadIdx.x < nw ? sk[1][threadIdx.x] : 0ull);
        if (threadIdx.x == 0) {
            atomicMax(slots, kr);
            atomicMax(slots + 1, kp);
        }
    }
}

// M7: coarse error with its ghost layer (rows first, then columns)
__device__ __forceinline__ double mg_ext(const MgLevel& Lc, int I, int J) {
    int i = I < 0 ? 0 : I >= Lc.nr ? Lc.nr - 1 : I;
    int j = J;
    double v;
    if (J < 0) {
        j = 0;
        v = Lc.phi[(size_t)j * Lc.nr + i];
        if (Lc.symmetry == 0) v = __dmul_rn(-Lc.beta, v);
    } else if (J >= Lc.nz) {
        j = Lc.nz - 1;
        v = __dmul_rn(-Lc.beta, Lc.phi[(size_t)j * Lc.nr + i]);
    } else {
        v = Lc.phi[(size_t)j * Lc.nr + i];
    }
    if (I >= Lc.nr) v = __dmul_rn(-Lc.beta, v);
    return v;
}

// M7: phi_f += bilinear interpolation of the coarse error, fine cell idx
template <typename IDX>
__device__ __forceinline__ void mg_prolong_cell(const MgLevel& Lc, double* phi_f, int nr_f, IDX idx) {
    const int j = (int)(idx / (IDX)nr_f), i = (int)(idx - (IDX)j * (IDX)nr_f);
    const int I = i >> 1, J = j >> 1, di = (i & 1) ? 1 : -1, dj = (j & 1) ? 1 : -1;
    const double C = mg_ext(Lc, I, J), H = mg_ext(Lc, I + di, J), V = mg_ext(Lc, I, J + dj), Dg = mg_ext(Lc, I + di, J + dj);
    const double e = __dmul_rn(__dadd_rn(__dadd_rn(__dadd_rn(__dmul_rn(9.0, C), __dmul_rn(3.0, H)), __dmul_rn(3.0, V)), Dg), 0.0625);
    phi_f[idx] = __dadd_rn(phi_f[idx], e);
}

// one thread per fine cell
template <typename IDX>
__global__ void __launch_bounds__(256) k_mg_prolong_add(const MgLevel Lcarg, double* phi_f, int nr_f, int nz_f,
                                                        const Ctl* __restrict__ ctl, const MgPtrs* __restrict__ pp) {
    if (ctl[blockIdx.y].done) return;
    if (phi_f == nullptr) phi_f = pp->phi;           // level 0
    phi_f += (size_t)blockIdx.y * nr_f * nz_f;
    const MgLevel Lc = mg_resolve(Lcarg, pp, blockIdx.y);
    const IDX n = (IDX)nr_f * (IDX)nz_f;
    for (IDX idx = (IDX)blockIdx.x * blockDim.x + threadIdx.x; idx < n; idx += (IDX)gridDim.x * blockDim.x)
        mg_prolong_cell<IDX>(Lc, phi_f, nr_f, idx);
}

// The tail of the V-cycle -- every level small enough for ONE CTA (<= kMgTailCells cells) down to the coarsest and back
// up -- as a single launch: these levels are a few thousand cells and purely launch / latency bound as separate
// kernels (six launches per level and cycle, plus 2 nc half-sweeps on the coarsest).  The error and the right-hand side
// of every tail level live in SHARED memory for the duration of the launch (<= 171 KB), the phases are the same device
// functions as above, separated by CTA barriers.  L[0] is the finest level of the tail, L[n-1] the coarsest (M6).
constexpr int kMgMaxLevels = 14;
constexpr int kMgTailCells = 8192;
struct MgTail {
    int n, nu1, nu2, nc;
    MgLevel L[kMgMaxLevels];
};
// doubles of dynamic shared memory the tail needs: phi and f of every level
inline size_t mg_tail_smem_doubles(const MgTail& T) {
    size_t d = 0;
    for (int l = 0; l < T.n; ++l) d += 2 * (size_t)T.L[l].nr * T.L[l].nz + 2 * (size_t)T.L[l].nr;      // phi, f, cE, cW
    return d;
}

__global__ void __launch_bounds__(1024) k_mg_tail(const MgTail T, const Ctl* __restrict__ ctl, const MgPtrs* __restrict__ pp) {
    extern __shared__ __align__(16) double mg_sm[];
    __shared__ MgLevel L[kMgMaxLevels];           // the levels with their arrays re-pointed to shared memory
    __shared__ double* fw[kMgMaxLevels];
    __shared__ double* cw[kMgMaxLevels];
    const int member = blockIdx.x;               // one CTA per batch member
    if (ctl[member].done) return;
    {
        if (threadIdx.x == 0) {
            double* p = mg_sm;
            for (int l = 0; l < T.n; ++l) {
                const size_t n = (size_t)T.L[l].nr * T.L[l].nz;
                L[l] = l == 0 ? mg_resolve(T.L[0], pp, member) : T.L[l];       // level 0 of the grid keeps its (member's) ghosts
                L[l].phi = p; fw[l] = p + n; L[l].src = fw[l];
                p += 2 * n;
                cw[l] = p;                        // the coefficient tables too: cE [nr], cW [nr]
                p += 2 * T.L[l].nr;
            }
        }
        __syncthreads();
        for (int l = 0; l < T.n; ++l) {
            for (int i = threadIdx.x; i < T.L[l].nr; i += blockDim.x) { cw[l][i] = T.L[l].cE[i]; cw[l][T.L[l].nr + i] = T.L[l].cW[i]; }
        }
        __syncthreads();
        if (threadIdx.x == 0)
            for (int l = 0; l < T.n; ++l) { L[l].cE = cw[l]; L[l].cW = cw[l] + T.L[l].nr; }
        const MgLevel G0 = mg_resolve(T.L[0], pp, member);
        const size_t n0 = (size_t)T.L[0].nr * T.L[0].nz;
        for (size_t i = threadIdx.x; i < n0; i += blockDim.x) { L[0].phi[i] = G0.phi[i]; fw[0][i] = G0.src[i]; }
        __syncthreads();
    }
    // (every phase works on a LOCAL copy of its level descriptor: read through the shared-memory struct, each field would
    // be re-fetched after every store to phi, which may alias it as far as the compiler knows)
    auto smooth = [&](const MgLevel& Lshared, int nsweeps) {
        const MgLevel Lv = Lshared;
        const unsigned n = (unsigned)((Lv.nr + 1) / 2) * (unsigned)Lv.nz;
        if (n <= 32u) {                           // a level of <= 64 cells: one warp, warp barriers instead of CTA barriers
            if (threadIdx.x < 32u) {
                for (int s = 0; s < 2 * nsweeps; ++s) {
                    if (threadIdx.x < n) mg_update_cell<unsigned>(Lv, threadIdx.x, s & 1);
                    __syncwarp();
                }
            }
            __syncthreads();
            return;
        }
        for (int s = 0; s < 2 * nsweeps; ++s) {
            for (unsigned idx = threadIdx.x; idx < n; idx += blockDim.x) mg_update_cell<unsigned>(Lv, idx, s & 1);
            __syncthreads();
        }
    };
    unsigned long long kr = 0ull, kp = 0ull;
    for (int l = 0; l + 1 < T.n; ++l) {                              // down
        smooth(L[l], T.nu1);
        const unsigned nc = (unsigned)L[l + 1].nr * (unsigned)L[l + 1].nz;
        {
            const MgLevel Lf = L[l];
            double* const fcw = fw[l + 1];
            double* const ecw = L[l + 1].phi;
            for (unsigned idx = threadIdx.x; idx < nc; idx += blockDim.x)
                mg_residual_block<true, false, unsigned>(Lf, idx, fcw, ecw, kr, kp);
        }
        __syncthreads();
    }
    smooth(L[T.n - 1], T.n == 1 ? T.nu1 + T.nu2 : T.nc);             // coarsest (a single-level grid: plain Gauss-Seidel)
    for (int l = T.n - 2; l >= 0; --l) {                             // up
        const unsigned nf = (unsigned)L[l].nr * (unsigned)L[l].nz;
        {
            const MgLevel Lc = L[l + 1];
            double* const pf = L[l].phi;
            const int nrf = L[l].nr;
            for (unsigned idx = threadIdx.x; idx < nf; idx += blockDim.x) mg_prolong_cell<unsigned>(Lc, pf, nrf, idx);
        }
        __syncthreads();
        smooth(L[l], T.nu2);
    }
    double* out0 = mg_resolve(T.L[0], pp, member).phi;
    const size_t n0 = (size_t)T.L[0].nr * T.L[0].nz;
    for (size_t i = threadIdx.x; i < n0; i += blockDim.x) out0[i] = L[0].phi[i];
}

// M8: the stopping ratio of the cycle just finished; resets the maxima for the next one
__global__ void k_mg_decide(Ctl* __restrict__ ctl_all, unsigned long long* __restrict__ slots_all, double D, double tol,
                            int max_cycles, double* __restrict__ hist_all, int hist_stride) {
    if (threadIdx.x != 0) return;
    Ctl* ctl = ctl_all + blockIdx.x;                       // one block per batch member
    unsigned long long* slots = slots_all + 2 * blockIdx.x;
    double* hist = hist_all + (size_t)blockIdx.x * hist_stride;
    if (ctl->done) return;
    const int cycle = ctl->sweeps + 1;
    const double R = stop_ratio(slots[0], slots[1], ctl->maxf, D);
    slots[0] = 0ull;
    slots[1] = 0ull;
    hist[cycle - 1] = R;
    ctl->sweeps = cycle;
    ctl->residual = R;
    if (is_nonfinite(R)) { ctl->status = -3; ctl->done = 1; }
    else if (tol > 0.0 && R <= tol) { ctl->status = 0; ctl->done = 1; }
    else if (cycle >= max_cycles) { ctl->status = tol > 0.0 ? 1 : 0; ctl->done = 1; }
}

}  // namespace snp
