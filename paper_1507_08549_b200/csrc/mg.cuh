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

// t = (A phi)(i, j) with the pinned tree (R10); ghosts per M2.  Also returns the row's diagonal and omega / diag.
__device__ __forceinline__ double mg_apply_at(const MgLevel& L, int i, int j, double pC, double& diag, double& w) {
    const size_t c = (size_t)j * L.nr + i;
    const bool mirror_row = L.symmetry == 1 && j == 0;
    const double cS = mirror_row ? 0.0 : L.iz2;
    diag = mirror_row ? L.D0 : L.D;
    w = mirror_row ? L.wD0 : L.wD;
    const double ghost = -__dmul_rn(L.beta, pC);
    const double pE = (i + 1 < L.nr) ? L.phi[c + 1] : (L.bE ? L.bE[j] : ghost);
    const double pW = (i > 0) ? L.phi[c - 1] : 0.0;
    const double pN = (j + 1 < L.nz) ? L.phi[c + L.nr] : (L.bN ? L.bN[i] : ghost);
    const double pS = (j > 0) ? L.phi[c - L.nr] : (L.symmetry == 1 ? 0.0 : (L.bS ? L.bS[i] : ghost));
    double t = __dmul_rn(L.cE[i], pE);
    t = __fma_rn(L.cW[i], pW, t);
    t = __fma_rn(L.iz2, pN, t);
    t = __fma_rn(cS, pS, t);
    t = __fma_rn(-diag, pC, t);
    return t;
}

// M3: one half-sweep of colour COL; one thread per cell of that colour
template <int COL>
__global__ void __launch_bounds__(256) k_mg_halfsweep(const MgLevel L) {
    const int half = (L.nr + 1) / 2;
    const size_t n = (size_t)half * L.nz;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < n; idx += (size_t)gridDim.x * blockDim.x) {
        const int j = (int)(idx / half), i = 2 * (int)(idx - (size_t)j * half) + ((j + COL) & 1);
        if (i >= L.nr) continue;
        const size_t c = (size_t)j * L.nr + i;
        const double pC = L.phi[c];
        double diag, w;
        const double t = mg_apply_at(L, i, j, pC, diag, w);
        const double res = __dsub_rn(__dmul_rn(L.scale, L.src[c]), t);
        L.phi[c] = __fma_rn(-w, res, pC);
    }
}

// M6: the coarsest level, nc sweeps by ONE CTA (the level is a few dozen cells; any size works)
__global__ void __launch_bounds__(1024) k_mg_coarse(const MgLevel L, int nc) {
    const int half = (L.nr + 1) / 2;
    const int n = half * L.nz;
    for (int s = 0; s < 2 * nc; ++s) {
        const int col = s & 1;
        for (int idx = threadIdx.x; idx < n; idx += blockDim.x) {
            const int j = idx / half, i = 2 * (idx - j * half) + ((j + col) & 1);
            if (i >= L.nr) continue;
            const size_t c = (size_t)j * L.nr + i;
            const double pC = L.phi[c];
            double diag, w;
            const double t = mg_apply_at(L, i, j, pC, diag, w);
            const double res = __dsub_rn(__dmul_rn(L.scale, L.src[c]), t);
            L.phi[c] = __fma_rn(-w, res, pC);
        }
        __syncthreads();
    }
}

// M4 + M5 + M8: one thread per 2 x 2 block of the level.  RESTRICT: the volume-weighted average of the four residuals
// becomes the right-hand side of the next coarser level, whose error is zeroed.  MAXIMA: max|res| and max|phi| of the
// level as order-preserving keys (warp REDUX, one atomicMax per warp) for the stopping ratio.
template <bool RESTRICT, bool MAXIMA>
__global__ void __launch_bounds__(256) k_mg_residual(const MgLevel L, double* __restrict__ fc, double* __restrict__ ec,
                                                     unsigned long long* __restrict__ slots) {
    const int nrc = (L.nr + 1) / 2, nzc = (L.nz + 1) / 2;
    const size_t n = (size_t)nrc * nzc;
    unsigned long long kr = 0ull, kp = 0ull;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < n; idx += (size_t)gridDim.x * blockDim.x) {
        const int J = (int)(idx / nrc), I = (int)(idx - (size_t)J * nrc);
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
    if (MAXIMA) {
        kr = warp_max_key(kr);
        kp = warp_max_key(kp);
        if ((threadIdx.x & 31) == 0) {
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

// M7: phi_f += bilinear interpolation of the coarse error; one thread per fine cell
__global__ void __launch_bounds__(256) k_mg_prolong_add(const MgLevel Lc, double* __restrict__ phi_f, int nr_f, int nz_f) {
    const size_t n = (size_t)nr_f * nz_f;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < n; idx += (size_t)gridDim.x * blockDim.x) {
        const int j = (int)(idx / nr_f), i = (int)(idx - (size_t)j * nr_f);
        const int I = i >> 1, J = j >> 1, di = (i & 1) ? 1 : -1, dj = (j & 1) ? 1 : -1;
        const double C = mg_ext(Lc, I, J), H = mg_ext(Lc, I + di, J), V = mg_ext(Lc, I, J + dj), Dg = mg_ext(Lc, I + di, J + dj);
        const double e = __dmul_rn(__dadd_rn(__dadd_rn(__dadd_rn(__dmul_rn(9.0, C), __dmul_rn(3.0, H)), __dmul_rn(3.0, V)), Dg), 0.0625);
        phi_f[idx] = __dadd_rn(phi_f[idx], e);
    }
}

// M8: the stopping ratio of the cycle just finished; resets the maxima for the next one
__global__ void k_mg_decide(Ctl* __restrict__ ctl, unsigned long long* __restrict__ slots, double D, double tol, int cycle,
                            int max_cycles, double* __restrict__ hist) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    if (ctl->done) return;
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
