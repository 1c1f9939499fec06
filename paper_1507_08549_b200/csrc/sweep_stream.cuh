// sweep_stream.cuh -- steps a-2 + a-3 with phi streamed from L2/HBM: one launch per colour.
// This is the general path (any grid size, any batch); the resident persistent kernel (sweep_resident.cuh) replaces
// it when the grid fits on chip.  PAPER.md:99: "successive overrelaxation method with the Gauss-Seidel method";
// red-black ordering, coefficients and the pinned expression tree are DESIGN.md R1, R3, R7, R10.
#pragma once
#include "common.cuh"

namespace snp {

constexpr int kStreamWarps = 8;      // warps per block
constexpr int kStreamRows = 4;       // rows per warp
constexpr int kStreamTileW = 64;     // cells per block row (32 lanes x one colour pair)
constexpr int kStreamTileH = kStreamWarps * kStreamRows;

// Device-side stopping decision for sweep k-1, evaluated redundantly (and identically) by every block at the start
// of both half-sweeps of sweep k: all blocks read the same final slot values, so all take the same branch.
// `writer` (one thread of the red launch) records it.  Returns true if no more updates may be applied.
__device__ __forceinline__ bool member_finished(const Geom& g, int member, int k, const unsigned long long* slots, Ctl* ctl,
                                                double* hist, bool writer) {
    if (k <= 1) return false;
    if (*(volatile int*)&ctl->done) return true;
    const double R = stop_value(g, slots[2 * (k - 2)], slots[2 * (k - 2) + 1],
                                g.rule != 0 ? g.slots0_x[(size_t)member * g.slots0_stride + k - 2] : 0ull, ctl->maxf);
    const bool bad = is_nonfinite(R);
    const bool stop = bad || (g.tol > 0.0 && R <= g.tol);
    if (writer) {
        hist[k - 2] = R;
        if (stop) {
            ctl->sweeps = k - 1;
            ctl->residual = R;
            ctl->status = bad ? -3 : 0;
            __threadfence();
            ctl->done = 1;
        }
    }
    return stop;
}

// Half-sweep of colour `colour` of sweep k (1-based).  grid = (ceil(nr/64), ceil(nz/32), nbatch), 256 threads.
// Lane l of a warp owns the cell pair (2k, 2k+1) of each of its rows and updates the one with (i+j)&1 == colour.
// slots[b][2*(k-1)+{0,1}] accumulate max|res| and max|phi_new| of sweep k as order-preserving u64 keys.
__global__ void __launch_bounds__(kStreamWarps * 32)
    k_halfsweep(Geom g, int colour, int k, int slot_stride, int hist_stride, const double* __restrict__ rho,
                double* __restrict__ phi, const double* __restrict__ bE, const double* __restrict__ bN,
                const double* __restrict__ bS, unsigned long long* __restrict__ slots, Ctl* __restrict__ ctl,
                double* __restrict__ hist) {
    const int b = blockIdx.z;
    unsigned long long* sl = slots + (size_t)b * slot_stride;
    __shared__ int s_fin;
    __shared__ unsigned long long s_red[2][kStreamWarps];
    if (threadIdx.x == 0) {
        const bool writer = colour == 0 && blockIdx.x == 0 && blockIdx.y == 0;
        s_fin = member_finished(g, b, k, sl, ctl + b, hist + (size_t)b * hist_stride, writer) ? 1 : 0;
    }
    __syncthreads();
    if (s_fin) return;

    const size_t ncell = (size_t)g.nr * g.nz;
    const double* rb = rho + (size_t)b * ncell;
    double* pb = phi + (size_t)b * ncell;
    const double* bEb = bE + (size_t)b * g.nz;
    const double* bNb = bN + (size_t)b * g.nr;
    const double* bSb = bS + (size_t)b * g.nr;

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int pair = blockIdx.x * 32 + lane;
    const int j0 = blockIdx.y * kStreamTileH + warp * kStreamRows;
    unsigned long long mres = 0ull, mphi = 0ull, mres0 = 0ull;
#pragma unroll
    for (int q = 0; q < kStreamRows; ++q) {
        const int j = j0 + q;
        const int i = 2 * pair + ((j + colour) & 1);
        if (j < g.nz && i < g.nr) {
            const size_t c = (size_t)j * g.nr + i;
            const bool mirror_row = (g.symmetry == 1 && j == 0);
            const double cS = mirror_row ? 0.0 : g.iz2;
            const double diag = mirror_row ? g.D0 : g.D;
            const double w = mirror_row ? g.wD0 : g.wD;
            const double pC = pb[c];
            const double pE = (i + 1 < g.nr) ? pb[c + 1] : bEb[j];
            const double pW = (i > 0) ? pb[c - 1] : 0.0;
            const double pN = (j + 1 < g.nz) ? pb[c + g.nr] : bNb[i];
            const double pS = (j > 0) ? pb[c - g.nr] : (g.symmetry == 1 ? 0.0 : bSb[i]);
            const double f = __dmul_rn(kFourPi, rb[c]);
            double res;
            const double pn = sor_update(g.cE[i], g.cW[i], g.iz2, cS, diag, w, pE, pW, pN, pS, pC, f, res);
            pb[c] = pn;
            const unsigned long long kr = abs_key(res), kp = abs_key(pn);
            mres = kr > mres ? kr : mres;
            mphi = kp > mphi ? kp : mphi;
            if (mirror_row) mres0 = kr > mres0 ? kr : mres0;
        }
    }
    if (g.rule != 0 && g.symmetry == 1 && j0 == 0) {         // rule 1 (R16): the warp that holds the equator row
        mres0 = warp_max_u64(mres0);
        if (lane == 0) atomicMax(g.slots0_x + (size_t)b * g.slots0_stride + k - 1, mres0);
    }
    mres = warp_max_u64(mres);
    mphi = warp_max_u64(mphi);
    if (lane == 0) {
        s_red[0][warp] = mres;
        s_red[1][warp] = mphi;
    }
    __syncthreads();
    if (threadIdx.x < 2) {
        unsigned long long v = 0ull;
#pragma unroll
        for (int w = 0; w < kStreamWarps; ++w) v = s_red[threadIdx.x][w] > v ? s_red[threadIdx.x][w] : v;
        atomicMax(&sl[2 * (k - 1) + threadIdx.x], v);
    }
}

// Closes a run: decides the last launched sweep `k_last` for every member that has not fired yet.  grid = nbatch.
__global__ void k_decide_last(Geom g, int k_last, int slot_stride, int hist_stride,
                              const unsigned long long* __restrict__ slots, Ctl* __restrict__ ctl,
                              double* __restrict__ hist) {
    const int b = blockIdx.x;
    if (threadIdx.x != 0) return;
    Ctl* c = ctl + b;
    if (c->done) return;
    if (k_last <= 0) {
        c->done = 1; c->sweeps = 0; c->residual = 0.0; c->status = g.tol > 0.0 ? 1 : 0;
        return;
    }
    const unsigned long long* sl = slots + (size_t)b * slot_stride;
    const double R = stop_value(g, sl[2 * (k_last - 1)], sl[2 * (k_last - 1) + 1],
                                g.rule != 0 ? g.slots0_x[(size_t)b * g.slots0_stride + k_last - 1] : 0ull, c->maxf);
    hist[(size_t)b * hist_stride + k_last - 1] = R;
    c->sweeps = k_last;
    c->residual = R;
    c->status = is_nonfinite(R) ? -3 : (g.tol > 0.0 ? (R <= g.tol ? 0 : 1) : 0);
    c->done = 1;
}

}  // namespace snp
