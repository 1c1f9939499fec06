// moments.cuh -- step a-1 (multipole moments) and a-1b (boundary fill).
// PAPER.md:99 gives only the monopole ("Roche approximation ... in general higher multipole terms are needed");
// the expansion to lmax, its scaling by L0 = nr*dr and the ghost placement are DESIGN.md R4-R6.
#pragma once
#include "common.cuh"

namespace snp {

constexpr int kMomThreads = 256;

// One pass over rho: per-block partial sums of M_l (l = 0..NL-1) and max|4 pi rho|.
//   M_l = sum rho_ij (s_ij/L0)^l P_l(z_j/s_ij) dV_i, dV_i = 2 pi r_i dr dz, by the division-free recurrence
//   R_0 = 1, R_1 = y, (l+1) R_{l+1} = (2l+1) y R_l - l (x^2+y^2) R_{l-1}, x = r/L0, y = z/L0.
// grid = (blocks, nbatch).  Reduction: registers -> warp shuffle -> shared -> partial[b][block][NL].
template <int NL>
__global__ void __launch_bounds__(kMomThreads) k_moments(const double* __restrict__ rho, Geom g, double L0,
                                                         double* __restrict__ partial, Ctl* __restrict__ ctl) {
    const int b = blockIdx.y;
    const size_t ncell = (size_t)g.nr * g.nz;
    const double* rb = rho + (size_t)b * ncell;
    double acc[NL];
#pragma unroll
    for (int l = 0; l < NL; ++l) acc[l] = 0.0;
    unsigned long long mf = 0ull;
    const double zoff = g.symmetry == 1 ? 0.5 : 0.5 - 0.5 * g.nz;
    for (size_t idx = (size_t)blockIdx.x * kMomThreads + threadIdx.x; idx < ncell;
         idx += (size_t)gridDim.x * kMomThreads) {
        const int j = (int)(idx / g.nr);
        const int i = (int)(idx - (size_t)j * g.nr);
        const double r = (i + 0.5) * g.dr;
        const double z = (j + zoff) * g.dz;
        const double x = r / L0, y = z / L0;
        const double s2 = x * x + y * y;
        const double rv = rb[idx];
        const double w = rv * (2.0 * kPi * r * g.dr * g.dz);
        const unsigned long long fk = abs_key(kFourPi * rv);
        mf = fk > mf ? fk : mf;
        double Rm = 1.0, Rc = y;          // R_{l-1}, R_l
        acc[0] += w;
        if (NL > 1) acc[1] += w * Rc;
#pragma unroll
        for (int l = 1; l < NL - 1; ++l) {
            // (the division by l + 1 as a multiplication by its rounded reciprocal: an IEEE fp64 division is ~18
            // instructions, a third of this kernel; the moments are not bit-pinned -- their summation order differs from any
            // serial sum anyway -- and stay within 1e-13 of the serial long-double sum, tests/test_gpu_parity.py)
            const double Rn = ((2 * l + 1) * y * Rc - l * s2 * Rm) * (1.0 / (l + 1));
            acc[l + 1] += w * Rn;
            Rm = Rc;
            Rc = Rn;
        }
    }
    __shared__ double sh[kMomThreads / 32][NL];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int l = 0; l < NL; ++l) {
        double v = acc[l];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (lane == 0) sh[warp][l] = v;
    }
    mf = warp_max_u64(mf);
    if (lane == 0) atomicMax((unsigned long long*)&ctl[b].maxf, mf);
    __syncthreads();
    if (threadIdx.x < NL) {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < kMomThreads / 32; ++w) v += sh[w][threadIdx.x];
        partial[((size_t)b * gridDim.x + blockIdx.x) * NL + threadIdx.x] = v;
    }
}

// Fixed-order final sum over blocks (deterministic), symmetry rule, then the ghost values
//   phi_b = -(1/L0) sum_l M_l I_l,  I_0 = 1/shat, I_1 = y/shat^3, (l+1) I_{l+1} = ((2l+1) y I_l - l I_{l-1})/shat^2
// at east (r=(nr+1/2)dr, z_j), north (r_i, z_{nz-1}+dz) and, for symmetry=0, south (r_i, z_0-dz) ghost centres.
// grid = (nbatch, slices): every block forms the moments itself (same fixed order, so every block gets the same bits;
// slice 0 stores them) and fills its slice of the ghost points, one point per thread and pass.
__global__ void __launch_bounds__(256) k_boundary(Geom g, double L0, int NL, int nblocks,
                                                  const double* __restrict__ partial, double* __restrict__ M,
                                                  double* __restrict__ bE, double* __restrict__ bN,
                                                  double* __restrict__ bS, int have_moments) {
    const int b = blockIdx.x;
    __shared__ double sM[kMaxL + 1];
    double* Mb = M + (size_t)b * (kMaxL + 1);
    for (int l = threadIdx.x; l <= g.lmax; l += blockDim.x) {
        double v;
        if (!have_moments) {
            v = 0.0;
            for (int k = 0; k < nblocks; ++k) v += partial[((size_t)b * nblocks + k) * NL + l];
            if (g.symmetry == 1) v = (l & 1) ? 0.0 : 2.0 * v;
            if (blockIdx.y == 0) Mb[l] = v;
        } else {
            v = Mb[l];
        }
        sM[l] = v;
    }
    __syncthreads();
    const double zoff = g.symmetry == 1 ? 0.5 : 0.5 - 0.5 * g.nz;
    const int npts = g.nz + g.nr + (g.symmetry == 0 ? g.nr : 0);
    for (int p = blockIdx.y * blockDim.x + threadIdx.x; p < npts; p += gridDim.y * blockDim.x) {
        double r, z;
        double* dst;
        if (p < g.nz) {
            r = (g.nr + 0.5) * g.dr;
            z = (p + zoff) * g.dz;
            dst = bE + (size_t)b * g.nz + p;
        } else if (p < g.nz + g.nr) {
            const int i = p - g.nz;
            r = (i + 0.5) * g.dr;
            z = (g.nz - 1 + zoff) * g.dz + g.dz;
            dst = bN + (size_t)b * g.nr + i;
        } else {
            const int i = p - g.nz - g.nr;
            r = (i + 0.5) * g.dr;
            z = (0 + zoff) * g.dz - g.dz;
            dst = bS + (size_t)b * g.nr + i;
        }
        const double x = r / L0, y = z / L0;
        const double s2 = x * x + y * y;
        const double s = sqrt(s2);
        double Im = 1.0 / s;
        double sum = sM[0] * Im;
        if (g.lmax >= 1) {
            double Ic = y / (s2 * s);
            sum += sM[1] * Ic;
            for (int l = 1; l < g.lmax; ++l) {
                const double In = ((2 * l + 1) * y * Ic - l * Im) / ((l + 1) * s2);
                sum += sM[l + 1] * In;
                Im = Ic;
                Ic = In;
            }
        }
        *dst = -sum / L0;
    }
}

}  // namespace snp
