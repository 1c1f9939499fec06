// gravity.cuh -- NEXT-1: the gravity field g = -grad phi that the momentum and energy
// equations of the paper use as source terms (eqs. 2-4: -rho dPhi/dr, -rho dPhi/dz).
// DESIGN.md R15: centred differences at the cell centres with the solver's own boundary handling -- reflecting
// axis (phi_{-1,j} = phi_{0,j}), reflecting equator when symmetry = 1, the Dirichlet ghosts bE / bN / bS of the last
// solve elsewhere; pinned arithmetic (lo - hi) * (0.5 / d).  HBM bound: 8 B read + 16 B written per cell.
#pragma once
#include "common.cuh"

namespace snp {

// Four consecutive cells of one row per thread (nr % 4 == 0, 16-byte aligned arrays).  grid = (ceil(nr/4/128) * nz, 1, nb).
__global__ void __launch_bounds__(128) k_gravity4(Geom g, int qx, const double* __restrict__ phi, const double* __restrict__ bE,
                                                  const double* __restrict__ bN, const double* __restrict__ bS,
                                                  double* __restrict__ gr, double* __restrict__ gz) {
    const int j = blockIdx.x / qx, b = blockIdx.z;             // grid.x = qx blocks per row x nz rows
    const int q = (blockIdx.x - j * qx) * blockDim.x + threadIdx.x;       // quad index in the row
    const int i0 = 4 * q;
    if (i0 >= g.nr) return;
    const size_t ncell = (size_t)g.nr * g.nz;
    const double* p = phi + (size_t)b * ncell;
    const size_t c = (size_t)j * g.nr + i0;
    const double hr = 0.5 / g.dr, hz = 0.5 / g.dz;
    const double2 c0 = *reinterpret_cast<const double2*>(p + c), c1 = *reinterpret_cast<const double2*>(p + c + 2);
    const double v[4] = {c0.x, c0.y, c1.x, c1.y};
    const double west = i0 > 0 ? p[c - 1] : v[0];                                    // reflecting axis
    const double east = i0 + 4 < g.nr ? p[c + 4] : bE[(size_t)b * g.nz + j];
    double n[4], s[4];
    if (j + 1 < g.nz) {
        const double2 a0 = *reinterpret_cast<const double2*>(p + c + g.nr), a1 = *reinterpret_cast<const double2*>(p + c + g.nr + 2);
        n[0] = a0.x; n[1] = a0.y; n[2] = a1.x; n[3] = a1.y;
    } else {
        const double2 a0 = *reinterpret_cast<const double2*>(bN + (size_t)b * g.nr + i0), a1 = *reinterpret_cast<const double2*>(bN + (size_t)b * g.nr + i0 + 2);
        n[0] = a0.x; n[1] = a0.y; n[2] = a1.x; n[3] = a1.y;
    }
    if (j > 0) {
        const double2 a0 = *reinterpret_cast<const double2*>(p + c - g.nr), a1 = *reinterpret_cast<const double2*>(p + c - g.nr + 2);
        s[0] = a0.x; s[1] = a0.y; s[2] = a1.x; s[3] = a1.y;
    } else if (g.symmetry == 1) {
        s[0] = v[0]; s[1] = v[1]; s[2] = v[2]; s[3] = v[3];                          // reflecting equator
    } else {
        const double2 a0 = *reinterpret_cast<const double2*>(bS + (size_t)b * g.nr + i0), a1 = *reinterpret_cast<const double2*>(bS + (size_t)b * g.nr + i0 + 2);
        s[0] = a0.x; s[1] = a0.y; s[2] = a1.x; s[3] = a1.y;
    }
    double r4[4], z4[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const double pW = k == 0 ? west : v[k - 1], pE = k == 3 ? east : v[k + 1];
        r4[k] = __dmul_rn(__dsub_rn(pW, pE), hr);
        z4[k] = __dmul_rn(__dsub_rn(s[k], n[k]), hz);
    }
    double* orow = gr + (size_t)b * ncell + c;
    double* zrow = gz + (size_t)b * ncell + c;
    *reinterpret_cast<double2*>(orow) = make_double2(r4[0], r4[1]);
    *reinterpret_cast<double2*>(orow + 2) = make_double2(r4[2], r4[3]);
    *reinterpret_cast<double2*>(zrow) = make_double2(z4[0], z4[1]);
    *reinterpret_cast<double2*>(zrow + 2) = make_double2(z4[2], z4[3]);
}

// One cell per thread: any grid, any alignment.  grid = (ceil(nr/128) * nz, 1, nb).
__global__ void __launch_bounds__(128) k_gravity1(Geom g, int qx, const double* __restrict__ phi, const double* __restrict__ bE,
                                                  const double* __restrict__ bN, const double* __restrict__ bS,
                                                  double* __restrict__ gr, double* __restrict__ gz) {
    const int j = blockIdx.x / qx, b = blockIdx.z;
    const int i = (blockIdx.x - j * qx) * blockDim.x + threadIdx.x;
    if (i >= g.nr) return;
    const size_t ncell = (size_t)g.nr * g.nz;
    const double* p = phi + (size_t)b * ncell;
    const size_t c = (size_t)j * g.nr + i;
    const double pC = p[c];
    const double pE = i + 1 < g.nr ? p[c + 1] : bE[(size_t)b * g.nz + j];
    const double pW = i > 0 ? p[c - 1] : pC;
    const double pN = j + 1 < g.nz ? p[c + g.nr] : bN[(size_t)b * g.nr + i];
    const double pS = j > 0 ? p[c - g.nr] : (g.symmetry == 1 ? pC : bS[(size_t)b * g.nr + i]);
    gr[(size_t)b * ncell + c] = __dmul_rn(__dsub_rn(pW, pE), 0.5 / g.dr);
    gz[(size_t)b * ncell + c] = __dmul_rn(__dsub_rn(pS, pN), 0.5 / g.dz);
}

}  // namespace snp
