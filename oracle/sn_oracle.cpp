// sn_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded fp64 CPU implementation of the self-gravity Poisson solve of
// arXiv 1507.08549 ("Phi ... satisfies the Poisson Equation nabla^2 Phi = 4 pi G rho";
// PAPER.md:99 "successive overrelaxation method with the Gauss-Seidel method ... in cylindrical
// coordinates ... inner boundaries are assumed to be reflecting and the outer boundaries are fixed by
// using the Roche approximation Phi(r,z) = -GM/sqrt(r^2+z^2) ... in general higher multipole terms are
// needed").  The paper gives no stencil, relaxation factor, ordering or stopping arithmetic; every such
// choice is a reading listed in DESIGN.md §3 (R1..R15), cited below as [R#].
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load this
// file's library.  It shares no code with paper_1507_08549_b200/csrc and is never called by the product.
//
// The method is an iteration, so this file follows the algorithm step by step; there is no blocking,
// fusion or reordering.  Compile with:  g++ -O2 -ffp-contract=off -mfma  (std::fma -> one rounding).
//
// What pins it (tests/test_oracle_pins.py, all `-m "not gpu"`):
//   * fixed point of the iteration  <- dense direct solve (numpy) on <=16x16 grids, both symmetries
//   * operator accuracy / order     <- n=1 polytrope closed form, error falls x4 per refinement
//   * uniform sphere                <- closed form -2 pi rho (R^2 - s^2/3) inside, -M/s outside
//   * moments / boundary            <- M_0 = sum rho dV; lmax=0 ghosts == Roche formula;
//                                      point-mass ring potential via elliptic K; Legendre closed forms
//   * reflecting boundary           <- mirrored full-plane solve == half-plane solve
//   * discrete Gauss law, linearity, omega formula vs Jacobi spectral radius, omega=1 == Gauss-Seidel
//   * gravity epilogue (sno_gravity) <- exact on quadratic potentials, closed-form polytrope field at O(h^2)
//   * iteration history (the per-sweep iterate): defined by this file; nothing external can pin it
//     beyond the above -- stated in DESIGN.md §5.
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>

namespace {

const double FOURPI = 12.566370614359172;      // 4*pi rounded to fp64 [R10]
const double J01 = 2.404825557695773;          // first zero of J0 [R8]
const double PI = 3.141592653589793;

struct Grid {
    int nr, nz, symmetry;
    double dr, dz;
    double L0;                                  // scaling length nr*dr for the harmonics [R6]
    double r(int i) const { return (i + 0.5) * dr; }                       // cell centre [R2]
    double z(int j) const {
        return symmetry == 1 ? (j + 0.5) * dz : (j + 0.5 - 0.5 * nz) * dz;   // [R2]
    }
};

Grid make_grid(int nr, int nz, double dr, double dz, int symmetry) {
    Grid g;
    g.nr = nr; g.nz = nz; g.dr = dr; g.dz = dz; g.symmetry = symmetry;
    g.L0 = nr * dr;
    return g;
}

// Regular solid harmonics R_l = (s/L0)^l P_l(cos theta), theta from +z, x = r/L0, y = z/L0 [R6]:
//   R_0 = 1, R_1 = y, (l+1) R_{l+1} = (2l+1) y R_l - l (x^2+y^2) R_{l-1}      (Legendre recurrence x s^l)
void regular_harmonics(double x, double y, int lmax, double* R) {
    const double s2 = x * x + y * y;
    R[0] = 1.0;
    if (lmax >= 1) R[1] = y;
    for (int l = 1; l < lmax; ++l)
        R[l + 1] = ((2 * l + 1) * y * R[l] - l * s2 * R[l - 1]) / (l + 1);
}

// Irregular solid harmonics I_l = P_l(cos theta) / shat^(l+1), shat = s/L0 [R6]:
//   I_0 = 1/shat, I_1 = y/shat^3, (l+1) I_{l+1} = ((2l+1) y I_l - l I_{l-1}) / shat^2
void irregular_harmonics(double x, double y, int lmax, double* I) {
    const double s2 = x * x + y * y;
    const double s = std::sqrt(s2);
    I[0] = 1.0 / s;
    if (lmax >= 1) I[1] = y / (s2 * s);
    for (int l = 1; l < lmax; ++l)
        I[l + 1] = ((2 * l + 1) * y * I[l] - l * I[l - 1]) / ((l + 1) * s2);
}

}  // namespace

extern "C" {

// [R8] default relaxation factor: optimal SOR omega for the lowest mode of the continuous operator on
// the (r,z) box, J0(j01 r/Lr) cos(kz z):  lambda = (j01/Lr)^2 + kz^2,  mu = 1 - lambda/(2/dr^2+2/dz^2),
// omega = 2/(1+sqrt(1-mu^2)).   Only + - * / sqrt.
double sno_default_omega(int nr, int nz, double dr, double dz, int symmetry) {
    const double Lr = (nr + 0.5) * dr;
    const double kz = symmetry == 1 ? PI / (2.0 * ((nz + 0.5) * dz)) : PI / ((nz + 1.0) * dz);
    const double a = J01 / Lr;
    const double lambda = a * a + kz * kz;
    const double D = 2.0 / (dr * dr) + 2.0 / (dz * dz);
    const double mu = 1.0 - lambda / D;
    return 2.0 / (1.0 + std::sqrt(1.0 - mu * mu));
}

void sno_regular_harmonics(double x, double y, int lmax, double* R) { regular_harmonics(x, y, lmax, R); }
void sno_irregular_harmonics(double x, double y, int lmax, double* I) { irregular_harmonics(x, y, lmax, I); }

// Step a-1 [NS (a)]: multipole moments about the origin, midpoint rule per cell [R5,R6],
//   M_l = sum_cells rho_ij (s_ij/L0)^l P_l(z_j/s_ij) dV_i,   dV_i = 2 pi r_i dr dz.
// symmetry=1: the mirrored half z<0 contributes (-1)^l times the same, so odd l vanish and even l double.
// M has lmax+1 entries (odd entries are 0 when symmetry=1).  l=0 is the "M" of the paper's Roche
// formula.  Accumulation in long double so the sum itself carries no visible rounding.
int sno_moments(int nr, int nz, double dr, double dz, int symmetry, int lmax, const double* rho, double* M) {
    if (nr < 1 || nz < 1 || lmax < 0 || !rho || !M) return -1;
    const Grid g = make_grid(nr, nz, dr, dz, symmetry);
    std::vector<long double> acc(lmax + 1, 0.0L);
    std::vector<double> R(lmax + 2);
    for (int j = 0; j < nz; ++j) {
        const double y = g.z(j) / g.L0;
        for (int i = 0; i < nr; ++i) {
            const double x = g.r(i) / g.L0;
            const double dV = 2.0 * PI * g.r(i) * dr * dz;
            const double w = rho[(size_t)j * nr + i] * dV;
            regular_harmonics(x, y, lmax, R.data());
            for (int l = 0; l <= lmax; ++l) acc[l] += (long double)(w * R[l]);
        }
    }
    for (int l = 0; l <= lmax; ++l) {
        if (symmetry == 1) M[l] = (l & 1) ? 0.0 : (double)(2.0L * acc[l]);
        else M[l] = (double)acc[l];
    }
    return 0;
}

// Step a-1b: exterior multipole potential at the ghost-cell centres one cell outside the grid [R4,R5],
//   phi_b(r,z) = -(1/L0) sum_l M_l P_l(cos theta) / shat^(l+1).
// bE[nz]: r = (nr+1/2) dr, z = z_j.  bN[nr]: r = r_i, z = z_{nz-1} + dz.  bS[nr] (symmetry=0 only):
// r = r_i, z = z_0 - dz.   With lmax = 0 this is the paper's Roche boundary -GM/sqrt(r^2+z^2), G = 1.
int sno_boundary(int nr, int nz, double dr, double dz, int symmetry, int lmax, const double* M,
                 double* bE, double* bN, double* bS) {
    if (nr < 1 || nz < 1 || lmax < 0 || !M || !bE || !bN) return -1;
    const Grid g = make_grid(nr, nz, dr, dz, symmetry);
    std::vector<double> I(lmax + 2);
    auto phi_b = [&](double r, double z) {
        irregular_harmonics(r / g.L0, z / g.L0, lmax, I.data());
        double sum = 0.0;
        for (int l = 0; l <= lmax; ++l) sum += M[l] * I[l];
        return -sum / g.L0;
    };
    const double rE = (nr + 0.5) * dr;
    for (int j = 0; j < nz; ++j) bE[j] = phi_b(rE, g.z(j));
    const double zN = g.z(nz - 1) + dz;
    for (int i = 0; i < nr; ++i) bN[i] = phi_b(g.r(i), zN);
    if (symmetry == 0 && bS) {
        const double zS = g.z(0) - dz;
        for (int i = 0; i < nr; ++i) bS[i] = phi_b(g.r(i), zS);
    }
    return 0;
}

// Steps a-2 + a-3: nsweeps red-black SOR sweeps in place [R1,R3,R7,R10].
// Conservative cell-centred 5-point cylindrical Laplacian [R1]:
//   (1/r_i)[r_{i+1/2}(p_{i+1,j}-p_{i,j}) - r_{i-1/2}(p_{i,j}-p_{i-1,j})]/dr^2 + (p_{i,j+1}-2p_{i,j}+p_{i,j-1})/dz^2 = 4 pi rho
//   => cE_i = (i+1)/(i+1/2)/dr^2, cW_i = i/(i+1/2)/dr^2 (cW_0 = 0: the regular/reflecting axis needs no ghost),
//      cN = cS = 1/dz^2, diag = 2/dr^2 + 2/dz^2.
// Reflecting equator (symmetry=1): ghost p_{i,-1} == p_{i,0} eliminated algebraically on row 0 [R3]:
//   cS = 0, diag = 2/dr^2 + 1/dz^2.
// One sweep = all cells with (i+j) even ("red"), then all with (i+j) odd ("black") [R7].
// Pinned arithmetic [R10]:  t = cE*pE; t = fma(cW,pW,t); t = fma(cN,pN,t); t = fma(cS,pS,t); t = fma(-diag,pC,t);
//   res = f - t;  pC <- fma(-(omega/diag), res, pC),  f = FOURPI*rho.
// Per sweep k (1-based) records Rabs[k-1] = max |res| seen (pre-update, both colours) and
// P[k-1] = max |p_new| [R9].  bS is ignored when symmetry=1.
int sno_sweeps_chg(int nr, int nz, double dr, double dz, int symmetry, double omega, const double* rho,
                   const double* bE, const double* bN, const double* bS, double* phi, int nsweeps,
                   double* Rabs_hist, double* P_hist, double* Chg_hist);

int sno_sweeps(int nr, int nz, double dr, double dz, int symmetry, double omega, const double* rho,
               const double* bE, const double* bN, const double* bS, double* phi, int nsweeps,
               double* Rabs_hist, double* P_hist) {
    return sno_sweeps_chg(nr, nz, dr, dz, symmetry, omega, rho, bE, bN, bS, phi, nsweeps, Rabs_hist, P_hist, nullptr);
}

// The same sweeps; additionally Chg[k-1] = max over the cells of |w_j * res| [R16]: the change of phi the update of
// sweep k applies to a cell is dphi = -(omega/diag_j) res (the update is phi <- fma(-w_j, res, phi))
// "relative changes of all grids".
int sno_sweeps_chg(int nr, int nz, double dr, double dz, int symmetry, double omega, const double* rho,
                   const double* bE, const double* bN, const double* bS, double* phi, int nsweeps,
                   double* Rabs_hist, double* P_hist, double* Chg_hist) {
    if (nr < 1 || nz < 1 || !rho || !bE || !bN || !phi || (symmetry == 0 && !bS)) return -1;
    const double ir2 = 1.0 / (dr * dr);
    const double iz2 = 1.0 / (dz * dz);
    const double D = 2.0 * ir2 + 2.0 * iz2;
    const double D0 = D - iz2;
    const double wD = omega / D;
    const double wD0 = omega / D0;
    std::vector<double> cE(nr), cW(nr);
    for (int i = 0; i < nr; ++i) {
        cE[i] = ((i + 1.0) / (i + 0.5)) * ir2;
        cW[i] = (i / (i + 0.5)) * ir2;
    }
    for (int k = 0; k < nsweeps; ++k) {
        double Rabs = 0.0, P = 0.0, Chg = 0.0;
        for (int colour = 0; colour < 2; ++colour) {
            for (int j = 0; j < nz; ++j) {
                const bool mirror_row = (symmetry == 1 && j == 0);
                const double cS = mirror_row ? 0.0 : iz2;
                const double diag = mirror_row ? D0 : D;
                const double w = mirror_row ? wD0 : wD;
                for (int i = (j + colour) & 1; i < nr; i += 2) {
                    const size_t c = (size_t)j * nr + i;
                    const double pC = phi[c];
                    const double pE = (i + 1 < nr) ? phi[c + 1] : bE[j];
                    const double pW = (i > 0) ? phi[c - 1] : 0.0;
                    const double pN = (j + 1 < nz) ? phi[c + nr] : bN[i];
                    const double pS = (j > 0) ? phi[c - nr] : (symmetry == 1 ? 0.0 : bS[i]);
                    const double f = FOURPI * rho[c];
                    double t = cE[i] * pE;
                    t = std::fma(cW[i], pW, t);
                    t = std::fma(iz2, pN, t);
                    t = std::fma(cS, pS, t);
                    t = std::fma(-diag, pC, t);
                    const double res = f - t;
                    const double pnew = std::fma(-w, res, pC);
                    phi[c] = pnew;
                    const double ares = std::fabs(res), apn = std::fabs(pnew);
                    if (ares > Rabs || ares != ares) Rabs = ares;
                    if (apn > P || apn != apn) P = apn;
                    const double achg = std::fabs(w * res);
                    if (achg > Chg || achg != achg) Chg = achg;
                }
            }
        }
        if (Rabs_hist) Rabs_hist[k] = Rabs;
        if (P_hist) P_hist[k] = P;
        if (Chg_hist) Chg_hist[k] = Chg;
    }
    return 0;
}

// [R9] stopping ratio of sweep k:  R_k = Rabs_k / (max|f| + Dfull * P_k),  Dfull = 2/dr^2 + 2/dz^2.
// This is the paper's "relative changes of all grids" test in residual units
// (max|dphi| = (omega/diag) max|res|), normalised so that fp64 rounding cannot hold it above tol.
// Rabs_k == 0 gives 0 (also for rho == 0, phi == 0).
double sno_ratio(double Rabs, double P, double maxf, double dr, double dz) {
    if (Rabs == 0.0) return 0.0;
    const double Dfull = 2.0 * (1.0 / (dr * dr)) + 2.0 * (1.0 / (dz * dz));
    return Rabs / std::fma(Dfull, P, maxf);
}

// The whole path: moments -> boundary -> sweeps until R_k <= tol (tol > 0) or max_sweeps; tol <= 0 runs
// exactly max_sweeps.  omega <= 0 selects the default formula.  If bE_in is non-NULL the ghost arrays are
// taken from the caller (test hook mirroring sn_poisson_set_boundary) and the moment step is skipped.
// Outputs: *sweeps (full sweeps applied), *residual (R_k of the last sweep), hist[k] = R_{k+1} (nullable,
// max_sweeps entries).  Returns 0 converged / fixed-sweep completed, 1 hit max_sweeps, -1 bad args, -3 non-finite.
int sno_solve_rule(int rule, int nr, int nz, double dr, double dz, int symmetry, int lmax, double omega,
                   const double* rho, double* phi, double tol, int max_sweeps, int* sweeps, double* residual,
                   double* hist, const double* bE_in, const double* bN_in, const double* bS_in);

int sno_solve(int nr, int nz, double dr, double dz, int symmetry, int lmax, double omega, const double* rho,
              double* phi, double tol, int max_sweeps, int* sweeps, double* residual, double* hist,
              const double* bE_in, const double* bN_in, const double* bS_in) {
    return sno_solve_rule(0, nr, nz, dr, dz, symmetry, lmax, omega, rho, phi, tol, max_sweeps, sweeps, residual, hist,
                          bE_in, bN_in, bS_in);
}

// [R16] the paper-literal stopping rule (rule = 1): "The iteration is stopped by default when the relative
// changes of all grids reach below 1e-8":  E_k = max|dphi| / max|phi_new| of sweep k, stop after the first sweep with
// E_k <= tol; max|dphi| == 0 gives 0.  rule = 0 is the residual rule R9 above.  `residual` / hist hold E_k then.
double sno_relchange(double Chg, double P) {
    if (Chg == 0.0) return 0.0;
    return Chg / P;
}

int sno_solve_rule(int rule, int nr, int nz, double dr, double dz, int symmetry, int lmax, double omega,
                   const double* rho, double* phi, double tol, int max_sweeps, int* sweeps, double* residual,
                   double* hist, const double* bE_in, const double* bN_in, const double* bS_in) {
    if (rule != 0 && rule != 1) return -1;
    if (nr < 2 || nz < 2 || !(dr > 0) || !(dz > 0) || (symmetry != 0 && symmetry != 1) || lmax < 0 ||
        !rho || !phi || max_sweeps < 0 || !sweeps || !residual)
        return -1;
    std::vector<double> M(lmax + 1), bE(nz), bN(nr), bS(nr, 0.0);
    if (bE_in) {
        std::memcpy(bE.data(), bE_in, sizeof(double) * nz);
        std::memcpy(bN.data(), bN_in, sizeof(double) * nr);
        if (symmetry == 0 && bS_in) std::memcpy(bS.data(), bS_in, sizeof(double) * nr);
    } else {
        sno_moments(nr, nz, dr, dz, symmetry, lmax, rho, M.data());
        sno_boundary(nr, nz, dr, dz, symmetry, lmax, M.data(), bE.data(), bN.data(), bS.data());
    }
    if (!(omega > 0)) omega = sno_default_omega(nr, nz, dr, dz, symmetry);
    double maxf = 0.0;
    for (size_t c = 0; c < (size_t)nr * nz; ++c) {
        const double a = std::fabs(FOURPI * rho[c]);
        if (a > maxf) maxf = a;
    }
    *sweeps = 0;
    *residual = 0.0;
    for (int k = 0; k < max_sweeps; ++k) {
        double Rabs, P, Chg;
        sno_sweeps_chg(nr, nz, dr, dz, symmetry, omega, rho, bE.data(), bN.data(), bS.data(), phi, 1, &Rabs, &P, &Chg);
        const double Rk = rule == 0 ? sno_ratio(Rabs, P, maxf, dr, dz) : sno_relchange(Chg, P);
        *sweeps = k + 1;
        *residual = Rk;
        if (hist) hist[k] = Rk;
        if (!(Rk == Rk) || std::isinf(Rk)) return -3;
        if (tol > 0 && Rk <= tol) return 0;
    }
    return tol > 0 ? 1 : 0;
}

// Test helper: y = L(phi) with the ghosts folded in (the discrete operator of sno_sweeps, plain arithmetic).
int sno_apply_operator(int nr, int nz, double dr, double dz, int symmetry, const double* phi, const double* bE,
                       const double* bN, const double* bS, double* out) {
    const double ir2 = 1.0 / (dr * dr), iz2 = 1.0 / (dz * dz);
    for (int j = 0; j < nz; ++j)
        for (int i = 0; i < nr; ++i) {
            const size_t c = (size_t)j * nr + i;
            const double cE = ((i + 1.0) / (i + 0.5)) * ir2, cW = (i / (i + 0.5)) * ir2;
            const double pE = (i + 1 < nr) ? phi[c + 1] : bE[j];
            const double pW = (i > 0) ? phi[c - 1] : 0.0;
            const double pN = (j + 1 < nz) ? phi[c + nr] : bN[i];
            const bool mirror_row = (symmetry == 1 && j == 0);
            const double pS = (j > 0) ? phi[c - nr] : (mirror_row ? phi[c] : bS[i]);
            out[c] = cE * (pE - phi[c]) - cW * (phi[c] - pW) + iz2 * (pN - phi[c]) - iz2 * (phi[c] - pS);
        }
    return 0;
}

// NEXT-1: the gravity field the momentum and energy equations use as source terms,
// PAPER.md:83-89, eqs. (2)-(4): -rho dPhi/dr, -rho dPhi/dz.  [R15] centred differences at the cell centres with the
// solver's own boundary handling: reflecting axis (phi_{-1,j} = phi_{0,j}), reflecting equator when symmetry = 1
// (phi_{i,-1} = phi_{i,0}), the Dirichlet ghosts bE / bN / bS elsewhere.  Pinned arithmetic: (lo - hi) * (0.5/d).
int sno_gravity(int nr, int nz, double dr, double dz, int symmetry, const double* phi, const double* bE,
                const double* bN, const double* bS, double* gr, double* gz) {
    const double hr = 0.5 / dr, hz = 0.5 / dz;
    for (int j = 0; j < nz; ++j)
        for (int i = 0; i < nr; ++i) {
            const size_t c = (size_t)j * nr + i;
            const double pE = (i + 1 < nr) ? phi[c + 1] : bE[j];
            const double pW = (i > 0) ? phi[c - 1] : phi[c];
            const double pN = (j + 1 < nz) ? phi[c + nr] : bN[i];
            const double pS = (j > 0) ? phi[c - nr] : (symmetry == 1 ? phi[c] : bS[i]);
            gr[c] = (pW - pE) * hr;
            gz[c] = (pS - pN) * hz;
        }
    return 0;
}

}  // extern "C"
