// mg_oracle.cpp -- CPU oracle of the red-black-smoothed multigrid variant of the Poisson solve (SURVEY.md section 8f,
// NEXT-4: "faster-converging variants on the same stencil ... red-black-smoothed multigrid"; not in the paper, which
// solves the same equation by SOR).
//
// TEST INFRASTRUCTURE, NOT THE PRODUCT.  Plain, slow, single-threaded fp64; shares no code with
// paper_1507_08549_b200/; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// load it.
//
// Same equation, same discretisation, same ghosts, same fixed point as oracle/sn_oracle.cpp (DESIGN.md section 2,
// readings R1-R10); only the ITERATION differs.  The algorithm is the textbook geometric V-cycle, step by step, on
// cell-centred grids (readings M1..M8):
//   M1  levels l = 0 .. L-1: (nr / 2^l) x (nz / 2^l) cells of size (2^l dr) x (2^l dz); a level is coarsened while both
//       of its cell counts are even and the coarser level keeps >= 4 cells per axis.
//   M2  operator on level l: the conservative 5-point stencil of R1 / R3 with that level's spacing (rediscretisation):
//       cE_i = ((i+1)/(i+1/2)) / dr_l^2, cW_i = (i/(i+1/2)) / dr_l^2, cN = cS = 1/dz_l^2, reflecting equator eliminated
//       (symmetry = 1).  Outer ghosts: level 0 takes the multipole ghosts bE / bN / bS; on level l >= 1 the unknown is an
//       ERROR, whose Dirichlet zero sits at the level-0 ghost centre, half a FINE cell outside the grid, not half a coarse
//       cell: linear extrapolation through that zero gives  ghost = -beta_l * (adjacent interior value),
//       beta_l = (1 - 2^-l) / (1 + 2^-l)   (beta_0 = 0).  Without it the V-cycle degrades with every level added.
//   M3  smoother: red-black Gauss-Seidel (red = (i+j) even first), the pinned update of R10 with omega = 1:
//       t = cE pE; t = fma(cW,pW,t); t = fma(cN,pN,t); t = fma(cS,pS,t); t = fma(-diag,pC,t); res = f - t;
//       pC = fma(-(1/diag), res, pC); a ghost that depends on pC (M2) is evaluated with the old pC.  nu1 sweeps before,
//       nu2 after the coarse-grid correction (defaults 1, 1).
//   M4  residual: res = f - t with the same tree.
//   M5  restriction (volume weighted, the volume of a cell is proportional to r_i = i + 1/2):
//       f_c(I,J) = ((r_a res(a,2J) + r_b res(b,2J)) + (r_a res(a,2J+1) + r_b res(b,2J+1))) / (2 (r_a + r_b)), a = 2I, b = 2I+1.
//   M6  coarsest level: nc red-black Gauss-Seidel sweeps from zero (default 12: 10 already give the cycle count of 30,
//       below 8 the V-cycle degrades -- the coarsest grid with its reflecting sides relaxes slowly).
//   M7  prolongation: bilinear, e_f(2I+a, 2J+b) = (((9 C + 3 H) + 3 V) + Dg) / 16 with H / V / Dg the coarse neighbours
//       towards the fine cell; the coarse error is extended by one ghost layer: reflected at the axis (and at the equator
//       when symmetry = 1), -beta_{l+1} times the edge value at the outer edges (rows first, then columns, so a corner
//       ghost is the column rule applied to the extended row).  phi_f += e_f.
//   M8  one cycle = one V-cycle from level 0.  After every cycle: res = f - A phi on level 0 (the TRUE residual of the
//       iterate), R = max|res| / fma(D, max|phi|, max|f|) (the ratio of R9); stop after the first cycle with R <= tol, or
//       at max_cycles.  `cycles` plays the role of `sweeps`.
//
// Pins (tests/test_mg_pins.py): the converged iterate equals the dense direct solve of the assembled system and the
// stagnated SOR iterate of sn_oracle.cpp (same fixed point); restriction conserves the volume integral; prolongation
// is exact for linear functions away from the edges; a vectorised numpy restatement of M1-M8 written in the test gives
// the same iterates and cycle counts; the residual drops by > 10x per V(1,1) cycle independently of the grid size (the
// textbook property this variant exists for).
#include <cmath>
#include <cstddef>
#include <vector>

namespace {

const double FOURPI = 12.566370614359172;

struct Level {
    int nr, nz, symmetry;
    double iz2, D, D0, beta;
    std::vector<double> cE, cW, phi, f;
};

Level make_level(int nr, int nz, double dr, double dz, int symmetry, int l) {
    Level L;
    L.nr = nr; L.nz = nz; L.symmetry = symmetry;
    const double ir2 = 1.0 / (dr * dr);
    L.iz2 = 1.0 / (dz * dz);
    L.D = 2.0 * ir2 + 2.0 * L.iz2;
    L.D0 = L.D - L.iz2;
    const double s = std::ldexp(1.0, -l);                 // 2^-l
    L.beta = (1.0 - s) / (1.0 + s);
    L.cE.resize(nr); L.cW.resize(nr);
    for (int i = 0; i < nr; ++i) {
        L.cE[i] = ((i + 1.0) / (i + 0.5)) * ir2;
        L.cW[i] = (i / (i + 0.5)) * ir2;
    }
    return L;
}

// t = (A phi)(i,j) with the pinned tree; ghosts: level 0 from bE/bN/bS, else -beta * pC
inline double apply_at(const Level& L, const double* phi, int i, int j, const double* bE, const double* bN,
                       const double* bS, double* diag_out) {
    const int nr = L.nr, nz = L.nz;
    const size_t c = (size_t)j * nr + i;
    const bool mirror_row = (L.symmetry == 1 && j == 0);
    const double cS = mirror_row ? 0.0 : L.iz2;
    const double diag = mirror_row ? L.D0 : L.D;
    const double pC = phi[c];
    const double ghost = -(L.beta * pC);
    const double pE = (i + 1 < nr) ? phi[c + 1] : (bE ? bE[j] : ghost);
    const double pW = (i > 0) ? phi[c - 1] : 0.0;
    const double pN = (j + 1 < nz) ? phi[c + nr] : (bN ? bN[i] : ghost);
    const double pS = (j > 0) ? phi[c - nr] : (L.symmetry == 1 ? 0.0 : (bS ? bS[i] : ghost));
    double t = L.cE[i] * pE;
    t = std::fma(L.cW[i], pW, t);
    t = std::fma(L.iz2, pN, t);
    t = std::fma(cS, pS, t);
    t = std::fma(-diag, pC, t);
    *diag_out = diag;
    return t;
}

// f of level 0 is 4 pi rho (scale = FOURPI on rho), of a coarse level the restricted residual (scale = 1)
void smooth(Level& L, const double* src, double scale, int nsweeps, const double* bE, const double* bN, const double* bS) {
    const double wD = 1.0 / L.D, wD0 = 1.0 / L.D0;
    for (int k = 0; k < nsweeps; ++k)
        for (int colour = 0; colour < 2; ++colour)
            for (int j = 0; j < L.nz; ++j)
                for (int i = (j + colour) & 1; i < L.nr; i += 2) {
                    double diag;
                    const double t = apply_at(L, L.phi.data(), i, j, bE, bN, bS, &diag);
                    const size_t c = (size_t)j * L.nr + i;
                    const double res = scale * src[c] - t;
                    L.phi[c] = std::fma(-(diag == L.D ? wD : wD0), res, L.phi[c]);
                }
}

void residual(const Level& L, const double* src, double scale, const double* bE, const double* bN, const double* bS,
              std::vector<double>& res) {
    res.resize((size_t)L.nr * L.nz);
    for (int j = 0; j < L.nz; ++j)
        for (int i = 0; i < L.nr; ++i) {
            double diag;
            const double t = apply_at(L, L.phi.data(), i, j, bE, bN, bS, &diag);
            res[(size_t)j * L.nr + i] = scale * src[(size_t)j * L.nr + i] - t;
        }
}

void restrict_to(const Level& Lf, const std::vector<double>& res, Level& Lc) {
    for (int J = 0; J < Lc.nz; ++J)
        for (int I = 0; I < Lc.nr; ++I) {
            const int a = 2 * I, b = 2 * I + 1;
            const double ra = a + 0.5, rb = b + 0.5;
            const double* r0 = &res[(size_t)(2 * J) * Lf.nr];
            const double* r1 = &res[(size_t)(2 * J + 1) * Lf.nr];
            const double num = (ra * r0[a] + rb * r0[b]) + (ra * r1[a] + rb * r1[b]);
            Lc.f[(size_t)J * Lc.nr + I] = num / (2.0 * (ra + rb));
        }
}

// coarse error with its ghost layer (M7)
inline double ext(const Level& Lc, int I, int J) {
    double sign = 1.0;
    int i = I, j = J;
    if (j < 0) { j = 0; if (Lc.symmetry == 0) sign = -Lc.beta; }
    else if (j >= Lc.nz) { j = Lc.nz - 1; sign = -Lc.beta; }
    double v = Lc.phi[(size_t)j * Lc.nr + (i < 0 ? 0 : i >= Lc.nr ? Lc.nr - 1 : i)];
    v = sign == 1.0 ? v : sign * v;                              // rows first
    if (i >= Lc.nr) v = -Lc.beta * v;                            // then columns (the axis reflects: factor 1)
    return v;
}

void prolong_add(const Level& Lc, Level& Lf) {
    for (int j = 0; j < Lf.nz; ++j)
        for (int i = 0; i < Lf.nr; ++i) {
            const int I = i >> 1, J = j >> 1;
            const int di = (i & 1) ? 1 : -1, dj = (j & 1) ? 1 : -1;
            const double C = ext(Lc, I, J), H = ext(Lc, I + di, J), V = ext(Lc, I, J + dj), Dg = ext(Lc, I + di, J + dj);
            const double e = (((9.0 * C + 3.0 * H) + 3.0 * V) + Dg) * 0.0625;
            Lf.phi[(size_t)j * Lf.nr + i] += e;
        }
}

void vcycle(std::vector<Level>& Ls, size_t l, const double* rho, const double* bE, const double* bN, const double* bS,
            int nu1, int nu2, int nc) {
    Level& L = Ls[l];
    const double* src = l == 0 ? rho : L.f.data();
    const double scale = l == 0 ? FOURPI : 1.0;
    const double *gE = l == 0 ? bE : nullptr, *gN = l == 0 ? bN : nullptr, *gS = l == 0 ? bS : nullptr;
    if (l + 1 == Ls.size()) {
        smooth(L, src, scale, l == 0 ? nu1 + nu2 : nc, gE, gN, gS);     // a single level: plain Gauss-Seidel
        return;
    }
    smooth(L, src, scale, nu1, gE, gN, gS);
    std::vector<double> res;
    residual(L, src, scale, gE, gN, gS, res);
    Level& Lc = Ls[l + 1];
    restrict_to(L, res, Lc);
    for (double& v : Lc.phi) v = 0.0;
    vcycle(Ls, l + 1, rho, bE, bN, bS, nu1, nu2, nc);
    prolong_add(Lc, L);
    smooth(L, src, scale, nu2, gE, gN, gS);
}

}  // namespace

extern "C" {

// number of levels of an nr x nz grid (M1)
int mgo_levels(int nr, int nz) {
    int n = 1;
    while (nr % 2 == 0 && nz % 2 == 0 && nr / 2 >= 4 && nz / 2 >= 4) { nr /= 2; nz /= 2; ++n; }
    return n;
}

double mgo_beta(int l) {
    const double s = std::ldexp(1.0, -l);
    return (1.0 - s) / (1.0 + s);
}

// pins: one restriction / one prolongation between a fine level l_f (>= 0) and the next coarser one
int mgo_restrict(int nr, int nz, const double* res, double* out) {
    Level Lf = make_level(nr, nz, 1.0, 1.0, 0, 0), Lc = make_level(nr / 2, nz / 2, 2.0, 2.0, 0, 1);
    Lc.f.resize((size_t)(nr / 2) * (nz / 2));
    restrict_to(Lf, std::vector<double>(res, res + (size_t)nr * nz), Lc);
    for (size_t k = 0; k < Lc.f.size(); ++k) out[k] = Lc.f[k];
    return 0;
}
int mgo_prolong(int nrc, int nzc, int symmetry, int lc, const double* ec, double* out) {
    Level Lc = make_level(nrc, nzc, 2.0, 2.0, symmetry, lc), Lf = make_level(2 * nrc, 2 * nzc, 1.0, 1.0, symmetry, lc - 1);
    Lc.phi.assign(ec, ec + (size_t)nrc * nzc);
    Lf.phi.assign((size_t)4 * nrc * nzc, 0.0);
    prolong_add(Lc, Lf);
    for (size_t k = 0; k < Lf.phi.size(); ++k) out[k] = Lf.phi[k];
    return 0;
}

// The solve.  phi: initial guess in, iterate after `cycles` V-cycles out.  hist (may be NULL): R after every cycle.
// status: 0 converged (or tol <= 0: max_cycles cycles run), 1 max_cycles reached, -3 non-finite ratio.
int mgo_solve(int nr, int nz, double dr, double dz, int symmetry, const double* rho, const double* bE, const double* bN,
              const double* bS, double* phi, double tol, int max_cycles, int nu1, int nu2, int nc, int* cycles_out,
              double* R_out, double* hist) {
    if (nr < 1 || nz < 1 || !rho || !bE || !bN || !phi || (symmetry == 0 && !bS) || max_cycles < 0 || nu1 < 0 || nu2 < 0 ||
        nu1 + nu2 < 1 || nc < 1)
        return -1;
    const int nlev = mgo_levels(nr, nz);
    std::vector<Level> Ls;
    for (int l = 0; l < nlev; ++l) {
        Ls.push_back(make_level(nr >> l, nz >> l, std::ldexp(dr, l), std::ldexp(dz, l), symmetry, l));
        Ls.back().phi.assign((size_t)(nr >> l) * (nz >> l), 0.0);
        Ls.back().f.assign(l == 0 ? 0 : (size_t)(nr >> l) * (nz >> l), 0.0);
    }
    const size_t n = (size_t)nr * nz;
    Ls[0].phi.assign(phi, phi + n);
    double maxf = 0.0;
    for (size_t k = 0; k < n; ++k) {
        const double a = std::fabs(FOURPI * rho[k]);
        if (a > maxf || a != a) maxf = a;
    }
    int cycles = 0, status = tol > 0.0 ? 1 : 0;
    double R = 0.0;
    std::vector<double> res;
    while (cycles < max_cycles) {
        vcycle(Ls, 0, rho, bE, bN, bS, nu1, nu2, nc);
        ++cycles;
        residual(Ls[0], rho, FOURPI, bE, bN, bS, res);
        double Rabs = 0.0, P = 0.0;
        for (size_t k = 0; k < n; ++k) {
            const double a = std::fabs(res[k]), p = std::fabs(Ls[0].phi[k]);
            if (a > Rabs || a != a) Rabs = a;
            if (p > P || p != p) P = p;
        }
        R = Rabs == 0.0 ? 0.0 : Rabs / std::fma(Ls[0].D, P, maxf);
        if (hist) hist[cycles - 1] = R;
        if (!(R == R) || std::isinf(R)) { status = -3; break; }
        if (tol > 0.0 && R <= tol) { status = 0; break; }
    }
    for (size_t k = 0; k < n; ++k) phi[k] = Ls[0].phi[k];
    *cycles_out = cycles;
    *R_out = R;
    return status;
}

}  // extern "C"
