// levelset_oracle.cpp -- CPU oracle of the level-set re-initialisation.
//
// TEST INFRASTRUCTURE, NOT THE PRODUCT.  Plain, slow, single-threaded fp64; shares no code with
// paper_1507_08549_b200/; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// load it.
//
// PAPER.md:131 (section 2.2): "First, we enumerate all positions where the flame front cut the grid, by finding all
// neighboring pairs of the scalar field where its values are of opposite signs.  The position of the flame front is
// obtained by linear interpolation.  Then the distances of all grid points to the flame front positions are compared,
// and the smallest one is chosen as the new value of S."  PAPER.md:133-141, eqs. (6)-(7):
//     S_new = H(d) S_old + (1 - H(d)) d,   H(d) = (1 - tanh((d - d0)/(Delta/3))) / (1 - tanh(-d0/(Delta/3))),  d0 = 3 Delta,
// "the values of S on the three closest neighboring grids around the flame front are unchanged".
// "the scalar field is defined on the corners of a grid".
//
// Readings where the paper is silent (L1..L6):
//   L1  nodes: S[j][i] lives at the cell corner (x_i, y_j) = (i dr, j dz), i in [0, nx), j in [0, ny) (nx = nr + 1 ...).
//   L2  "neighboring pairs": the two grid edges leaving a node towards +x and +y (every edge once).  "opposite signs":
//       one value < 0 and the other >= 0 (S >= 0 is ash; a node with S == 0 is itself a crossing of its edges).
//   L3  crossing of the edge a -> b of length h:  t = S_a / (S_a - S_b),  position = fma(t, h, x_a)   (linear interpolation).
//   L4  d_min = sqrt(min over crossings of (dx*dx + dy*dy)) with dd = fma(dy, dy, dx*dx); the distance carries the sign
//       of S_old ("positive (negative) values of S to be full of ash (fuel)"): d = copysign(d_min, S_old).
//   L5  H is evaluated at the unsigned d_min; Delta is an argument (the paper's cells are square: Delta = dr = dz).
//   L6  no crossing anywhere: S is returned unchanged and the count is 0.  Only crossings inside the grid count (no
//       mirror images across the axis or the equator).
//
// Pins (tests/test_levelset_pins.py): a circle of radius R (exact signed distance in, exact signed distance out to
// O(Delta^2)), a tilted straight line (linear interpolation is exact for a linear S: every crossing lies on the line, so
// d equals the distance to the nearest crossing and is bounded by the exact point-line distance from below), nodes
// within 3 Delta of the front unchanged to < 1e-7 relative, far nodes equal to the distance, the
// crossing list against a brute-force pure-Python enumeration, H(0) = 1, H(inf) = 0, idempotence on an exact distance
// field away from kinks.
#include <cmath>
#include <cstddef>
#include <limits>
#include <vector>

extern "C" {

// H(d) of eq. (7).
double lso_H(double d, double delta) {
    const double d0 = 3.0 * delta, w = delta / 3.0;
    return (1.0 - std::tanh((d - d0) / w)) / (1.0 - std::tanh(-d0 / w));
}

// Enumerate the crossings [L2, L3] in the order: for j, for i: edge (i,j)-(i+1,j), then edge (i,j)-(i,j+1).
// cx, cy: capacity 2*nx*ny each (may be NULL to count only).  Returns the number of crossings.
long lso_crossings(int nx, int ny, double dr, double dz, const double* S, double* cx, double* cy) {
    long n = 0;
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            const double sa = S[(size_t)j * nx + i];
            const double xa = i * dr, ya = j * dz;
            if (i + 1 < nx) {
                const double sb = S[(size_t)j * nx + i + 1];
                if ((sa < 0.0) != (sb < 0.0)) {
                    const double t = sa / (sa - sb);
                    if (cx) { cx[n] = std::fma(t, dr, xa); cy[n] = ya; }
                    ++n;
                }
            }
            if (j + 1 < ny) {
                const double sb = S[(size_t)(j + 1) * nx + i];
                if ((sa < 0.0) != (sb < 0.0)) {
                    const double t = sa / (sa - sb);
                    if (cx) { cx[n] = xa; cy[n] = std::fma(t, dz, ya); }
                    ++n;
                }
            }
        }
    return n;
}

// The whole re-initialisation.  S_new may alias nothing.  dist (nullable) receives the signed distance d [L4].
// Returns the number of crossings (0: S_new = S_old [L6]), or -1 on bad arguments.
long lso_reinit(int nx, int ny, double dr, double dz, double delta, const double* S_old, double* S_new, double* dist) {
    if (nx < 2 || ny < 2 || !(dr > 0) || !(dz > 0) || !(delta > 0) || !S_old || !S_new) return -1;
    std::vector<double> cx((size_t)2 * nx * ny), cy((size_t)2 * nx * ny);
    const long nc = lso_crossings(nx, ny, dr, dz, S_old, cx.data(), cy.data());
    if (nc == 0) {
        for (size_t k = 0; k < (size_t)nx * ny; ++k) {
            S_new[k] = S_old[k];
            if (dist) dist[k] = std::copysign(std::numeric_limits<double>::infinity(), S_old[k]);
        }
        return 0;
    }
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            const double x = i * dr, y = j * dz;
            double best = std::numeric_limits<double>::infinity();
            for (long c = 0; c < nc; ++c) {
                const double dx = x - cx[c], dy = y - cy[c];
                const double dd = std::fma(dy, dy, dx * dx);
                if (dd < best) best = dd;
            }
            const double dmin = std::sqrt(best);
            const double so = S_old[(size_t)j * nx + i];
            const double d = std::copysign(dmin, so);
            const double h = lso_H(dmin, delta);
            S_new[(size_t)j * nx + i] = h * so + (1.0 - h) * d;
            if (dist) dist[(size_t)j * nx + i] = d;
        }
    return nc;
}

}  // extern "C"
