"""Pins of the multigrid oracle (oracle/mg_oracle.cpp, readings M1-M8) against things other
than itself: the dense direct solve and the stagnated SOR iterate (same fixed point), conservation of the restriction,
linear exactness of the prolongation, the extrapolated coarse Dirichlet factor, a vectorised numpy restatement of the
whole V-cycle written here, and the textbook property the variant exists for (grid-independent > 10x residual drop per
cycle).  CPU only."""
import numpy as np
import pytest

import oracle
import workloads as W


# ---- a vectorised numpy restatement of M1-M8 (independent of the oracle's C++: whole-array operations, padded arrays) --
class NpLevel:
    def __init__(s, nr, nz, dr, dz, sym, lev):
        s.nr, s.nz, s.sym = nr, nz, sym
        ir2, iz2 = 1 / dr ** 2, 1 / dz ** 2
        i = np.arange(nr)
        s.cE, s.cW, s.iz2 = ((i + 1.0) / (i + 0.5)) * ir2, (i / (i + 0.5)) * ir2, iz2
        s.D = 2 * ir2 + 2 * iz2
        s.diag, s.cS = np.full(nz, s.D), np.full(nz, iz2)
        if sym == 1:
            s.diag[0], s.cS[0] = s.D - iz2, 0.0
        s.beta = (1 - 2.0 ** -lev) / (1 + 2.0 ** -lev)
        jj, ii = np.meshgrid(np.arange(nz), np.arange(nr), indexing="ij")
        s.masks = [((ii + jj) & 1) == c for c in (0, 1)]

    def apply(s, phi, g):
        P = np.zeros((s.nz + 2, s.nr + 2))
        P[1:-1, 1:-1] = phi
        P[1:-1, -1] = g[0] - s.beta * phi[:, -1]
        P[-1, 1:-1] = g[1] - s.beta * phi[-1, :]
        if s.sym == 0:
            P[0, 1:-1] = g[2] - s.beta * phi[0, :]
        return (s.cE * P[1:-1, 2:] + s.cW * P[1:-1, :-2] + s.iz2 * P[2:, 1:-1] + s.cS[:, None] * P[:-2, 1:-1]
                - s.diag[:, None] * phi)

    def smooth(s, phi, f, n, g):
        for _ in range(n):
            for c in (0, 1):
                phi = np.where(s.masks[c], phi - (f - s.apply(phi, g)) / s.diag[:, None], phi)
        return phi


def np_restrict(res):
    r = np.arange(res.shape[1]) + 0.5
    wr = res * r
    return (wr[0::2, 0::2] + wr[0::2, 1::2] + wr[1::2, 0::2] + wr[1::2, 1::2]) / (2 * (r[0::2] + r[1::2]))


def np_prolong(Lc, e):
    nzc, nrc = e.shape
    E = np.zeros((nzc + 2, nrc + 2))
    E[1:-1, 1:-1] = e
    E[0, 1:-1] = e[0] if Lc.sym == 1 else -Lc.beta * e[0]
    E[-1, 1:-1] = -Lc.beta * e[-1]
    E[:, 0] = E[:, 1]
    E[:, -1] = -Lc.beta * E[:, -2]
    out = np.zeros((2 * nzc, 2 * nrc))
    for a, da in ((0, -1), (1, 1)):
        for b, db in ((0, -1), (1, 1)):
            out[a::2, b::2] = (9 * E[1:-1, 1:-1] + 3 * E[1:-1, 1 + db:nrc + 1 + db] + 3 * E[1 + da:nzc + 1 + da, 1:-1]
                               + E[1 + da:nzc + 1 + da, 1 + db:nrc + 1 + db]) / 16
    return out


def np_vcycle(Ls, l, phi, f, g, nu1, nu2, nc):
    L = Ls[l]
    if l == len(Ls) - 1:
        return L.smooth(phi, f, nc if l else nu1 + nu2, g)
    phi = L.smooth(phi, f, nu1, g)
    fc = np_restrict(f - L.apply(phi, g))
    ec = np_vcycle(Ls, l + 1, np.zeros_like(fc), fc, (0.0, 0.0, 0.0), nu1, nu2, nc)
    return L.smooth(phi + np_prolong(Ls[l + 1], ec), f, nu2, g)


def np_mg_solve(w, ghosts, tol, max_cycles, nu1=1, nu2=1, nc=12):
    nr, nz, dr, dz = w.nr, w.nz, w.dr, w.dz
    Ls = []
    while True:
        Ls.append(NpLevel(nr, nz, dr, dz, w.symmetry, len(Ls)))
        if nr % 2 or nz % 2 or nr // 2 < 4 or nz // 2 < 4:
            break
        nr, nz, dr, dz = nr // 2, nz // 2, 2 * dr, 2 * dz
    f = 12.566370614359172 * w.rho
    phi, hist = np.zeros_like(f), []
    for _ in range(max_cycles):
        phi = np_vcycle(Ls, 0, phi, f, ghosts, nu1, nu2, nc)
        hist.append(np.abs(f - Ls[0].apply(phi, ghosts)).max() / (np.abs(f).max() + Ls[0].D * np.abs(phi).max()))
        if hist[-1] <= tol:
            break
    return phi, hist, len(Ls)


def ghosts_of(w):
    M = oracle.moments(w.rho, w.dr, w.dz, w.symmetry, w.lmax)
    bE, bN, bS = oracle.boundary(w.nr, w.nz, w.dr, w.dz, w.symmetry, w.lmax, M)
    return bE, bN, (bS if bS is not None else np.zeros(w.nr))


# ---- pins --------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("make", [lambda: W.random_smooth(32, 48, 1, 3), lambda: W.random_smooth(40, 24, 0, 4),
                                  lambda: W.cfg1(64), lambda: W.cfg3(64).first])
@pytest.mark.parametrize("nu", [(1, 1), (2, 1)])
def test_numpy_restatement_gives_the_same_iterates(make, nu):
    w = make()
    g = ghosts_of(w)
    want_phi, want_hist, nlev = np_mg_solve(w, g, 1e-10, 30, *nu)
    got = oracle.mg_solve(w.rho, np.zeros_like(w.rho), w.dr, w.dz, w.symmetry, w.lmax, 1e-10, 30, *nu)
    assert oracle.mg_levels(w.nr, w.nz) == nlev and nlev >= 3
    assert got["cycles"] == len(want_hist) and got["status"] == 0
    want_hist = np.array(want_hist)
    big = want_hist > 1e-9                           # below that the ratio feels the rounding of the two evaluation orders
    assert np.allclose(got["history"][big], want_hist[big], rtol=1e-5)
    assert np.allclose(got["history"][~big], want_hist[~big], rtol=0.2)
    assert np.abs(got["phi"] - want_phi).max() <= 1e-12 * np.abs(want_phi).max()


def test_fixed_point_is_the_direct_solution_and_the_sor_fixed_point():
    for w in (W.random_smooth(16, 16, 1, 5), W.random_smooth(12, 16, 0, 6)):
        g = ghosts_of(w)
        got = oracle.mg_solve(w.rho, np.zeros_like(w.rho), w.dr, w.dz, w.symmetry, w.lmax, 0.0, 40)     # to stagnation
        # dense direct solve of the assembled system (face by face, ghost terms on the right-hand side)
        n = w.nr * w.nz
        A, b = np.zeros((n, n)), (12.566370614359172 * w.rho).ravel().copy()
        ir2, iz2 = 1 / w.dr ** 2, 1 / w.dz ** 2
        for j in range(w.nz):
            for i in range(w.nr):
                k = j * w.nr + i
                cE, cW = (i + 1.0) / (i + 0.5) * ir2, i / (i + 0.5) * ir2
                A[k, k] -= cE + cW
                if i + 1 < w.nr: A[k, k + 1] += cE
                else: b[k] -= cE * g[0][j]
                if i > 0: A[k, k - 1] += cW
                A[k, k] -= iz2
                if j + 1 < w.nz: A[k, k + w.nr] += iz2
                else: b[k] -= iz2 * g[1][i]
                if j > 0: A[k, k] -= iz2; A[k, k - w.nr] += iz2
                elif w.symmetry == 0: A[k, k] -= iz2; b[k] -= iz2 * g[2][i]
        exact = np.linalg.solve(A, b).reshape(w.nz, w.nr)
        assert np.abs(got["phi"] - exact).max() <= 5e-13 * np.abs(exact).max()
        sor = oracle.solve(w.rho, np.zeros_like(w.rho), w.dr, w.dz, w.symmetry, w.lmax, 0.0, 3000)
        assert np.abs(got["phi"] - sor["phi"]).max() <= 5e-13 * np.abs(exact).max()


def test_restriction_conserves_the_volume_integral_and_constants():
    rng = np.random.default_rng(2)
    res = rng.standard_normal((12, 20))
    rc = oracle.mg_restrict(res)
    rf, rcw = np.arange(20) + 0.5, 2.0 * (np.arange(10) + 0.5)          # r in units of the FINE dr
    # volumes: fine r_i dr dz, coarse r_I (2 dr)(2 dz)
    assert abs((res * rf).sum() - 4.0 * (rc * rcw).sum()) <= 1e-13 * np.abs(res * rf).sum()
    assert np.allclose(oracle.mg_restrict(np.full((8, 8), 3.25)), 3.25, rtol=1e-15)
    assert np.allclose(rc, np_restrict(res), rtol=1e-14)


def test_prolongation_is_exact_for_linear_functions_inside_and_mirrors_at_the_axis():
    nzc, nrc = 6, 7
    I, J = np.meshgrid(np.arange(nrc), np.arange(nzc))
    xc, yc = 2.0 * (I + 0.5), 2.0 * (J + 0.5)
    ec = 1.5 + 0.25 * xc - 0.75 * yc
    out = oracle.mg_prolong(ec, 0, 1)
    i, j = np.meshgrid(np.arange(2 * nrc), np.arange(2 * nzc))
    want = 1.5 + 0.25 * (i + 0.5) - 0.75 * (j + 0.5)
    assert np.abs(out - want)[2:-2, 2:-2].max() < 1e-13              # bilinear interpolation reproduces linear functions
    # axis: the ghost mirrors, so a function of z only is reproduced in the first fine columns too
    ez = np.tile((0.5 * yc[:, :1]), (1, nrc))
    assert np.abs(oracle.mg_prolong(ez, 0, 1)[2:-2, :2] - 0.5 * (j[2:-2, :2] + 0.5)).max() < 1e-13
    # equator mirror (symmetry = 1): a function of r only is reproduced in the first fine rows
    er = np.tile(0.125 * xc[:1, :], (nzc, 1))
    assert np.abs(oracle.mg_prolong(er, 1, 1)[:2, 2:-2] - 0.125 * (i[:2, 2:-2] + 0.5)).max() < 1e-13
    assert np.allclose(oracle.mg_prolong(ec, 1, 2), np_prolong(NpLevel(nrc, nzc, 1, 1, 1, 2), ec), rtol=1e-14)


def test_coarse_dirichlet_factor_puts_the_zero_at_the_fine_ghost_centre():
    """M2: on level l the line through (last cell centre, e) and (ghost centre, -beta_l e) vanishes half a FINE cell
    outside the grid, for every l."""
    for l in range(0, 9):
        h = 2.0 ** l                                                   # coarse spacing in fine cells
        x_last, x_ghost, beta = -0.5 * h, 0.5 * h, oracle.mg_beta(l)   # distances from the domain edge
        zero = x_last + (x_ghost - x_last) * 1.0 / (1.0 + beta)        # e + (x - x_last)/(h) (-beta e - e) = 0
        assert abs(zero - 0.5) < 1e-12


@pytest.mark.parametrize("sym", [1, 0])
def test_textbook_multigrid_convergence_independent_of_the_grid(sym):
    cycles = []
    for n in (32, 64, 128, 256):
        w = W.cfg1(n) if sym == 1 else W.cfg3(n).first
        r = oracle.mg_solve_workload(w)
        assert r["status"] == 0 and r["residual"] <= 1e-10
        rates = r["history"][1:] / r["history"][:-1]
        assert rates.max() < 0.2 and np.exp(np.log(rates).mean()) < 0.1, rates      # > 10x per V(1,1) cycle on average
        cycles.append(r["cycles"])
    assert max(cycles) - min(cycles) <= 2 and max(cycles) <= 10, cycles


def test_counting_and_status():
    w = W.cfg1(64)
    r = oracle.mg_solve_workload(w)
    k = r["cycles"]
    assert r["history"][-1] <= 1e-10 < r["history"][-2]                # first crossing
    short = oracle.mg_solve(w.rho, np.zeros_like(w.rho), w.dr, w.dz, w.symmetry, w.lmax, 1e-10, k - 1)
    assert short["status"] == 1 and short["cycles"] == k - 1
    assert np.array_equal(short["history"], r["history"][:-1])
    fixed = oracle.mg_solve(w.rho, np.zeros_like(w.rho), w.dr, w.dz, w.symmetry, w.lmax, 0.0, 3)
    assert fixed["status"] == 0 and fixed["cycles"] == 3
    # warm start from the converged iterate: one cycle suffices
    warm = oracle.mg_solve(w.rho, r["phi"], w.dr, w.dz, w.symmetry, w.lmax, 1e-10, 10)
    assert warm["cycles"] == 1
