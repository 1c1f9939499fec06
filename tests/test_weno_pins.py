"""Pins of the WENO-5 / global Lax-Friedrichs oracle (oracle/weno_oracle.cpp) against
things other than itself: exact polynomial reconstruction, the classical linear weights, fifth-order convergence on a
smooth flow, conservation, a brute-force pure-Python restatement, mirror symmetry, and the paper's four shock tubes
(Table 3) against an exact Riemann solver written here (Toro's two-shock / rarefaction pressure
function, restated).  CPU only."""
import math

import numpy as np
import pytest

import oracle

GAMMA = 1.4


# ---- helpers -----------------------------------------------------------------------------------------------------------
def cons(rho, vr, vz, p, gamma=GAMMA):
    rho, vr, vz, p = (np.asarray(a, dtype=np.float64) for a in (rho, vr, vz, p))
    return np.stack([rho, rho * vr, rho * vz, p / (gamma - 1.0) + 0.5 * rho * (vr * vr + vz * vz)])


def cell_average(poly, lo, hi):
    """exact average of the polynomial (numpy poly1d) over [lo, hi]"""
    P = poly.integ()
    return (P(hi) - P(lo)) / (hi - lo)


# ---- the reconstruction (W5) -----------------------------------------------------------------------------------------
def test_candidates_reproduce_quadratics_and_the_linear_weights_give_fifth_order():
    rng = np.random.default_rng(1)
    h = 0.37
    edges = (np.arange(-2, 4) - 0.5) * h            # cells i-2 .. i+2 around x_i = 0; face at x = h/2
    for deg in range(5):
        poly = np.poly1d(rng.standard_normal(deg + 1))
        a, b, c, d, e = (cell_average(poly, edges[k], edges[k + 1]) for k in range(5))
        q, beta = oracle.weno_candidates(a, b, c, d, e)
        exact = poly(0.5 * h)
        if deg <= 2:                                 # every third-order candidate is exact
            assert np.allclose(q, exact, rtol=0, atol=1e-13 * (1 + abs(exact)))
        # the classical linear weights (1/10, 6/10, 3/10) give the fifth-order value, exact up to degree 4
        assert abs(0.1 * q[0] + 0.6 * q[1] + 0.3 * q[2] - exact) <= 1e-12 * (1 + abs(exact))


def test_smoothness_indicators_and_weights_on_known_data():
    # linear data: all three indicators equal (=1 for unit slope) -> the nonlinear weights ARE the linear ones
    q, beta = oracle.weno_candidates(0.0, 1.0, 2.0, 3.0, 4.0)
    assert np.array_equal(beta, [1.0, 1.0, 1.0])
    assert abs(oracle.weno5(0.0, 1.0, 2.0, 3.0, 4.0) - 2.5) < 1e-15
    # a step right of the face: the stencil that crosses it is switched off (ENO property)
    v = oracle.weno5(1.0, 1.0, 1.0, 1.0, 0.0)
    assert abs(v - 1.0) < 1e-6
    # a step left of cell c: only the rightmost stencil (c, d, e) is smooth
    v = oracle.weno5(0.0, 0.0, 1.0, 1.0, 1.0)
    assert abs(v - 1.0) < 1e-6
    # beta of a pure parabola x^2 sampled at -2..2 (typed by hand): stencil 0: s = 2, t = 4-4+0 = 0 ... use the formula's
    # own definition on integers: a..e = 4,1,0,1,4
    q, beta = oracle.weno_candidates(4.0, 1.0, 0.0, 1.0, 4.0)
    assert np.allclose(beta, [13.0 / 12.0 * 4 + 0.25 * 0.0, 13.0 / 12.0 * 4 + 0.0, 13.0 / 12.0 * 4 + 0.25 * 0.0])


def test_constant_state_has_zero_divergence_exactly():
    U = cons(np.full((5, 12), 1.3), 0.4, -0.7, 2.0)
    for bc in ([0, 0, 0, 0], [2, 2, 2, 2], [0, 0, 2, 2]):
        L = oracle.weno_rhs(U, 0.1, 0.2, GAMMA, bc)
        assert np.array_equal(L, np.zeros_like(L))
    # a wall at rest: reflecting boundaries keep a fluid at rest at rest
    U = cons(np.full((5, 12), 1.3), 0.0, 0.0, 2.0)
    assert np.abs(oracle.weno_rhs(U, 0.1, 0.2, GAMMA, [1, 1, 1, 1])).max() == 0.0


def _advection_error(n, axis):
    x = (np.arange(n) + 0.5) / n
    rho1 = 1.0 + 0.2 * np.sin(2 * np.pi * x)
    if axis == 0:
        rho = np.tile(rho1, (4, 1))
        U = cons(rho, 1.0, 0.0, 1.0)
        L = oracle.weno_rhs(U, 1.0 / n, 1.0 / n, GAMMA, [2, 2, 2, 2])
        got = L[0][0]
    else:
        rho = np.tile(rho1[:, None], (1, 4))
        U = cons(rho, 0.0, 1.0, 1.0)
        L = oracle.weno_rhs(U, 1.0 / n, 1.0 / n, GAMMA, [2, 2, 2, 2])
        got = L[0][:, 0]
    # exact: d(rho)/dt = -v d(rho)/dx; a finite-DIFFERENCE scheme approximates the POINT value of the derivative
    exact = -0.2 * 2 * np.pi * np.cos(2 * np.pi * x)
    return np.abs(got - exact).mean()


@pytest.mark.parametrize("axis", [0, 1])
def test_fifth_order_on_a_smooth_flow(axis):
    errs = [_advection_error(n, axis) for n in (20, 40, 80, 160)]
    ratios = [errs[k] / errs[k + 1] for k in range(3)]
    assert errs[-1] < 5e-8
    assert all(28.0 < r < 40.0 for r in ratios), (errs, ratios)       # 2^5 = 32: fifth order, not third, not sixth


def test_conservation_telescoping():
    rng = np.random.default_rng(3)
    nz, nr = 7, 11
    U = cons(1.0 + 0.3 * rng.random((nz, nr)), 0.4 * rng.standard_normal((nz, nr)), 0.4 * rng.standard_normal((nz, nr)),
             1.0 + 0.5 * rng.random((nz, nr)))
    dr, dz = 0.1, 0.13
    L = oracle.weno_rhs(U, dr, dz, GAMMA, [2, 2, 2, 2])
    assert np.abs(L.sum(axis=(1, 2))).max() < 1e-11            # periodic: the fluxes telescope to zero
    F, G = oracle.weno_face_fluxes(U, dr, dz, GAMMA, [0, 0, 0, 0])
    L = oracle.weno_rhs(U, dr, dz, GAMMA, [0, 0, 0, 0])
    want = -(F[:, 1:, 1:] - F[:, 1:, :-1]) / dr - (G[:, 1:, 1:] - G[:, :-1, 1:]) / dz
    assert np.abs(L[:, 1:, 1:] - want).max() < 1e-12


# ---- brute force in pure Python, written from the formulas W2-W7, not from the oracle --------------------------------------
def _py_weno(v):
    a, b, c, d, e = v
    q = [(2 * a - 7 * b + 11 * c) / 6, (-b + 5 * c + 2 * d) / 6, (2 * c + 5 * d - e) / 6]
    beta = [13 / 12 * (a - 2 * b + c) ** 2 + (a - 4 * b + 3 * c) ** 2 / 4,
            13 / 12 * (b - 2 * c + d) ** 2 + (b - d) ** 2 / 4,
            13 / 12 * (c - 2 * d + e) ** 2 + (3 * c - 4 * d + e) ** 2 / 4]
    al = [dk / (1e-6 + bk) ** 2 for dk, bk in zip((0.1, 0.6, 0.3), beta)]
    return sum(w * x for w, x in zip(al, q)) / sum(al)


def _py_rhs(U, dr, dz, gamma, bc):
    _, nz, nr = U.shape

    def src(i, n, lo, hi):
        if i < 0:
            return (0, 1) if lo == 0 else ((-1 - i, -1) if lo == 1 else (i + n, 1))
        if i >= n:
            return (n - 1, 1) if hi == 0 else ((2 * n - 1 - i, -1) if hi == 1 else (i - n, 1))
        return i, 1

    def state(i, j):
        si, fr = src(i, nr, bc[0], bc[1])
        sj, fz = src(j, nz, bc[2], bc[3])
        u = [float(U[c, sj, si]) for c in range(4)]
        u[1] *= fr
        u[2] *= fz
        return u

    def prim(u):
        p = (gamma - 1) * (u[3] - (u[1] ** 2 + u[2] ** 2) / (2 * u[0]))
        return u[1] / u[0], u[2] / u[0], p

    def flux(u, d):
        vr, vz, p = prim(u)
        v = (vr, vz)[d]
        f = [u[1 + d], u[1] * v, u[2] * v, (u[3] + p) * v]
        f[1 + d] += p
        return f

    al = [0.0, 0.0]
    for j in range(nz):
        for i in range(nr):
            u = state(i, j)
            vr, vz, p = prim(u)
            c = math.sqrt(gamma * p / u[0])
            al = [max(al[0], abs(vr) + c), max(al[1], abs(vz) + c)]

    def face(i, j, d):
        cells = [state(i - 2 + k, j) if d == 0 else state(i, j - 2 + k) for k in range(6)]
        fl = [flux(u, d) for u in cells]
        out = []
        for c in range(4):
            fp = [0.5 * (fl[k][c] + al[d] * cells[k][c]) for k in range(6)]
            fm = [0.5 * (fl[k][c] - al[d] * cells[k][c]) for k in range(6)]
            out.append(_py_weno(fp[0:5]) + _py_weno(fm[5:0:-1]))
        return out

    L = np.zeros_like(U)
    for j in range(nz):
        for i in range(nr):
            fe, fw, gn, gs = face(i, j, 0), face(i - 1, j, 0), face(i, j, 1), face(i, j - 1, 1)
            for c in range(4):
                L[c, j, i] = -(fe[c] - fw[c]) / dr - (gn[c] - gs[c]) / dz
    return L, al


@pytest.mark.parametrize("bc", [[0, 0, 0, 0], [1, 0, 1, 0], [2, 2, 0, 1], [1, 1, 2, 2]])
def test_brute_force_python_restatement(bc):
    rng = np.random.default_rng(7)
    nz, nr = 6, 9
    U = cons(1.0 + 0.5 * rng.random((nz, nr)), rng.standard_normal((nz, nr)), rng.standard_normal((nz, nr)),
             0.5 + rng.random((nz, nr)))
    U[:, :, 5:] *= 3.0                                  # a jump: the nonlinear weights matter
    want, al = _py_rhs(U, 0.1, 0.07, GAMMA, bc)
    got = oracle.weno_rhs(U, 0.1, 0.07, GAMMA, bc)
    assert np.allclose(oracle.weno_max_speeds(U, 0.1, 0.07, GAMMA, bc), al, rtol=1e-15)
    assert np.abs(got - want).max() <= 1e-11 * np.abs(want).max()


def test_reflecting_boundary_is_the_mirror_image():
    rng = np.random.default_rng(11)
    nz, nr = 5, 8
    U = cons(1.0 + 0.5 * rng.random((nz, nr)), rng.standard_normal((nz, nr)), rng.standard_normal((nz, nr)),
             0.5 + rng.random((nz, nr)))
    full = np.concatenate([U[:, :, ::-1] * np.array([1, -1, 1, 1])[:, None, None], U], axis=2)    # mirrored in r
    Lf = oracle.weno_rhs(full, 0.1, 0.1, GAMMA, [0, 0, 0, 0])
    Lh = oracle.weno_rhs(U, 0.1, 0.1, GAMMA, [1, 0, 0, 0], alpha=oracle.weno_max_speeds(full, 0.1, 0.1, GAMMA, [0, 0, 0, 0]))
    assert np.abs(Lf[:, :, nr:] - Lh).max() <= 1e-12 * np.abs(Lh).max()
    # and the mirrored half is the mirror image (the r-momentum equation is odd)
    assert np.abs(Lf[:, :, :nr][:, :, ::-1] * np.array([1, -1, 1, 1])[:, None, None] - Lh).max() <= 1e-12 * np.abs(Lh).max()


# ---- the paper's shock tubes (Table 3) against an exact Riemann solver ---------------------------------------------------
def exact_riemann(rl, ul, pl, rr, ur, pr, xi, g=GAMMA):
    """Exact solution of the Riemann problem at the similarity coordinates xi = (x - x0) / t (ideal gas).  Star-region
    pressure by Newton iteration on the two-shock / two-rarefaction pressure function, then sampling."""
    cl, cr = math.sqrt(g * pl / rl), math.sqrt(g * pr / rr)

    def fk(p, rk, pk, ck):
        if p > pk:                                   # shock
            A, B = 2.0 / ((g + 1) * rk), (g - 1) / (g + 1) * pk
            return (p - pk) * math.sqrt(A / (p + B)), math.sqrt(A / (p + B)) * (1 - (p - pk) / (2 * (p + B)))
        return 2 * ck / (g - 1) * ((p / pk) ** ((g - 1) / (2 * g)) - 1), 1.0 / (rk * ck) * (p / pk) ** (-(g + 1) / (2 * g))

    p = max(1e-8, ((cl + cr - 0.5 * (g - 1) * (ur - ul)) / (cl / pl ** ((g - 1) / (2 * g)) + cr / pr ** ((g - 1) / (2 * g))))
            ** (2 * g / (g - 1)))                    # two-rarefaction guess (positive by construction)
    for _ in range(200):
        fl, dl = fk(p, rl, pl, cl)
        fr, dr_ = fk(p, rr, pr, cr)
        pn = max(1e-10, p - (fl + fr + ur - ul) / (dl + dr_))
        if abs(pn - p) <= 1e-14 * (pn + p):
            p = pn
            break
        p = pn
    ps = p
    us = 0.5 * (ul + ur) + 0.5 * (fk(ps, rr, pr, cr)[0] - fk(ps, rl, pl, cl)[0])
    out = np.zeros((3, len(xi)))
    for n, s in enumerate(xi):
        if s <= us:                                  # left of the contact
            if ps > pl:
                sl = ul - cl * math.sqrt((g + 1) / (2 * g) * ps / pl + (g - 1) / (2 * g))
                w = (rl, ul, pl) if s <= sl else (rl * ((ps / pl + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * ps / pl + 1)), us, ps)
            else:
                cs = cl * (ps / pl) ** ((g - 1) / (2 * g))
                if s <= ul - cl:
                    w = (rl, ul, pl)
                elif s >= us - cs:
                    w = (rl * (ps / pl) ** (1 / g), us, ps)
                else:
                    c = 2 / (g + 1) * (cl + (g - 1) / 2 * (ul - s))
                    w = (rl * (c / cl) ** (2 / (g - 1)), 2 / (g + 1) * (cl + (g - 1) / 2 * ul + s), pl * (c / cl) ** (2 * g / (g - 1)))
        else:
            if ps > pr:
                sr = ur + cr * math.sqrt((g + 1) / (2 * g) * ps / pr + (g - 1) / (2 * g))
                w = (rr, ur, pr) if s >= sr else (rr * ((ps / pr + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * ps / pr + 1)), us, ps)
            else:
                cs = cr * (ps / pr) ** ((g - 1) / (2 * g))
                if s >= ur + cr:
                    w = (rr, ur, pr)
                elif s <= us + cs:
                    w = (rr * (ps / pr) ** (1 / g), us, ps)
                else:
                    c = 2 / (g + 1) * (cr - (g - 1) / 2 * (ur - s))
                    w = (rr * (c / cr) ** (2 / (g - 1)), 2 / (g + 1) * (-cr + (g - 1) / 2 * ur + s), pr * (c / cr) ** (2 * g / (g - 1)))
        out[:, n] = w
    return out


def test_exact_riemann_solver_reproduces_the_textbook_star_states():
    """The solver used as the pin is itself checked on Sod's problem (p* = 0.30313, u* = 0.92745: the classic values)."""
    w = exact_riemann(1.0, 0.0, 1.0, 0.125, 0.0, 0.1, np.array([0.5]))
    assert abs(w[2, 0] - 0.30313) < 1e-5 and abs(w[1, 0] - 0.92745) < 1e-5


def _table3():
    rows = []
    for line in open(__file__.replace("test_weno_pins.py", "golden/paper_table3_shocktubes.txt")):
        if line.strip() and not line.startswith("#"):
            rows.append([float(t) for t in line.split()])
    return rows


def _run_tube(row, n):
    _, t0, x0, rl, ul, pl, rr, ur, pr = row
    x = (np.arange(n) + 0.5) / n
    left = x < x0
    U = cons(np.where(left, rl, rr)[None, :], np.where(left, ul, ur)[None, :], 0.0, np.where(left, pl, pr)[None, :])
    # one row, dz so large that the z term of the time step vanishes: the 1-D Courant number 0.5 of PAPER.md:402
    Uf, steps = oracle.weno_evolve(U, 1.0 / n, 1.0e30, GAMMA, [0, 0, 0, 0], 0.5, t0)
    ex = exact_riemann(rl, ul, pl, rr, ur, pr, (x - x0) / t0)
    rho, v = Uf[0, 0], Uf[1, 0] / Uf[0, 0]
    p = (GAMMA - 1) * (Uf[3, 0] - 0.5 * rho * v * v)
    return (np.abs(rho - ex[0]).mean() / np.abs(ex[0]).mean(), np.abs(v - ex[1]).mean() / max(1.0, np.abs(ex[1]).max()),
            np.abs(p - ex[2]).mean() / np.abs(ex[2]).mean(), steps, rho, p)


@pytest.mark.parametrize("test", [1, 2, 3, 4])
def test_paper_shock_tubes_against_the_exact_solution(test):
    """PAPER.md:391-398 (Table 3): Toro's tests as the paper runs them (gamma = 1.4, Courant number 0.5), here on 400
    cells (the paper's 2000 are covered for test 1 below); L1 errors relative to the exact solution, and positivity."""
    row = list(_table3()[test - 1])
    assert int(row[0]) == test
    if test == 2:
        # The paper is at odds with itself: Table 3 prints t0 = 0.5, the text shows test 2 "at t0 = 0.15"
        # (Toro's value); at t = 0.5 both rarefactions (head speed 2.75) have long left the unit interval.  Reading W9
        # (DESIGN.md): t0 = 0.15.
        row[1] = 0.15
    e200 = _run_tube(row, 200)
    e400 = _run_tube(row, 400)
    tol = {1: 5e-3, 2: 1e-2, 3: 2e-2, 4: 6e-2}[test]        # L1(rho) / mean(rho); measured 4.0e-3, 7.6e-3, 1.4e-2, 4.4e-2
    assert e400[0] < tol and e400[1] < tol and e400[2] < tol, (e400[:4], tol)
    assert 0.4 < e400[0] / e200[0] < 0.7                 # first-order convergence in L1 across discontinuities
    assert e400[4].min() > 0 and e400[5].min() > 0


def test_paper_test1_at_the_papers_resolution():
    """"a spatial domain of interval [0,1] with 2000 computing cells"; test 1 only (the oracle is slow)."""
    row = _table3()[0]
    e = _run_tube(row, 2000)
    assert e[0] < 1.5e-3 and e[1] < 1.5e-3 and e[2] < 1.5e-3, e[:4]
