"""Pins for the CPU oracle (oracle/sn_oracle.cpp) against things other than itself.

The paper prints no worked Poisson example (PAPER.md:99 is the whole description), so the pins are what the
mathematics fixes: closed forms, a dense direct solve of the flux-form discretisation, refinement order,
the Roche formula of PAPER.md:99, Legendre polynomials and the exact ring potential from scipy, symmetry,
the discrete Gauss law, and a brute-force pure-Python red-black SOR on a tiny grid.
Each test names the plausible mistake it would catch.
"""
import math

import numpy as np
import pytest
from scipy import special

import workloads as W

FOURPI = 4.0 * math.pi


# ----------------------------------------------------------------------------------------------------------
# helpers that do NOT use the oracle
# ----------------------------------------------------------------------------------------------------------
def dense_direct(rho, dr, dz, symmetry, bE, bN, bS):
    """Assemble the conservative flux-form 5-point cylindrical Laplacian (R1) face by face and
    solve it with LAPACK.  Written from fluxes through cell faces, not from the oracle's coefficient tables."""
    nz, nr = rho.shape
    n = nr * nz
    A = np.zeros((n, n))
    b = FOURPI * rho.reshape(-1).copy()
    for j in range(nz):
        for i in range(nr):
            c = j * nr + i
            r_c = (i + 0.5) * dr
            # radial faces: area factor r_face / r_centre
            for (di, r_face) in ((+1, (i + 1) * dr), (-1, i * dr)):
                k = (r_face / r_c) / dr ** 2
                if k == 0.0:
                    continue                      # axis face has zero area: regular / reflecting axis
                A[c, c] -= k
                if 0 <= i + di < nr:
                    A[c, c + di] += k
                else:
                    b[c] -= k * bE[j]             # Dirichlet ghost at r = (nr+1/2) dr
            k = 1.0 / dz ** 2
            # north face
            A[c, c] -= k
            if j + 1 < nz:
                A[c, c + nr] += k
            else:
                b[c] -= k * bN[i]
            # south face
            if j > 0:
                A[c, c] -= k
                A[c, c - nr] += k
            elif symmetry == 0:
                A[c, c] -= k
                b[c] -= k * bS[i]
            # symmetry == 1, j == 0: reflecting equator, zero flux -> nothing
    return np.linalg.solve(A, b).reshape(nz, nr), A


def legendre_all(lmax, mu):
    return np.array([special.eval_legendre(l, mu) for l in range(lmax + 1)])


def ring_potential(m, r0, z0, r, z):
    """Exact potential (G=1) of a thin ring of mass m, radius r0, height z0 at field point (r,z)."""
    d2 = (r + r0) ** 2 + (z - z0) ** 2
    k2 = 4.0 * r * r0 / d2
    return -m * (2.0 / math.pi) * special.ellipk(k2) / math.sqrt(d2)


def python_rb_sor(rho, phi, dr, dz, symmetry, omega, bE, bN, bS, nsweeps):
    """Brute-force red-black SOR in plain Python (Gauss-Seidel form: solve each cell's equation, over-relax)."""
    nz, nr = rho.shape
    phi = phi.copy()
    for _ in range(nsweeps):
        for colour in (0, 1):
            for j in range(nz):
                for i in range(nr):
                    if (i + j) % 2 != colour:
                        continue
                    kE = (i + 1.0) / (i + 0.5) / dr ** 2
                    kW = i / (i + 0.5) / dr ** 2
                    kN = 1.0 / dz ** 2
                    kS = 0.0 if (symmetry == 1 and j == 0) else 1.0 / dz ** 2
                    pE = phi[j, i + 1] if i + 1 < nr else bE[j]
                    pW = phi[j, i - 1] if i > 0 else 0.0
                    pN = phi[j + 1, i] if j + 1 < nz else bN[i]
                    pS = phi[j - 1, i] if j > 0 else (0.0 if symmetry == 1 else bS[i])
                    gs = (kE * pE + kW * pW + kN * pN + kS * pS - FOURPI * rho[j, i]) / (kE + kW + kN + kS)
                    phi[j, i] = (1.0 - omega) * phi[j, i] + omega * gs
    return phi


def stagnate(O, w, omega=None, nsweeps=3000):
    """Run the oracle far past convergence (fixed sweeps)."""
    return O.solve(w.rho, np.zeros_like(w.rho), w.dr, w.dz, w.symmetry, w.lmax, 0.0, nsweeps, omega=omega)


# ----------------------------------------------------------------------------------------------------------
# harmonics, moments, boundary
# ----------------------------------------------------------------------------------------------------------
def test_regular_and_irregular_harmonics_match_legendre(oracle):
    """Catches a wrong recurrence coefficient / swapped x,y / missing s^2 factor."""
    lmax = 12
    for k in range(40):
        x = W.uniform(11, 0, 2 * k, 0.0, 1.5)
        y = W.uniform(11, 0, 2 * k + 1, -1.5, 1.5)
        s = math.hypot(x, y)
        P = legendre_all(lmax, y / s)
        R = oracle.regular_harmonics(x, y, lmax)
        I = oracle.irregular_harmonics(x, y, lmax)
        ls = np.arange(lmax + 1)
        np.testing.assert_allclose(R, s ** ls * P, rtol=1e-12, atol=1e-13)
        np.testing.assert_allclose(I, P / s ** (ls + 1), rtol=1e-11, atol=1e-13)


def test_harmonics_low_order_closed_forms(oracle):
    """P_2 = (3mu^2-1)/2, P_3 = (5mu^3-3mu)/2, P_4 = (35mu^4-30mu^2+3)/8 typed out."""
    x, y = 0.3, -0.7
    s2 = x * x + y * y
    R = oracle.regular_harmonics(x, y, 4)
    assert R[0] == 1.0 and R[1] == y
    assert R[2] == pytest.approx(0.5 * (3 * y * y - s2), rel=1e-14)
    assert R[3] == pytest.approx(0.5 * (5 * y ** 3 - 3 * y * s2), rel=1e-14)
    assert R[4] == pytest.approx((35 * y ** 4 - 30 * y * y * s2 + 3 * s2 * s2) / 8, rel=1e-13)


@pytest.mark.parametrize("symmetry", [0, 1])
def test_monopole_is_mass_and_roche_boundary(oracle, symmetry):
    """M_0 == sum rho dV (x2 mirrored); lmax=0 ghosts == -M/sqrt(r^2+z^2) (PAPER.md:99 Roche formula)."""
    w = W.random_smooth(24, 20, symmetry, seed=5)
    r, z = W.cell_centres(w.nr, w.nz, w.dr, w.dz, symmetry)
    mass = float(np.sum(w.rho * (2 * math.pi * r[None, :] * w.dr * w.dz))) * (2 if symmetry else 1)
    M = oracle.moments(w.rho, w.dr, w.dz, symmetry, 0)
    assert M[0] == pytest.approx(mass, rel=1e-13)
    bE, bN, bS = oracle.boundary(w.nr, w.nz, w.dr, w.dz, symmetry, 0, M)
    rE = (w.nr + 0.5) * w.dr
    np.testing.assert_allclose(bE, -mass / np.sqrt(rE ** 2 + z ** 2), rtol=1e-13)
    zN = z[-1] + w.dz
    np.testing.assert_allclose(bN, -mass / np.sqrt(r ** 2 + zN ** 2), rtol=1e-13)
    if symmetry == 0:
        zS = z[0] - w.dz
        assert zS == pytest.approx(-zN)
        np.testing.assert_allclose(bS, -mass / np.sqrt(r ** 2 + zS ** 2), rtol=1e-13)
    else:
        assert bS is None


def test_moments_against_independent_quadrature(oracle):
    """All l: M_l == sum rho s^l P_l(cos) dV with scipy Legendre (full plane), and even-l doubling (half plane)."""
    lmax = 9
    w = W.random_smooth(20, 28, 0, seed=6)
    r, z = W.cell_centres(w.nr, w.nz, w.dr, w.dz, 0)
    L0 = w.nr * w.dr
    rr, zz = np.meshgrid(r, z)
    s = np.hypot(rr, zz)
    dV = 2 * math.pi * rr * w.dr * w.dz
    want = np.array([np.sum(w.rho * (s / L0) ** l * special.eval_legendre(l, zz / s) * dV) for l in range(lmax + 1)])
    got = oracle.moments(w.rho, w.dr, w.dz, 0, lmax)
    np.testing.assert_allclose(got, want, rtol=1e-11, atol=1e-15)
    # half-plane of the upper half of a z-symmetric density == full-plane moments; odd l vanish
    wu = W.random_smooth(20, 14, 1, seed=6)
    full = np.concatenate([wu.rho[::-1], wu.rho], axis=0)
    Mfull = oracle.moments(full, wu.dr, wu.dz, 0, lmax)
    Mhalf = oracle.moments(wu.rho, wu.dr, wu.dz, 1, lmax)
    np.testing.assert_allclose(Mhalf[0::2], Mfull[0::2], rtol=1e-12)
    assert np.all(Mhalf[1::2] == 0.0)
    assert np.max(np.abs(Mfull[1::2])) < 1e-14 * abs(Mfull[0])


def test_sphere_moments_closed_form(oracle):
    """Uniform sphere [CFG 0]: M_0 -> (4/3) pi R^3 rho, higher even moments -> 0 (stair-cased edge, so loose)."""
    w = W.cfg0(64)
    M = oracle.moments(w.rho, w.dr, w.dz, 1, 8)
    exact = 4.0 / 3.0 * math.pi * 0.6 ** 3
    assert abs(M[0] / exact - 1) < 1e-3
    assert np.max(np.abs(M[2:])) < 1e-3 * M[0]
    w2 = W.cfg0(256)
    M2 = oracle.moments(w2.rho, w2.dr, w2.dz, 1, 8)
    assert abs(M2[0] / exact - 1) < abs(M[0] / exact - 1)


@pytest.mark.parametrize("symmetry", [0, 1])
def test_point_mass_boundary_converges_to_ring_potential(oracle, symmetry):
    """A single-cell density is a thin ring; its multipole ghosts must converge to the exact ring potential
    (elliptic K) as lmax grows -- catches a wrong sign, a wrong power of s, or theta measured from the wrong axis."""
    nr, nz = 32, 32 if symmetry else 64
    dr = dz = 1.0 / nr
    rho = np.zeros((nz, nr))
    i0, j0 = 5, (4 if symmetry else nz // 2 + 6)
    rho[j0, i0] = 1.0
    r, z = W.cell_centres(nr, nz, dr, dz, symmetry)
    m = 2 * math.pi * r[i0] * dr * dz
    errs = []
    for lmax in (0, 4, 16, 40):
        M = oracle.moments(rho, dr, dz, symmetry, lmax)
        bE, bN, bS = oracle.boundary(nr, nz, dr, dz, symmetry, lmax, M)
        rE = (nr + 0.5) * dr
        exact = np.array([ring_potential(m, r[i0], z[j0], rE, zz) for zz in z])
        if symmetry:
            exact += np.array([ring_potential(m, r[i0], -z[j0], rE, zz) for zz in z])
        errs.append(np.max(np.abs(bE - exact)) / np.max(np.abs(exact)))
    assert errs[0] > errs[1] > errs[2] > errs[3]
    assert errs[3] < 1e-9 and errs[0] > 1e-4


# ----------------------------------------------------------------------------------------------------------
# fixed point of the iteration: dense direct solve
# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("nr,nz,symmetry", [(16, 16, 1), (12, 16, 0), (7, 9, 1), (9, 6, 0)])
def test_sor_fixed_point_equals_dense_direct_solve(oracle, nr, nz, symmetry):
    """Catches any wrong coefficient, the equator/axis treatment, ghost placement and the sign of f."""
    w = W.random_smooth(nr, nz, symmetry, seed=7, lmax=4, dr=0.05, dz=0.04)
    M = oracle.moments(w.rho, w.dr, w.dz, symmetry, w.lmax)
    bE, bN, bS = oracle.boundary(nr, nz, w.dr, w.dz, symmetry, w.lmax, M)
    direct, _ = dense_direct(w.rho, w.dr, w.dz, symmetry, bE, bN, bS)
    out = oracle.solve(w.rho, np.zeros_like(w.rho), w.dr, w.dz, symmetry, w.lmax, 0.0, 600, omega=1.6)
    assert np.max(np.abs(out["phi"] - direct)) <= 5e-14 * np.max(np.abs(direct))
    # the whole-path solve used the same ghosts internally: injecting them gives the same bits
    out2 = oracle.solve(w.rho, np.zeros_like(w.rho), w.dr, w.dz, symmetry, w.lmax, 0.0, 600, omega=1.6,
                        boundary_arrays=(bE, bN, bS))
    assert np.array_equal(out["phi"], out2["phi"])


@pytest.mark.parametrize("symmetry", [0, 1])
def test_iteration_history_matches_bruteforce_python(oracle, symmetry):
    """Per-sweep iterate (ordering red-first, in-place Gauss-Seidel use of new values, omega) on a tiny grid."""
    w = W.random_smooth(6, 5, symmetry, seed=8, lmax=2, dr=0.1, dz=0.13)
    M = oracle.moments(w.rho, w.dr, w.dz, symmetry, 2)
    bE, bN, bS = oracle.boundary(6, 5, w.dr, w.dz, symmetry, 2, M)
    phi0 = np.array([[W.uniform(9, 0, j * 6 + i, -1, 1) for i in range(6)] for j in range(5)])
    for omega in (1.0, 1.7):
        for k in (1, 2, 5):
            got, _, _ = oracle.sweeps(w.rho, phi0, w.dr, w.dz, symmetry, omega, bE, bN, bS, k)
            want = python_rb_sor(w.rho, phi0, w.dr, w.dz, symmetry, omega, bE, bN, bS, k)
            np.testing.assert_allclose(got, want, rtol=0, atol=2e-13 * np.max(np.abs(want)))
    # a black-first ordering or a Jacobi (old values) update would differ at O(1)
    got1, _, _ = oracle.sweeps(w.rho, phi0, w.dr, w.dz, symmetry, 1.0, bE, bN, bS, 1)
    assert np.max(np.abs(got1 - phi0)) > 1e-3


# ----------------------------------------------------------------------------------------------------------
# closed forms
# ----------------------------------------------------------------------------------------------------------
def polytrope_n1_exact(s, R=0.8, rho_c=1.0):
    """phi -> 0 at infinity: inside -4 pi rho_c (R/pi)^2 [1 + sin(pi s/R)/(pi s/R)], outside -M/s, M = 4 rho_c R^3/pi
    (R13: the north_star text omits the constant '1 +')."""
    x = math.pi * s / R
    M = 4.0 * rho_c * R ** 3 / math.pi
    return np.where(s < R, -FOURPI * rho_c * (R / math.pi) ** 2 * (1.0 + np.sin(x) / x), -M / s)


def test_polytrope_closed_form_second_order(oracle):
    """Operator accuracy: error vs the closed form must fall x4 per refinement (32 -> 64 -> 128)."""
    errs = []
    for n in (32, 64, 128):
        w = W.cfg1(n, tol=1e-12)
        out = oracle.solve_workload(w)
        assert out["status"] == 0
        r, z = W.cell_centres(n, n, w.dr, w.dz, 1)
        s = np.hypot(r[None, :], z[:, None])
        errs.append(np.max(np.abs(out["phi"] - polytrope_n1_exact(s))))
    assert errs[0] < 1.3e-3 and errs[2] < 8e-5
    assert 3.3 < errs[0] / errs[1] < 4.6
    assert 3.6 < errs[1] / errs[2] < 4.4


def test_cfg1_full_size_closed_form_and_sweeps(oracle):
    """[CFG 1] 256x256 to tol 1e-10: error 1.7e-5 against the closed form; status 0."""
    w = W.cfg1()
    out = oracle.solve_workload(w, history=True)
    r, z = W.cell_centres(w.nr, w.nz, w.dr, w.dz, 1)
    s = np.hypot(r[None, :], z[:, None])
    err = np.max(np.abs(out["phi"] - polytrope_n1_exact(s)))
    assert err < 2.5e-5
    assert out["status"] == 0 and out["residual"] <= 1e-10
    assert out["hist"][-2] > 1e-10            # first crossing, not a later one
    assert 1000 < out["sweeps"] < 2000


def test_cfg0_uniform_sphere_closed_form(oracle):
    """[CFG 0]: -2 pi rho (R^2 - s^2/3) inside, -M/s outside; stair-cased edge => fixed tolerance (R14)."""
    w = W.cfg0()
    out = oracle.solve_workload(w)
    assert out["sweeps"] == 4000 and out["status"] == 0
    r, z = W.cell_centres(64, 64, w.dr, w.dz, 1)
    s = np.hypot(r[None, :], z[:, None])
    R = 0.6
    M = 4.0 / 3.0 * math.pi * R ** 3
    exact = np.where(s < R, -2 * math.pi * (R * R - s * s / 3), -M / s)
    assert np.max(np.abs(out["phi"] - exact)) < 3e-3 * np.max(np.abs(exact))


# ----------------------------------------------------------------------------------------------------------
# invariants
# ----------------------------------------------------------------------------------------------------------
def test_reflecting_equator_equals_mirrored_full_plane(oracle):
    """PAPER.md:99 'inner boundaries reflecting': half-plane solve == upper half of the mirrored full-plane solve."""
    wu = W.random_smooth(16, 12, 1, seed=10, lmax=6)
    full_rho = np.ascontiguousarray(np.concatenate([wu.rho[::-1], wu.rho], axis=0))
    half = oracle.solve(wu.rho, np.zeros_like(wu.rho), wu.dr, wu.dz, 1, 6, 0.0, 1500, omega=1.7)
    full = oracle.solve(full_rho, np.zeros_like(full_rho), wu.dr, wu.dz, 0, 6, 0.0, 1500, omega=1.7)
    scale = np.max(np.abs(half["phi"]))
    assert np.max(np.abs(full["phi"][12:] - half["phi"])) < 1e-13 * scale
    assert np.max(np.abs(full["phi"][:12] - half["phi"][::-1])) < 1e-13 * scale


@pytest.mark.parametrize("symmetry", [0, 1])
def test_discrete_gauss_law(oracle, symmetry):
    """Conservative form telescopes: sum 4 pi rho dV == sum over outer faces of (dphi/dn) dA at the fixed point."""
    w = W.random_smooth(20, 16, symmetry, seed=12, lmax=6)
    M = oracle.moments(w.rho, w.dr, w.dz, symmetry, 6)
    bE, bN, bS = oracle.boundary(w.nr, w.nz, w.dr, w.dz, symmetry, 6, M)
    phi = stagnate(oracle, w, omega=1.7, nsweeps=2500)["phi"]
    r, _ = W.cell_centres(w.nr, w.nz, w.dr, w.dz, symmetry)
    lhs = np.sum(FOURPI * w.rho * 2 * math.pi * r[None, :] * w.dr * w.dz)
    rE = w.nr * w.dr
    flux = np.sum((bE - phi[:, -1]) / w.dr * 2 * math.pi * rE * w.dz)
    flux += np.sum((bN - phi[-1, :]) / w.dz * 2 * math.pi * r * w.dr)
    if symmetry == 0:
        flux += np.sum((bS - phi[0, :]) / w.dz * 2 * math.pi * r * w.dr)
    assert flux == pytest.approx(lhs, rel=1e-11)
    # and the residual of the plain-arithmetic operator vanishes there
    res = oracle.apply_operator(phi, w.dr, w.dz, symmetry, bE, bN, bS) - FOURPI * w.rho
    assert np.max(np.abs(res)) < 1e-9 * np.max(np.abs(FOURPI * w.rho))


def test_linearity_and_length_scaling(oracle):
    a = W.random_smooth(14, 14, 1, seed=13, lmax=4)
    b = W.random_smooth(14, 14, 1, seed=14, lmax=4)
    pa = stagnate(oracle, a, 1.6, 800)["phi"]
    pb = stagnate(oracle, b, 1.6, 800)["phi"]
    c = W.Workload("c", 14, 14, a.dr, a.dz, 1, 4, 0.0, 800, np.ascontiguousarray(2.0 * a.rho - 0.5 * b.rho))
    pc = stagnate(oracle, c, 1.6, 800)["phi"]
    np.testing.assert_allclose(pc, 2.0 * pa - 0.5 * pb, atol=1e-13 * np.max(np.abs(pa)))
    # dr,dz -> 3 dr, 3 dz with the same rho values: phi -> 9 phi
    d = W.Workload("d", 14, 14, 3 * a.dr, 3 * a.dz, 1, 4, 0.0, 800, a.rho)
    pd = stagnate(oracle, d, 1.6, 800)["phi"]
    np.testing.assert_allclose(pd, 9.0 * pa, rtol=1e-12)


@pytest.mark.parametrize("nr,nz,symmetry", [(16, 16, 1), (12, 24, 0)])
def test_default_omega_tracks_jacobi_spectral_radius(oracle, nr, nz, symmetry):
    """omega formula (R8): mu must approximate the Jacobi spectral radius of the assembled matrix."""
    dr = dz = 1.0 / nr
    rho = np.zeros((nz, nr))
    _, A = dense_direct(rho, dr, dz, symmetry, np.zeros(nz), np.zeros(nr), np.zeros(nr))
    Dg = np.diag(A)
    J = np.eye(nr * nz) - A / Dg[:, None]
    mu_true = np.max(np.abs(np.linalg.eigvals(J)))
    omega_true = 2.0 / (1.0 + math.sqrt(1.0 - mu_true ** 2))
    omega = oracle.default_omega(nr, nz, dr, dz, symmetry)
    assert 1.0 < omega < 2.0
    assert abs(omega - omega_true) < 0.01
    # typed-out formula, independent evaluation
    Lr = (nr + 0.5) * dr
    kz = math.pi / (2 * (nz + 0.5) * dz) if symmetry else math.pi / ((nz + 1) * dz)
    mu = 1 - ((2.404825557695773 / Lr) ** 2 + kz ** 2) / (2 / dr ** 2 + 2 / dz ** 2)
    assert omega == pytest.approx(2 / (1 + math.sqrt(1 - mu * mu)), rel=1e-14)


def test_survey_probe_values_for_default_omega(oracle):
    assert oracle.default_omega(64, 64, 1 / 64, 1 / 64, 1) == pytest.approx(1.93895, abs=2e-5)
    assert oracle.default_omega(256, 256, 1 / 256, 1 / 256, 1) == pytest.approx(1.98428765, abs=1e-8)
    assert oracle.default_omega(128, 256, 1 / 128, 1 / 128, 0) == pytest.approx(1.96888068, abs=1e-8)


# ----------------------------------------------------------------------------------------------------------
# stopping rule and the solve contract
# ----------------------------------------------------------------------------------------------------------
def test_stopping_rule_and_sweep_count(oracle):
    w = W.random_smooth(24, 24, 1, seed=15, lmax=6)
    M = oracle.moments(w.rho, w.dr, w.dz, 1, 6)
    bE, bN, bS = oracle.boundary(24, 24, w.dr, w.dz, 1, 6, M)
    omega = oracle.default_omega(24, 24, w.dr, w.dz, 1)
    out = oracle.solve(w.rho, np.zeros_like(w.rho), w.dr, w.dz, 1, 6, 1e-9, 5000, history=True)
    k = out["sweeps"]
    assert out["status"] == 0 and out["hist"][k - 1] <= 1e-9 and np.all(out["hist"][: k - 1] > 1e-9)
    # history == ratio assembled from the raw per-sweep maxima, independently
    phi, Rabs, P = oracle.sweeps(w.rho, np.zeros_like(w.rho), w.dr, w.dz, 1, omega, bE, bN, bS, k)
    assert np.array_equal(phi, out["phi"])
    maxf = np.max(np.abs(12.566370614359172 * w.rho))
    Dfull = 2 / w.dr ** 2 + 2 / w.dz ** 2
    np.testing.assert_allclose(out["hist"], Rabs / (maxf + Dfull * P), rtol=1e-14)
    assert out["residual"] == out["hist"][-1]
    # Rabs really is the max pre-update residual of the first sweep: recompute sweep 1 by brute force
    want1 = python_rb_sor(w.rho, np.zeros_like(w.rho), w.dr, w.dz, 1, omega, bE, bN, bS, 1)
    assert P[0] == pytest.approx(np.max(np.abs(want1)), rel=1e-13)
    # max_sweeps hit -> status 1; fixed-sweep mode -> status 0 with exactly max_sweeps
    out1 = oracle.solve(w.rho, np.zeros_like(w.rho), w.dr, w.dz, 1, 6, 1e-9, k - 1)
    assert out1["status"] == 1 and out1["sweeps"] == k - 1
    out2 = oracle.solve(w.rho, np.zeros_like(w.rho), w.dr, w.dz, 1, 6, 0.0, 7)
    assert out2["status"] == 0 and out2["sweeps"] == 7
    # warm start from the converged phi stops at once
    out3 = oracle.solve(w.rho, stagnate(oracle, w, nsweeps=2000)["phi"], w.dr, w.dz, 1, 6, 1e-9, 100)
    assert out3["sweeps"] == 1 and out3["status"] == 0


def test_relative_change_relation_to_paper_rule(oracle):
    """PAPER.md:99 stops on relative change; R9: max|dphi| = (omega/diag) max|res| ties R_k to it."""
    w = W.random_smooth(20, 20, 0, seed=16, lmax=4)
    M = oracle.moments(w.rho, w.dr, w.dz, 0, 4)
    bE, bN, bS = oracle.boundary(20, 20, w.dr, w.dz, 0, 4, M)
    omega = 1.5
    p0, _, _ = oracle.sweeps(w.rho, np.zeros_like(w.rho), w.dr, w.dz, 0, omega, bE, bN, bS, 30)
    p1, Rabs, _ = oracle.sweeps(w.rho, p0, w.dr, w.dz, 0, omega, bE, bN, bS, 1)
    D = 2 / w.dr ** 2 + 2 / w.dz ** 2
    assert np.max(np.abs(p1 - p0)) == pytest.approx(omega / D * Rabs[0], rel=1e-9)


@pytest.mark.parametrize("symmetry", [0, 1])
def test_paper_literal_rule_picks_the_sweep_of_a_bruteforce_python_sor(oracle, symmetry):
    """R16 / PAPER.md:99 "stopped ... when the relative changes of all grids reach below 1e-8": an independent pure-Python
    red-black SOR that measures max|phi_new - phi_old| / max|phi_new| sweep by sweep stops at the same sweep as the
    oracle's rule 1, and the oracle's E_k equals that ratio to the rounding of the difference (|dphi| ~ 1e-5 |phi| here,
    so ~1e-11 relative); with symmetry = 1 the mirror row (diag = D - 1/dz^2, larger omega/diag) is part of the maximum."""
    nr, nz, tol = 10, 8, 1e-5
    w = W.random_smooth(nr, nz, symmetry, seed=60 + symmetry, lmax=4)
    M = oracle.moments(w.rho, w.dr, w.dz, symmetry, 4)
    bnd = oracle.boundary(nr, nz, w.dr, w.dz, symmetry, 4, M)
    omega = oracle.default_omega(nr, nz, w.dr, w.dz, symmetry)
    ref = oracle.solve(w.rho, np.zeros_like(w.rho), w.dr, w.dz, symmetry, 4, tol, 500, boundary_arrays=bnd, rule=1,
                       history=True)
    assert ref["status"] == 0 and 10 < ref["sweeps"] < 500
    phi = np.zeros_like(w.rho)
    stop = None
    for k in range(1, 500):
        new = python_rb_sor(w.rho, phi, w.dr, w.dz, symmetry, omega, bnd[0], bnd[1], bnd[2], 1)
        E = np.max(np.abs(new - phi)) / np.max(np.abs(new))
        assert ref["hist"][k - 1] == pytest.approx(E, rel=1e-8)
        phi = new
        if E <= tol:
            stop = k
            break
    assert stop == ref["sweeps"] and ref["residual"] == ref["hist"][-1] <= tol
    assert np.max(np.abs(phi - ref["phi"])) <= 1e-12 * np.max(np.abs(phi))
    # the change is (omega/diag_j) |res| cell by cell: max over the rows with their own diag (mirror row: D0 < D)
    p1, Rabs, Pk, Chg = oracle.sweeps_chg(w.rho, np.zeros_like(w.rho), w.dr, w.dz, symmetry, omega, *bnd, 3)
    assert oracle.relchange(Chg[2], Pk[2]) == ref["hist"][2] and oracle.relchange(0.0, 0.0) == 0.0
    D = 2 / w.dr ** 2 + 2 / w.dz ** 2
    assert Chg[0] >= omega / D * Rabs[0] * (1 - 1e-15)
    if symmetry == 0:
        assert Chg[0] == omega / D * Rabs[0]
    # rule 0 is untouched by the new argument
    a = oracle.solve(w.rho, np.zeros_like(w.rho), w.dr, w.dz, symmetry, 4, 1e-9, 500, boundary_arrays=bnd)
    b = oracle.solve(w.rho, np.zeros_like(w.rho), w.dr, w.dz, symmetry, 4, 1e-9, 500, boundary_arrays=bnd, rule=0)
    assert a["sweeps"] == b["sweeps"] and np.array_equal(a["phi"], b["phi"])


def test_degenerate_inputs(oracle):
    z = np.zeros((8, 8))
    out = oracle.solve(z, z, 0.1, 0.1, 1, 4, 1e-10, 50)
    assert out["status"] == 0 and out["sweeps"] == 1 and out["residual"] == 0.0 and np.all(out["phi"] == 0)
    bad = oracle.solve(z, z, -0.1, 0.1, 1, 4, 1e-10, 50)
    assert bad["status"] == -1
    rho = np.full((8, 8), np.nan)
    out = oracle.solve(rho, z, 0.1, 0.1, 1, 0, 1e-10, 50)
    assert out["status"] == -3
    # smallest legal grid, odd sizes, lmax = 0
    w = W.random_smooth(2, 2, 0, seed=17, lmax=0)
    out = oracle.solve_workload(w)
    assert out["status"] == 0
    w = W.random_smooth(5, 3, 1, seed=18, lmax=1)
    out = oracle.solve_workload(w)
    assert out["status"] == 0


def test_wd_config_quadrupole_is_small(oracle):
    """'the quadruple term gives a less than 1% correction to the monopole term' at the boundary."""
    w = W.cfg2(128)
    M = oracle.moments(w.rho, w.dr, w.dz, 1, 2)
    b0 = oracle.boundary(w.nr, w.nz, w.dr, w.dz, 1, 0, M[:1])[0]
    b2 = oracle.boundary(w.nr, w.nz, w.dr, w.dz, 1, 2, M)[0]
    assert np.max(np.abs(b2 - b0) / np.abs(b0)) < 0.01
    # mass of the bubble-free synthetic star == Table 5's 1.377 Msun in code units, to quadrature error
    w0 = W.cfg4b(128)
    assert oracle.moments(w0.rho, w0.dr, w0.dz, 1, 0)[0] == pytest.approx(W.M_WD_CODE, rel=0.01)


# ----------------------------------------------------------------------------------------------------------
# NEXT-1: gravity epilogue g = -grad phi (eqs. 2-4; R15)
# ----------------------------------------------------------------------------------------------------------
def _ghost_samples(fun, nr, nz, dr, dz, symmetry):
    """fun(r, z) sampled at the east / north / south ghost-cell centres (R4)."""
    r, z = W.cell_centres(nr, nz, dr, dz, symmetry)
    bE = fun((nr + 0.5) * dr, z)
    bN = fun(r, z[-1] + dz)
    bS = fun(r, z[0] - dz)
    return r, z, bE, bN, bS


@pytest.mark.parametrize("symmetry", [0, 1])
def test_gravity_is_exact_on_quadratic_potentials(oracle, symmetry):
    """Centred differences are exact for a + b r^2 + c z^2 (+ d z when there is no equatorial mirror), including the
    reflecting axis (phi is even in r) and equator rows and the rows / columns next to the Dirichlet ghosts."""
    nr, nz, dr, dz = 11, 9, 0.07, 0.11
    a, b, c, d = 1.5, -3.0, 0.7, (0.0 if symmetry == 1 else 2.5)
    fun = lambda r, z: a + b * r ** 2 + c * z ** 2 + d * z
    r, z, bE, bN, bS = _ghost_samples(fun, nr, nz, dr, dz, symmetry)
    phi = fun(r[None, :], z[:, None])
    gr, gz = oracle.gravity(phi, dr, dz, symmetry, bE, bN, bS)
    assert np.allclose(gr, -2 * b * r[None, :] * np.ones((nz, 1)), rtol=0, atol=1e-13)
    assert np.allclose(gz, -(2 * c * z[:, None] + d) * np.ones((1, nr)), rtol=0, atol=1e-13)


def test_gravity_second_order_on_the_polytrope_field(oracle):
    """The analytic n=1 polytrope potential (R13) sampled on the grid: the differenced field converges to the closed
    form g = -dphi/ds s_hat at second order (error x1/4 per refinement), inside and outside the star."""
    R = 0.8
    k = np.pi / R

    def phi_fun(r, z):
        s = np.hypot(r, z)
        x = k * s
        return np.where(s < R, -4 * np.pi / k ** 2 * (1 + np.sin(x) / x), -(4 * R ** 3 / np.pi) / s)

    def g_mag(s):        # -dphi/ds
        x = k * s
        inside = 4 * np.pi / k * (x * np.cos(x) - np.sin(x)) / x ** 2
        return np.where(s < R, inside, -(4 * R ** 3 / np.pi) / s ** 2)

    errs = []
    for n in (32, 64, 128):
        dr = dz = 1.0 / n
        r, z, bE, bN, bS = _ghost_samples(phi_fun, n, n, dr, dz, 1)
        phi = phi_fun(r[None, :], z[:, None])
        gr, gz = oracle.gravity(phi, dr, dz, 1, bE, bN, bS)
        s = np.hypot(r[None, :], z[:, None])
        g = g_mag(s)
        errs.append(max(np.max(np.abs(gr - g * r[None, :] / s)), np.max(np.abs(gz - g * z[:, None] / s))))
    assert errs[0] < 2e-2 and 3.0 < errs[0] / errs[1] < 5.0 and 3.0 < errs[1] / errs[2] < 5.0


def test_gravity_of_the_solved_polytrope_and_mirror_antisymmetry(oracle):
    """End to end: the solved cfg-1 potential differenced by the oracle matches the closed-form field; on a full
    plane with a z-symmetric density g_z is odd and g_r even in z."""
    w = W.cfg1(64)
    ref = oracle.solve_workload(w)
    M = oracle.moments(w.rho, w.dr, w.dz, 1, w.lmax)
    bnd = oracle.boundary(w.nr, w.nz, w.dr, w.dz, 1, w.lmax, M)
    gr, gz = oracle.gravity(ref["phi"], w.dr, w.dz, 1, *bnd)
    r, z = W.cell_centres(w.nr, w.nz, w.dr, w.dz, 1)
    s = np.hypot(r[None, :], z[:, None])
    R, k = 0.8, np.pi / 0.8
    x = k * s
    g = np.where(s < R, 4 * np.pi / k * (x * np.cos(x) - np.sin(x)) / x ** 2, -(4 * R ** 3 / np.pi) / s ** 2)
    assert np.max(np.abs(gr - g * r[None, :] / s)) < 5e-3 and np.max(np.abs(gz - g * z[:, None] / s)) < 5e-3
    # mirrored full plane
    rho_full = np.concatenate([w.rho[::-1], w.rho])
    full = oracle.solve(rho_full, np.zeros_like(rho_full), w.dr, w.dz, 0, w.lmax, 0.0, 3000)
    Mf = oracle.moments(rho_full, w.dr, w.dz, 0, w.lmax)
    bf = oracle.boundary(w.nr, 2 * w.nz, w.dr, w.dz, 0, w.lmax, Mf)
    grf, gzf = oracle.gravity(full["phi"], w.dr, w.dz, 0, *bf)
    assert np.max(np.abs(gzf + gzf[::-1])) < 1e-9 and np.max(np.abs(grf - grf[::-1])) < 1e-9
