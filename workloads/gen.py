"""Seeded synthetic density grids for the five BASELINE.json configs.

This module is *input generation only*.  It feeds both the CPU oracle (tests,
``bench.py``'s cpu_baseline leg) and the CUDA path, and holds none of the
method's arithmetic: no multipole moments, no stencil, no relaxation.  It
imports neither ``oracle`` nor ``paper_1507_08549_b200``.

The paper's own workloads are white-dwarf density fields from its hydro runs
("500 x 500 ... grid size ~11 km"; Table 5:
rho_c = 3e9 g/cm^3, M = 1.377 Msun).  Those fields are not available, so the
grids below are seeded stand-ins that take their shape and scale from those
lines; the recipe is stated in DESIGN.md §4 and SURVEY.md §8(d).

Layout of every returned grid: ``rho[j, i]`` (C order, r fastest), i in
[0, nr) radial, j in [0, nz) vertical; cell centres r_i = (i + 1/2) dr and
z_j = (j + 1/2) dz (symmetry=1) or (j + 1/2 - nz/2) dz (symmetry=0).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from functools import lru_cache

import numpy as np

# ----------------------------------------------------------------------------
# counter-based RNG (SplitMix64 finaliser over seed/stream/counter)
# ----------------------------------------------------------------------------
_M64 = (1 << 64) - 1
_GOLD = 0x9E3779B97F4A7C15


def _mix64(x: int) -> int:
    x &= _M64
    x = ((x ^ (x >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    x = ((x ^ (x >> 27)) * 0x94D049BB133111EB) & _M64
    return x ^ (x >> 31)


def u01(seed: int, stream: int, counter: int) -> float:
    """Uniform double in [0,1): a pure function of (seed, stream, counter)."""
    k = _mix64(seed * _GOLD + 0x1234567)
    k = _mix64(k ^ (stream * 0xD1B54A32D192ED03 & _M64))
    z = _mix64(k + (counter + 1) * _GOLD)
    return (z >> 11) * (1.0 / 9007199254740992.0)


def uniform(seed: int, stream: int, counter: int, lo: float, hi: float) -> float:
    return lo + (hi - lo) * u01(seed, stream, counter)


# ----------------------------------------------------------------------------
# units: length 5000 km -> 1, density 1e9 g/cm^3 -> 1, G = 1
# ----------------------------------------------------------------------------
KM = 1.0 / 5000.0                     # one km in code length units
MSUN_G = 1.989e33
RHO0_CGS = 1.0e9
L_CGS = 5.0e8
M_WD_CODE = 1.377 * MSUN_G / (RHO0_CGS * L_CGS ** 3)   # PAPER.md:488 (Table 5) M = 1.377 Msun
RHO_FLOOR = 1.0e-12                   # 1e-3 g/cm^3 in code units ([CFG 2] "floor 1e-3 g/cm^3")


@dataclass
class Workload:
    """A Poisson problem: grid, solver arguments and the density field."""
    name: str
    nr: int
    nz: int
    dr: float
    dz: float
    symmetry: int
    lmax: int
    tol: float
    max_sweeps: int
    rho: np.ndarray                   # (nz, nr) float64, C-contiguous
    omega: float | None = None        # None -> library / oracle default formula
    meta: dict = field(default_factory=dict)

    @property
    def cells(self) -> int:
        return self.nr * self.nz


def cell_centres(nr, nz, dr, dz, symmetry):
    r = (np.arange(nr, dtype=np.float64) + 0.5) * dr
    if symmetry == 1:
        z = (np.arange(nz, dtype=np.float64) + 0.5) * dz
    else:
        z = (np.arange(nz, dtype=np.float64) + 0.5 - 0.5 * nz) * dz
    return r, z


# ----------------------------------------------------------------------------
# Lane-Emden n = 3 (classical RK4, textbook xi_1 = 6.89685, -xi_1^2 theta' = 2.01824)
# ----------------------------------------------------------------------------
@lru_cache(maxsize=None)
def lane_emden(n: float = 3.0, h: float = 1.0e-3):
    """Integrate theta'' + (2/xi) theta' + theta^n = 0 outward with RK4.

    Returns (xi, theta, xi1, minus_xi1sq_dtheta) with theta > 0 on xi < xi1.
    """
    def rhs(x, th, ph):               # ph = dtheta/dxi
        return ph, -(max(th, 0.0) ** n) - 2.0 * ph / x

    # series start: theta = 1 - x^2/6 + n x^4/120
    x = h
    th = 1.0 - x * x / 6.0 + n * x ** 4 / 120.0
    ph = -x / 3.0 + n * x ** 3 / 30.0
    xs = [0.0, x]
    ths = [1.0, th]
    phs = [0.0, ph]
    while th > 0.0 and x < 50.0:
        k1t, k1p = rhs(x, th, ph)
        k2t, k2p = rhs(x + 0.5 * h, th + 0.5 * h * k1t, ph + 0.5 * h * k1p)
        k3t, k3p = rhs(x + 0.5 * h, th + 0.5 * h * k2t, ph + 0.5 * h * k2p)
        k4t, k4p = rhs(x + h, th + h * k3t, ph + h * k3p)
        th_new = th + h * (k1t + 2 * k2t + 2 * k3t + k4t) / 6.0
        ph_new = ph + h * (k1p + 2 * k2p + 2 * k3p + k4p) / 6.0
        x += h
        th, ph = th_new, ph_new
        xs.append(x)
        ths.append(th)
        phs.append(ph)
    # linear interpolation of the first zero between the last two samples
    x0, x1 = xs[-2], xs[-1]
    t0, t1 = ths[-2], ths[-1]
    xi1 = x0 + (x1 - x0) * t0 / (t0 - t1)
    dth = phs[-2] + (phs[-1] - phs[-2]) * (xi1 - x0) / (x1 - x0)
    ths[-1] = 0.0
    xs[-1] = xi1
    return (np.asarray(xs), np.asarray(ths), float(xi1), float(-xi1 * xi1 * dth))


def wd_scale_length(rho_c: float) -> float:
    """Lane-Emden length a with M = 4 pi a^3 rho_c (-xi1^2 theta'(xi1)) = 1.377 Msun."""
    _, _, _, mfac = lane_emden()
    return (M_WD_CODE / (4.0 * math.pi * rho_c * mfac)) ** (1.0 / 3.0)


def wd_profile(s: np.ndarray, rho_c: float) -> np.ndarray:
    """n=3 polytrope density rho_c theta(s/a)^3 with the floor applied."""
    xi, th, xi1, _ = lane_emden()
    a = wd_scale_length(rho_c)
    theta = np.interp(s / a, xi, th, right=0.0)
    return np.maximum(rho_c * theta ** 3, RHO_FLOOR)


def _bubbles(seed: int, stream: int, nb: int, s_max: float, half_plane: bool,
             z_shift: float = 0.0):
    """nb Gaussian deficits: (r_k, z_k, A_k, w_k); centres uniform in area within s<s_max."""
    out = []
    for k in range(nb):
        A = uniform(seed, stream, 4 * k + 0, 0.05, 0.30)
        w = uniform(seed, stream, 4 * k + 1, 20.0 * KM, 100.0 * KM)
        s = s_max * math.sqrt(u01(seed, stream, 4 * k + 2))
        ang = u01(seed, stream, 4 * k + 3) * (0.5 * math.pi if half_plane else math.pi)
        # polar angle from +z; (r,z) half-plane has r >= 0
        out.append((s * math.sin(ang), s * math.cos(ang) + z_shift, A, w))
    return out


def _apply_bubbles(rho, r, z, bubbles):
    for (rk, zk, A, w) in bubbles:
        gr = np.exp(-((r - rk) ** 2) / (2.0 * w * w))
        gz = np.exp(-((z - zk) ** 2) / (2.0 * w * w))
        rho *= 1.0 - A * np.outer(gz, gr)
    return rho


# ----------------------------------------------------------------------------
# the configs
# ----------------------------------------------------------------------------
def cfg0(n: int = 64) -> Workload:
    """[CFG 0] uniform-density sphere rho=1 for s<0.6 on the unit half-plane grid."""
    dr = dz = 1.0 / n
    r, z = cell_centres(n, n, dr, dz, 1)
    s = np.sqrt(r[None, :] ** 2 + z[:, None] ** 2)
    rho = np.where(s < 0.6, 1.0, 0.0).astype(np.float64)
    return Workload("cfg0_sphere", n, n, dr, dz, 1, 8, 0.0, 4000, np.ascontiguousarray(rho),
                    omega=1.9, meta={"R": 0.6, "rho_c": 1.0})


def cfg1(n: int = 256, lmax: int = 16, tol: float = 1e-10, max_sweeps: int = 20000) -> Workload:
    """[CFG 1] n=1 polytrope rho = sinc(pi s / R), R = 0.8, on the unit half-plane grid."""
    dr = dz = 1.0 / n
    R = 0.8
    r, z = cell_centres(n, n, dr, dz, 1)
    s = np.sqrt(r[None, :] ** 2 + z[:, None] ** 2)
    x = np.pi * s / R
    rho = np.where(s < R, np.sin(x) / x, 0.0)
    return Workload("cfg1_polytrope_n1", n, n, dr, dz, 1, lmax, tol, max_sweeps,
                    np.ascontiguousarray(rho), meta={"R": R, "rho_c": 1.0})


def wd_half_plane(n: int, rho_c: float, nb: int, seed: int, lmax: int = 16,
                  tol: float = 1e-10, max_sweeps: int = 40000, name: str = "wd") -> Workload:
    """n x n half-plane grid over 0..5000 km, n=3 WD with nb seeded ash bubbles."""
    dr = dz = 1.0 / n
    r, z = cell_centres(n, n, dr, dz, 1)
    s = np.sqrt(r[None, :] ** 2 + z[:, None] ** 2)
    rho = wd_profile(s, rho_c)
    bub = _bubbles(seed, 1, nb, 1000.0 * KM, True)
    rho = _apply_bubbles(rho, r, z, bub)
    return Workload(name, n, n, dr, dz, 1, lmax, tol, max_sweeps, np.ascontiguousarray(rho),
                    meta={"rho_c": rho_c, "bubbles": bub, "seed": seed,
                          "a": wd_scale_length(rho_c)})


def cfg2(n: int = 512) -> Workload:
    """[CFG 2] 512 x 512, rho_c = 3 (3e9 g/cm^3), 20 bubbles, seed 2."""
    return wd_half_plane(n, 3.0, 20, seed=2, name="cfg2_wd512")


@dataclass
class Cfg3Sequence:
    """[CFG 3] 1024 x 2048 full-plane warm-started sequence; rho(t) by seeded smooth perturbations."""
    first: Workload
    nsteps: int
    seed: int

    def perturbation(self, t: int) -> np.ndarray:
        """g_t: sum of 8 seeded unit-amplitude +/- Gaussian blobs (separable exponentials)."""
        w0 = self.first
        r, z = cell_centres(w0.nr, w0.nz, w0.dr, w0.dz, 0)
        g = np.zeros((w0.nz, w0.nr))
        for k in range(8):
            sign = 1.0 if u01(self.seed, 100 + t, 5 * k) < 0.5 else -1.0
            w = uniform(self.seed, 100 + t, 5 * k + 1, 100.0 * KM, 500.0 * KM)
            s = 1500.0 * KM * math.sqrt(u01(self.seed, 100 + t, 5 * k + 2))
            ang = u01(self.seed, 100 + t, 5 * k + 3) * math.pi
            rk, zk = s * math.sin(ang), s * math.cos(ang)
            g += sign * np.outer(np.exp(-((z - zk) ** 2) / (2 * w * w)),
                                 np.exp(-((r - rk) ** 2) / (2 * w * w)))
        return g

    def step(self, rho: np.ndarray, t: int) -> np.ndarray:
        """rho_{t} = rho_{t-1} * (1 + 1e-3 g_t), t >= 1."""
        return np.ascontiguousarray(rho * (1.0 + 1.0e-3 * self.perturbation(t)))


def cfg3(nr: int = 1024, nz: int | None = None, nsteps: int = 100, lmax: int = 32) -> Cfg3Sequence:
    nz = 2 * nr if nz is None else nz
    dr = dz = 1.0 / nr
    seed = 3
    r, z = cell_centres(nr, nz, dr, dz, 0)
    zc = 50.0 * KM
    s = np.sqrt(r[None, :] ** 2 + (z[:, None] - zc) ** 2)
    rho = wd_profile(s, 3.0)
    # one off-centre bubble: centre at 300-800 km from the star's centre
    A = uniform(seed, 1, 0, 0.05, 0.30)
    w = uniform(seed, 1, 1, 20.0 * KM, 100.0 * KM)
    sb = uniform(seed, 1, 2, 300.0 * KM, 800.0 * KM)
    ang = u01(seed, 1, 3) * math.pi
    bub = [(sb * math.sin(ang), sb * math.cos(ang) + zc, A, w)]
    rho = _apply_bubbles(rho, r, z, bub)
    first = Workload("cfg3_full_plane_seq", nr, nz, dr, dz, 0, lmax, 1e-10, 80000,
                     np.ascontiguousarray(rho), meta={"bubbles": bub, "z_centre": zc, "seed": seed})
    return Cfg3Sequence(first, nsteps, seed)


def cfg4a_member(b: int, n: int = 512) -> Workload:
    """[CFG 4a] batch member b: rho_c in U[1,5], 5..30 bubbles, seed 4000+b."""
    seed = 4000 + b
    rho_c = uniform(seed, 0, 0, 1.0, 5.0)
    nb = 5 + int(u01(seed, 0, 1) * 26.0)
    return wd_half_plane(n, rho_c, nb, seed=seed, name=f"cfg4a_{b:02d}")


def cfg4a(nbatch: int = 64, n: int = 512) -> list[Workload]:
    return [cfg4a_member(b, n) for b in range(nbatch)]


def cfg4b(n: int, max_sweeps: int = 2000) -> Workload:
    """[CFG 4b] size sweep: cfg-2 WD without bubbles on an n x n half-plane grid, fixed sweeps."""
    w = wd_half_plane(n, 3.0, 0, seed=2, name=f"cfg4b_{n}")
    w.tol = 0.0
    w.max_sweeps = max_sweeps
    return w


def random_smooth(nr: int, nz: int, symmetry: int, seed: int, lmax: int = 8,
                  dr: float | None = None, dz: float | None = None) -> Workload:
    """Small generic test grid: a few seeded Gaussian clumps (positive density) + uniform floor."""
    dr = 1.0 / nr if dr is None else dr
    dz = dr if dz is None else dz
    r, z = cell_centres(nr, nz, dr, dz, symmetry)
    Lr, Lz = nr * dr, nz * dz
    rho = np.full((nz, nr), 1.0e-3)
    for k in range(5):
        A = uniform(seed, 7, 4 * k, 0.2, 1.0)
        w = uniform(seed, 7, 4 * k + 1, 0.05, 0.2) * min(Lr, Lz)
        rk = uniform(seed, 7, 4 * k + 2, 0.0, 0.6 * Lr)
        zk = uniform(seed, 7, 4 * k + 3, 0.0 if symmetry else -0.3 * Lz, 0.3 * Lz)
        rho += A * np.outer(np.exp(-((z - zk) ** 2) / (2 * w * w)),
                            np.exp(-((r - rk) ** 2) / (2 * w * w)))
    return Workload(f"smooth_{nr}x{nz}_s{symmetry}_{seed}", nr, nz, dr, dz, symmetry, lmax,
                    1e-10, 20000, np.ascontiguousarray(rho), meta={"seed": seed})


# ----------------------------------------------------------------------------
# NEXT-2: a flame front for the level-set re-initialisation ("An initial three-finger flame front is
# imposed, which is comparable with the c3 flame"; "500 grids in each direction")
# ----------------------------------------------------------------------------
def levelset_front(ncells: int = 500, seed: int = 7, distort: float = 0.5):
    """S on the (ncells+1)^2 cell CORNERS of the unit (r,z) quadrant, dr = dz = 1/ncells.  Zero contour: three fingers,
    s = R0 (1 + A cos(12 theta - pi)) (maxima at theta = pi/12, pi/4, 5 pi/12 from the z axis; dR/dtheta = 0 on the axis
    and on the equator).  S > 0 inside (ash).  The magnitude is distorted by a smooth seeded factor 1 + distort * u(r,z),
    |u| <= 1, so that |grad S| != 1 -- what an advection step leaves behind and re-initialisation has to repair.
    Returns (S, dr)."""
    n = ncells + 1
    dr = 1.0 / ncells
    x = np.arange(n) * dr
    X, Y = np.meshgrid(x, x)                      # X: r (fastest index), Y: z
    s = np.hypot(X, Y)
    theta = np.arctan2(X, Y)                      # from the +z axis
    R = 0.3 * (1.0 + 0.25 * np.cos(12.0 * theta - math.pi))
    u = np.zeros_like(s)
    for k in range(4):
        kx = uniform(seed, 1, 3 * k, 2.0, 9.0)
        ky = uniform(seed, 1, 3 * k + 1, 2.0, 9.0)
        ph = uniform(seed, 1, 3 * k + 2, 0.0, 2.0 * math.pi)
        u += 0.25 * np.sin(kx * X * math.pi + ph) * np.cos(ky * Y * math.pi)
    return np.ascontiguousarray((R - s) * (1.0 + distort * u)), dr


# ----------------------------------------------------------------------------
# NEXT-3: conserved hydro states for the WENO-5 / global Lax-Friedrichs flux reconstruction.  Inputs only:
# the conversion primitive -> conserved is the definition of the state vector ("tau = rho eps + rho v^2 / 2"
# with the gamma-law EOS of PAPER.md:402), not part of the method under test.
# ----------------------------------------------------------------------------
def hydro_state(rho, vr, vz, p, gamma: float = 1.4) -> np.ndarray:
    """U = (rho, rho v_r, rho v_z, tau) of shape (4, nz, nr) from primitive fields."""
    rho, vr, vz, p = np.broadcast_arrays(*(np.asarray(a, dtype=np.float64) for a in (rho, vr, vz, p)))
    return np.ascontiguousarray(np.stack([rho, rho * vr, rho * vz, p / (gamma - 1.0) + 0.5 * rho * (vr * vr + vz * vz)]))


def shock_tube(rho_l, v_l, p_l, rho_r, v_r, p_r, x0: float, n: int, rows: int = 1, axis: int = 0, gamma: float = 1.4):
    """Left / right states meeting at x0 on n cells of [0, 1] (the values of the paper's Table 3 are in
    tests/golden/paper_table3_shocktubes.txt), `rows` identical copies along the other axis.  Returns (U, dx)."""
    x = (np.arange(n) + 0.5) / n
    left = x < x0
    rho, v, p = np.where(left, rho_l, rho_r), np.where(left, v_l, v_r), np.where(left, p_l, p_r)
    if axis == 0:
        U = hydro_state(np.tile(rho, (rows, 1)), np.tile(v, (rows, 1)), 0.0, np.tile(p, (rows, 1)), gamma)
    else:
        U = hydro_state(np.tile(rho[:, None], (1, rows)), 0.0, np.tile(v[:, None], (1, rows)), np.tile(p[:, None], (1, rows)), gamma)
    return U, 1.0 / n


def hydro_blobs(nr: int = 500, nz: int = 500, seed: int = 11, gamma: float = 1.4, jump: float = 0.0):
    """2-D state on the unit (r, z) quadrant, dr = 1/nr, dz = 1/nz (the paper's hydro grids are 500 x 500):
    a smooth background with seeded Gaussian over-densities / over-pressures and a seeded smooth velocity field; `jump`
    > 0 adds a sharp circular density / pressure step (the nonlinear weights then matter).  Returns (U, dr, dz)."""
    dr, dz = 1.0 / nr, 1.0 / nz
    r = (np.arange(nr) + 0.5) * dr
    z = (np.arange(nz) + 0.5) * dz
    R, Z = np.meshgrid(r, z)
    rho = np.full((nz, nr), 1.0)
    p = np.full((nz, nr), 1.0)
    for k in range(6):
        A = uniform(seed, 21, 5 * k, 0.2, 1.5)
        w = uniform(seed, 21, 5 * k + 1, 0.04, 0.15)
        rk = uniform(seed, 21, 5 * k + 2, 0.1, 0.9)
        zk = uniform(seed, 21, 5 * k + 3, 0.1, 0.9)
        g = np.exp(-((R - rk) ** 2 + (Z - zk) ** 2) / (2 * w * w))
        rho += A * g
        p += uniform(seed, 21, 5 * k + 4, 0.5, 3.0) * A * g
    vr = 0.6 * np.sin(2 * math.pi * R * uniform(seed, 22, 0, 0.5, 2.0)) * np.cos(math.pi * Z * uniform(seed, 22, 1, 0.5, 2.0))
    vz = 0.6 * np.cos(math.pi * R * uniform(seed, 22, 2, 0.5, 2.0)) * np.sin(2 * math.pi * Z * uniform(seed, 22, 3, 0.5, 2.0))
    if jump > 0.0:
        inside = np.hypot(R - 0.4, Z - 0.45) < 0.2
        rho = np.where(inside, rho * (1.0 + jump), rho)
        p = np.where(inside, p * (1.0 + 3.0 * jump), p)
    return hydro_state(rho, vr, vz, p, gamma), dr, dz
