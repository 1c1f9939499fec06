"""ctypes loader for the CPU oracle (oracle/sn_oracle.cpp).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this
package.  It imports nothing from paper_1507_08549_b200 and the product never imports it.
Argument marshalling only: every number comes out of sn_oracle.cpp.
"""
from __future__ import annotations

import ctypes as C
import os
import platform
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sn_oracle.cpp")
_LIB = os.path.join(_HERE, "libsn_oracle.so")
CXXFLAGS = ["-O2", "-ffp-contract=off", "-fPIC", "-shared", "-std=c++17"]
if platform.machine() in ("x86_64", "AMD64"):
    CXXFLAGS.insert(2, "-mfma")              # std::fma as one instruction; aarch64 has fused multiply-add in the base ISA

_lib = None
_dp = C.POINTER(C.c_double)


_EXTRA = {name: (os.path.join(_HERE, name + "_oracle.cpp"), os.path.join(_HERE, "lib" + name + "_oracle.so"))
          for name in ("levelset", "weno", "mg")}
_extra_libs = {}


def _compile(src, lib, force):
    if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(src):
        subprocess.check_call(["g++", *CXXFLAGS, "-o", lib, src])
    return lib


def build(force: bool = False) -> str:
    """Compile every oracle with g++ (one translation unit, one shared library each)."""
    _compile(_SRC, _LIB, force)
    for src, lib in _EXTRA.values():
        if os.path.exists(src):
            _compile(src, lib, force)
    return _LIB


def extra_lib(name):
    """ctypes handle of oracle/<name>_oracle.cpp (NEXT rows: level-set re-initialisation, WENO)."""
    if name not in _extra_libs:
        src, lib = _EXTRA[name]
        _extra_libs[name] = C.CDLL(_compile(src, lib, False))
    return _extra_libs[name]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.sno_default_omega.restype = C.c_double
        _lib.sno_default_omega.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_int]
        _lib.sno_ratio.restype = C.c_double
        _lib.sno_ratio.argtypes = [C.c_double] * 5
        _lib.sno_regular_harmonics.argtypes = [C.c_double, C.c_double, C.c_int, _dp]
        _lib.sno_irregular_harmonics.argtypes = [C.c_double, C.c_double, C.c_int, _dp]
        _lib.sno_moments.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int, _dp, _dp]
        _lib.sno_boundary.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int, _dp, _dp, _dp, _dp]
        _lib.sno_sweeps.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, C.c_double, _dp, _dp, _dp,
                                    _dp, _dp, C.c_int, _dp, _dp]
        _lib.sno_solve.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int, C.c_double, _dp,
                                   _dp, C.c_double, C.c_int, C.POINTER(C.c_int), _dp, _dp, _dp, _dp, _dp]
        _lib.sno_solve_rule.argtypes = [C.c_int] + _lib.sno_solve.argtypes
        _lib.sno_sweeps_chg.argtypes = _lib.sno_sweeps.argtypes + [_dp]
        _lib.sno_relchange.restype = C.c_double
        _lib.sno_relchange.argtypes = [C.c_double, C.c_double]
        _lib.sno_gravity.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, _dp, _dp, _dp, _dp, _dp, _dp]
        _lib.sno_apply_operator.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, _dp, _dp, _dp,
                                            _dp, _dp]
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def default_omega(nr, nz, dr, dz, symmetry) -> float:
    return lib().sno_default_omega(nr, nz, dr, dz, symmetry)


def ratio(Rabs, P, maxf, dr, dz) -> float:
    return lib().sno_ratio(Rabs, P, maxf, dr, dz)


def regular_harmonics(x, y, lmax):
    out = np.zeros(lmax + 2)
    lib().sno_regular_harmonics(x, y, lmax, _p(out))
    return out[: lmax + 1]


def irregular_harmonics(x, y, lmax):
    out = np.zeros(lmax + 2)
    lib().sno_irregular_harmonics(x, y, lmax, _p(out))
    return out[: lmax + 1]


def moments(rho, dr, dz, symmetry, lmax):
    rho = _f64(rho)
    nz, nr = rho.shape
    M = np.zeros(lmax + 1)
    rc = lib().sno_moments(nr, nz, dr, dz, symmetry, lmax, _p(rho), _p(M))
    assert rc == 0
    return M


def boundary(nr, nz, dr, dz, symmetry, lmax, M):
    M = _f64(M)
    bE, bN, bS = np.zeros(nz), np.zeros(nr), np.zeros(nr)
    rc = lib().sno_boundary(nr, nz, dr, dz, symmetry, lmax, _p(M), _p(bE), _p(bN), _p(bS))
    assert rc == 0
    return bE, bN, (bS if symmetry == 0 else None)


def sweeps(rho, phi, dr, dz, symmetry, omega, bE, bN, bS, nsweeps):
    """nsweeps red-black SOR sweeps; returns (phi_new, Rabs[nsweeps], P[nsweeps])."""
    rho = _f64(rho)
    nz, nr = rho.shape
    phi = np.array(phi, dtype=np.float64, order="C", copy=True)
    bE, bN = _f64(bE), _f64(bN)
    bS = _f64(bS) if bS is not None else np.zeros(nr)
    Rabs, P = np.zeros(max(nsweeps, 1)), np.zeros(max(nsweeps, 1))
    rc = lib().sno_sweeps(nr, nz, dr, dz, symmetry, omega, _p(rho), _p(bE), _p(bN), _p(bS), _p(phi), nsweeps,
                          _p(Rabs), _p(P))
    assert rc == 0
    return phi, Rabs[:nsweeps], P[:nsweeps]


def sweeps_chg(rho, phi, dr, dz, symmetry, omega, bE, bN, bS, nsweeps):
    """sweeps() plus Chg[k] = max |w_j res| of every sweep (R16).  Returns (phi_new, Rabs, P, Chg)."""
    rho = _f64(rho)
    nz, nr = rho.shape
    phi = np.array(phi, dtype=np.float64, order="C", copy=True)
    bE, bN = _f64(bE), _f64(bN)
    bS = _f64(bS) if bS is not None else np.zeros(nr)
    n = max(nsweeps, 1)
    Rabs, P, Chg = np.zeros(n), np.zeros(n), np.zeros(n)
    rc = lib().sno_sweeps_chg(nr, nz, dr, dz, symmetry, omega, _p(rho), _p(bE), _p(bN), _p(bS), _p(phi), nsweeps,
                              _p(Rabs), _p(P), _p(Chg))
    assert rc == 0
    return phi, Rabs[:nsweeps], P[:nsweeps], Chg[:nsweeps]


def relchange(Chg, P) -> float:
    return lib().sno_relchange(Chg, P)


def solve(rho, phi0, dr, dz, symmetry, lmax, tol, max_sweeps, omega=None, boundary_arrays=None,
          history=False, rule=0):
    """Whole path.  rule 0: residual rule R9; rule 1: the paper-literal relative-change rule R16.
    Returns dict(phi, sweeps, residual, status[, hist])."""
    rho = _f64(rho)
    nz, nr = rho.shape
    phi = np.array(phi0, dtype=np.float64, order="C", copy=True)
    nsw, res = C.c_int(0), C.c_double(0.0)
    hist = np.zeros(max(max_sweeps, 1)) if history else None
    bE = bN = bS = None
    if boundary_arrays is not None:
        bE, bN, bS = boundary_arrays
        bE, bN = _f64(bE), _f64(bN)
        bS = _f64(bS) if bS is not None else np.zeros(nr)
    rc = lib().sno_solve_rule(int(rule), nr, nz, dr, dz, symmetry, lmax, -1.0 if omega is None else float(omega),
                              _p(rho), _p(phi), tol, max_sweeps, C.byref(nsw), C.byref(res), _p(hist), _p(bE), _p(bN),
                              _p(bS))
    out = {"phi": phi, "sweeps": nsw.value, "residual": res.value, "status": rc}
    if history:
        out["hist"] = hist[: nsw.value]
    return out


def apply_operator(phi, dr, dz, symmetry, bE, bN, bS):
    phi = _f64(phi)
    nz, nr = phi.shape
    bS = _f64(bS) if bS is not None else np.zeros(nr)
    out = np.zeros_like(phi)
    lib().sno_apply_operator(nr, nz, dr, dz, symmetry, _p(phi), _p(_f64(bE)), _p(_f64(bN)), _p(bS), _p(out))
    return out


def gravity(phi, dr, dz, symmetry, bE, bN, bS):
    """(g_r, g_z) = -grad phi at the cell centres (R15)."""
    phi = _f64(phi)
    nz, nr = phi.shape
    bS = _f64(bS) if bS is not None else np.zeros(nr)
    gr, gz = np.zeros_like(phi), np.zeros_like(phi)
    lib().sno_gravity(nr, nz, dr, dz, symmetry, _p(phi), _p(_f64(bE)), _p(_f64(bN)), _p(bS), _p(gr), _p(gz))
    return gr, gz


def solve_workload(w, phi0=None, history=False):
    """Convenience: run the whole path on a workloads.Workload."""
    phi0 = np.zeros_like(w.rho) if phi0 is None else phi0
    return solve(w.rho, phi0, w.dr, w.dz, w.symmetry, w.lmax, w.tol, w.max_sweeps, omega=w.omega,
                 history=history)


# ---- NEXT-2: level-set re-initialisation (oracle/levelset_oracle.cpp) ------------------------------------------------
def _ls():
    L = extra_lib("levelset")
    L.lso_H.restype = C.c_double
    L.lso_H.argtypes = [C.c_double, C.c_double]
    L.lso_crossings.restype = C.c_long
    L.lso_crossings.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, _dp, _dp, _dp]
    L.lso_reinit.restype = C.c_long
    L.lso_reinit.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, _dp, _dp, _dp]
    return L


def levelset_H(d, delta) -> float:
    return _ls().lso_H(float(d), float(delta))


def levelset_crossings(S, dr, dz):
    """(cx, cy) of every grid-edge crossing of the zero contour, in the oracle's enumeration order."""
    S = _f64(S)
    ny, nx = S.shape
    cx, cy = np.zeros(2 * nx * ny), np.zeros(2 * nx * ny)
    n = _ls().lso_crossings(nx, ny, dr, dz, _p(S), _p(cx), _p(cy))
    return cx[:n].copy(), cy[:n].copy()


def levelset_reinit(S, dr, dz, delta=None):
    """Returns dict(S=S_new, dist=signed minimum distance, crossings=count)."""
    S = _f64(S)
    ny, nx = S.shape
    out, dist = np.zeros_like(S), np.zeros_like(S)
    n = _ls().lso_reinit(nx, ny, dr, dz, dr if delta is None else delta, _p(S), _p(out), _p(dist))
    assert n >= 0
    return {"S": out, "dist": dist, "crossings": int(n)}


# ---- NEXT-3: WENO-5 / global Lax-Friedrichs flux reconstruction (oracle/weno_oracle.cpp) ----------------------------
_ip = C.POINTER(C.c_int)


def _wn():
    L = extra_lib("weno")
    L.wno_weno5.restype = C.c_double
    L.wno_weno5.argtypes = [C.c_double] * 5
    L.wno_candidates.argtypes = [C.c_double] * 5 + [_dp, _dp]
    L.wno_max_speeds.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, _ip, _dp, _dp, _dp]
    L.wno_rhs.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, _ip, _dp, C.c_double, C.c_double, _dp]
    L.wno_face_fluxes.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, _ip, _dp, _dp, _dp]
    L.wno_step.restype = C.c_double
    L.wno_step.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, _ip, C.c_double, _dp]
    L.wno_evolve.restype = C.c_int
    L.wno_evolve.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, _ip, C.c_double, C.c_double,
                             C.c_int, _dp]
    return L


def _bc(bc):
    return (C.c_int * 4)(*[int(b) for b in bc])


def weno5(a, b, c, d, e) -> float:
    return _wn().wno_weno5(float(a), float(b), float(c), float(d), float(e))


def weno_candidates(a, b, c, d, e):
    q, beta = np.zeros(3), np.zeros(3)
    _wn().wno_candidates(float(a), float(b), float(c), float(d), float(e), _p(q), _p(beta))
    return q, beta


def _u4(U):
    U = _f64(U)
    assert U.ndim == 3 and U.shape[0] == 4, "U must be (4, nz, nr)"
    return U


def weno_max_speeds(U, dr, dz, gamma, bc):
    U = _u4(U)
    ar, az = C.c_double(), C.c_double()
    _wn().wno_max_speeds(U.shape[2], U.shape[1], dr, dz, gamma, _bc(bc), _p(U), C.byref(ar), C.byref(az))
    return ar.value, az.value


def weno_rhs(U, dr, dz, gamma, bc, alpha=None):
    """L(U) = -(dF/dr + dG/dz) (W6); alpha = (alpha_r, alpha_z) or None for the global maxima of U (W4)."""
    U = _u4(U)
    L = np.zeros_like(U)
    ar, az = (-1.0, -1.0) if alpha is None else alpha
    _wn().wno_rhs(U.shape[2], U.shape[1], dr, dz, gamma, _bc(bc), _p(U), ar, az, _p(L))
    return L


def weno_face_fluxes(U, dr, dz, gamma, bc):
    U = _u4(U)
    F, G = np.zeros_like(U), np.zeros_like(U)
    _wn().wno_face_fluxes(U.shape[2], U.shape[1], dr, dz, gamma, _bc(bc), _p(U), _p(F), _p(G))
    return F, G


def weno_step(U, dr, dz, gamma, bc, cfl):
    """One SSP-RK3 step (W8) on a copy; returns (U_new, dt)."""
    U = _u4(U).copy()
    dt = _wn().wno_step(U.shape[2], U.shape[1], dr, dz, gamma, _bc(bc), cfl, _p(U))
    return U, dt


def weno_evolve(U, dr, dz, gamma, bc, cfl, t_end, max_steps=1000000):
    U = _u4(U).copy()
    n = _wn().wno_evolve(U.shape[2], U.shape[1], dr, dz, gamma, _bc(bc), cfl, t_end, max_steps, _p(U))
    return U, n


# ---- NEXT-4: red-black-smoothed multigrid variant of the Poisson solve (oracle/mg_oracle.cpp) ------------------------
def _mg():
    L = extra_lib("mg")
    L.mgo_levels.restype = C.c_int
    L.mgo_levels.argtypes = [C.c_int, C.c_int]
    L.mgo_beta.restype = C.c_double
    L.mgo_beta.argtypes = [C.c_int]
    L.mgo_restrict.argtypes = [C.c_int, C.c_int, _dp, _dp]
    L.mgo_prolong.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, _dp, _dp]
    L.mgo_solve.restype = C.c_int
    L.mgo_solve.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, _dp, _dp, _dp, _dp, _dp, C.c_double,
                            C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int), _dp, _dp]
    return L


def mg_levels(nr, nz) -> int:
    return _mg().mgo_levels(int(nr), int(nz))


def mg_beta(l) -> float:
    return _mg().mgo_beta(int(l))


def mg_restrict(res):
    res = _f64(res)
    nz, nr = res.shape
    out = np.zeros((nz // 2, nr // 2))
    _mg().mgo_restrict(nr, nz, _p(res), _p(out))
    return out


def mg_prolong(ec, symmetry, lc):
    """Bilinear prolongation (M7) of the level-lc error ec onto a zero fine field."""
    ec = _f64(ec)
    nzc, nrc = ec.shape
    out = np.zeros((2 * nzc, 2 * nrc))
    _mg().mgo_prolong(nrc, nzc, int(symmetry), int(lc), _p(ec), _p(out))
    return out


def mg_solve(rho, phi0, dr, dz, symmetry, lmax, tol, max_cycles, nu1=1, nu2=1, nc=12, ghosts=None):
    """Multigrid solve (M1-M8) with the multipole ghosts of the SOR oracle (or the given (bE, bN, bS)).
    Returns dict(phi, cycles, status, residual, history)."""
    rho, phi = _f64(rho), _f64(phi0).copy()
    nz, nr = rho.shape
    if ghosts is None:
        M = moments(rho, dr, dz, symmetry, lmax)
        ghosts = boundary(nr, nz, dr, dz, symmetry, lmax, M)
    bE, bN, bS = (_f64(g) if g is not None else np.zeros(nr) for g in ghosts)
    cyc, R = C.c_int(0), C.c_double(0.0)
    hist = np.zeros(max(1, max_cycles))
    st = _mg().mgo_solve(nr, nz, dr, dz, symmetry, _p(rho), _p(bE), _p(bN), _p(bS), _p(phi), tol, max_cycles, nu1, nu2,
                         nc, C.byref(cyc), C.byref(R), _p(hist))
    assert st >= -3 and st != -1, "bad argument"
    return {"phi": phi, "cycles": cyc.value, "status": st, "residual": R.value, "history": hist[:cyc.value].copy()}


def mg_solve_workload(w, phi0=None, **kw):
    phi0 = np.zeros_like(w.rho) if phi0 is None else phi0
    return mg_solve(w.rho, phi0, w.dr, w.dz, w.symmetry, w.lmax, w.tol, kw.pop("max_cycles", 60), **kw)
