"""Thin ctypes binding over libsn_poisson.so -- same names as include/sn_poisson.h, argument marshalling only.

PyTorch is used by callers for device memory and streams (``tensor.data_ptr()``,
``torch.cuda.current_stream().cuda_stream``); nothing here computes anything.  There is no CPU fallback:
if the library is missing or no sm_100 device is usable the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsn_poisson.so")       # the in-tree build, always (no environment override)

# every symbol include/sn_poisson.h declares
EXPORTS = (
    "sn_poisson_create", "sn_poisson_solve", "sn_poisson_solve_host", "sn_poisson_solve_batch",
    "sn_poisson_solve_batch_host", "sn_poisson_solve_sequence_host", "sn_poisson_probe_l2",
    "sn_poisson_set_stop_rule", "sn_poisson_solve_gravity", "sn_poisson_solve_mg", "sn_poisson_solve_mg_host", "sn_poisson_solve_mg_batch",
    "sn_poisson_destroy", "sn_poisson_gravity", "sn_poisson_set_omega", "sn_poisson_get_omega", "sn_poisson_get_moments",
    "sn_poisson_set_boundary", "sn_poisson_get_boundary", "sn_poisson_get_history", "sn_poisson_set_option",
    "sn_poisson_get_stat", "sn_poisson_last_error", "sn_poisson_version", "sn_poisson_moments_static", "sn_poisson_solve_mg_batch_host",
)


# every symbol include/sn_levelset.h declares (NEXT-2)
EXPORTS_LEVELSET = (
    "sn_levelset_create", "sn_levelset_reinit", "sn_levelset_reinit_host", "sn_levelset_get_stat",
    "sn_levelset_destroy", "sn_levelset_last_error",
)


# every symbol include/sn_weno.h declares (NEXT-3)
EXPORTS_WENO = (
    "sn_weno_create", "sn_weno_max_speeds", "sn_weno_rhs", "sn_weno_step", "sn_weno_evolve", "sn_weno_rhs_host",
    "sn_weno_get_stat", "sn_weno_destroy", "sn_weno_last_error",
)


class sn_poisson_result(C.Structure):
    _fields_ = [("sweeps", C.c_int32), ("status", C.c_int32), ("residual", C.c_double)]

    def __repr__(self):
        return f"sn_poisson_result(sweeps={self.sweeps}, status={self.status}, residual={self.residual:.3e})"


class SnPoissonError(RuntimeError):
    pass


_lib = None
_vp = C.c_void_p
_dp = C.POINTER(C.c_double)


def load():
    """dlopen the library (built in-tree by ``paper_1507_08549_b200.build``).  Fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise SnPoissonError(f"{LIB_PATH} not found: run `python -c 'import __graft_entry__ as g; g.build()'` "
                             "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    lib.sn_poisson_create.restype = _vp
    lib.sn_poisson_create.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int]
    lib.sn_poisson_solve.restype = sn_poisson_result
    lib.sn_poisson_solve.argtypes = [_vp, _vp, _vp, C.c_double, C.c_int, _vp]
    lib.sn_poisson_solve_host.restype = sn_poisson_result
    lib.sn_poisson_solve_host.argtypes = [_vp, _vp, _vp, C.c_double, C.c_int, _vp]
    lib.sn_poisson_solve_mg.restype = sn_poisson_result
    lib.sn_poisson_solve_mg.argtypes = [_vp, _vp, _vp, C.c_double, C.c_int, _vp]
    lib.sn_poisson_solve_mg_batch.restype = C.c_int
    lib.sn_poisson_solve_mg_batch.argtypes = [_vp, C.c_int, _vp, _vp, C.c_double, C.c_int, _vp, C.POINTER(sn_poisson_result)]
    lib.sn_poisson_solve_mg_batch_host.restype = C.c_int
    lib.sn_poisson_solve_mg_batch_host.argtypes = [_vp, C.c_int, _vp, _vp, C.c_double, C.c_int, _vp,
                                                   C.POINTER(sn_poisson_result)]
    lib.sn_poisson_solve_mg_host.restype = sn_poisson_result
    lib.sn_poisson_solve_mg_host.argtypes = [_vp, _vp, _vp, C.c_double, C.c_int, _vp]
    lib.sn_poisson_solve_batch.restype = C.c_int
    lib.sn_poisson_solve_batch.argtypes = [_vp, C.c_int, _vp, _vp, C.c_double, C.c_int, _vp,
                                           C.POINTER(sn_poisson_result)]
    lib.sn_poisson_solve_batch_host.restype = C.c_int
    lib.sn_poisson_solve_batch_host.argtypes = [_vp, C.c_int, _vp, _vp, C.c_double, C.c_int, _vp,
                                                C.POINTER(sn_poisson_result)]
    lib.sn_poisson_solve_sequence_host.restype = C.c_int
    lib.sn_poisson_solve_sequence_host.argtypes = [_vp, C.c_int, _vp, _vp, _vp, C.c_double, C.c_int, _vp,
                                                   C.POINTER(sn_poisson_result)]
    lib.sn_poisson_probe_l2.restype = C.c_int
    lib.sn_poisson_probe_l2.argtypes = [C.c_int, _dp, _dp, _vp]
    lib.sn_poisson_destroy.restype = None
    lib.sn_poisson_destroy.argtypes = [_vp]
    lib.sn_poisson_gravity.restype = C.c_int
    lib.sn_poisson_gravity.argtypes = [_vp, C.c_int, _vp, _vp, _vp, _vp]
    lib.sn_poisson_solve_gravity.restype = C.c_int
    lib.sn_poisson_solve_gravity.argtypes = [_vp, C.c_int, _vp, _vp, _vp, _vp, C.c_double, C.c_int, _vp,
                                             C.POINTER(sn_poisson_result)]
    lib.sn_poisson_set_stop_rule.restype = C.c_int
    lib.sn_poisson_set_stop_rule.argtypes = [_vp, C.c_int]
    lib.sn_poisson_set_omega.restype = C.c_int
    lib.sn_poisson_set_omega.argtypes = [_vp, C.c_double]
    lib.sn_poisson_get_omega.restype = C.c_double
    lib.sn_poisson_get_omega.argtypes = [_vp]
    lib.sn_poisson_get_moments.restype = C.c_int
    lib.sn_poisson_get_moments.argtypes = [_vp, _dp]
    lib.sn_poisson_set_boundary.restype = C.c_int
    lib.sn_poisson_set_boundary.argtypes = [_vp, _dp, _dp, _dp]
    lib.sn_poisson_get_boundary.restype = C.c_int
    lib.sn_poisson_get_boundary.argtypes = [_vp, _dp, _dp, _dp]
    lib.sn_poisson_get_history.restype = C.c_int
    lib.sn_poisson_get_history.argtypes = [_vp, _dp, C.c_int]
    lib.sn_poisson_set_option.restype = C.c_int
    lib.sn_poisson_set_option.argtypes = [_vp, C.c_char_p, C.c_int64]
    lib.sn_poisson_get_stat.restype = C.c_int
    lib.sn_poisson_get_stat.argtypes = [_vp, C.c_char_p, _dp]
    lib.sn_poisson_last_error.restype = C.c_char_p
    lib.sn_poisson_last_error.argtypes = []
    lib.sn_poisson_version.restype = C.c_char_p
    lib.sn_poisson_version.argtypes = []
    lib.sn_poisson_moments_static.restype = C.c_int
    lib.sn_poisson_moments_static.argtypes = [_vp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int,
                                              _vp, _vp, _vp]
    lib.sn_levelset_create.restype = _vp
    lib.sn_levelset_create.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double]
    lib.sn_levelset_reinit.restype = C.c_int64
    lib.sn_levelset_reinit.argtypes = [_vp, _vp, _vp, _vp, _vp]
    lib.sn_levelset_reinit_host.restype = C.c_int64
    lib.sn_levelset_reinit_host.argtypes = [_vp, _vp, _vp, _vp, _vp]
    lib.sn_levelset_get_stat.restype = C.c_int
    lib.sn_levelset_get_stat.argtypes = [_vp, C.c_char_p, _dp]
    lib.sn_levelset_destroy.restype = None
    lib.sn_levelset_destroy.argtypes = [_vp]
    lib.sn_levelset_last_error.restype = C.c_char_p
    lib.sn_levelset_last_error.argtypes = []
    lib.sn_weno_create.restype = _vp
    lib.sn_weno_create.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.POINTER(C.c_int)]
    lib.sn_weno_max_speeds.restype = C.c_int
    lib.sn_weno_max_speeds.argtypes = [_vp, _vp, _dp, _vp]
    lib.sn_weno_rhs.restype = C.c_int
    lib.sn_weno_rhs.argtypes = [_vp, _vp, _vp, C.c_double, C.c_double, _vp]
    lib.sn_weno_step.restype = C.c_int
    lib.sn_weno_step.argtypes = [_vp, _vp, C.c_double, _dp, _vp]
    lib.sn_weno_evolve.restype = C.c_int
    lib.sn_weno_evolve.argtypes = [_vp, _vp, C.c_double, C.c_double, C.c_int, _vp]
    lib.sn_weno_rhs_host.restype = C.c_int
    lib.sn_weno_rhs_host.argtypes = [_vp, _vp, _vp, _vp]
    lib.sn_weno_get_stat.restype = C.c_int
    lib.sn_weno_get_stat.argtypes = [_vp, C.c_char_p, _dp]
    lib.sn_weno_destroy.restype = None
    lib.sn_weno_destroy.argtypes = [_vp]
    lib.sn_weno_last_error.restype = C.c_char_p
    lib.sn_weno_last_error.argtypes = []
    _lib = lib
    return lib


def sn_poisson_last_error() -> str:
    return load().sn_poisson_last_error().decode()


def sn_poisson_version() -> str:
    return load().sn_poisson_version().decode()


def sn_poisson_create(nr, nz, dr, dz, symmetry, lmax):
    """Returns an opaque handle (int) or raises SnPoissonError with the library's message."""
    h = load().sn_poisson_create(int(nr), int(nz), float(dr), float(dz), int(symmetry), int(lmax))
    if not h:
        raise SnPoissonError("sn_poisson_create failed: " + sn_poisson_last_error())
    return h


def sn_poisson_destroy(h):
    load().sn_poisson_destroy(h)


def sn_poisson_solve(h, rho_ptr, phi_ptr, tol, max_sweeps, stream=0) -> sn_poisson_result:
    """rho_ptr / phi_ptr: DEVICE addresses (ints, e.g. tensor.data_ptr()); stream: cudaStream_t as int."""
    return load().sn_poisson_solve(h, rho_ptr, phi_ptr, float(tol), int(max_sweeps), stream or None)


def sn_poisson_solve_host(h, rho_ptr, phi_ptr, tol, max_sweeps, stream=0) -> sn_poisson_result:
    """rho_ptr / phi_ptr: HOST addresses (ints, e.g. numpy ``arr.ctypes.data`` or a pinned tensor's data_ptr())."""
    return load().sn_poisson_solve_host(h, rho_ptr, phi_ptr, float(tol), int(max_sweeps), stream or None)


def sn_poisson_solve_mg(h, rho_ptr, phi_ptr, tol, max_cycles, stream=0) -> sn_poisson_result:
    """Multigrid variant (NEXT-4); DEVICE addresses; `sweeps` of the result = V-cycles."""
    return load().sn_poisson_solve_mg(h, rho_ptr, phi_ptr, float(tol), int(max_cycles), stream or None)


def sn_poisson_solve_mg_batch(h, nbatch, rho_ptr, phi_ptr, tol, max_cycles, stream=0):
    """Multigrid variant, nbatch independent solves; returns a list of sn_poisson_result."""
    out = (sn_poisson_result * int(nbatch))()
    rc = load().sn_poisson_solve_mg_batch(h, int(nbatch), rho_ptr, phi_ptr, float(tol), int(max_cycles), stream or None, out)
    if rc != 0:
        raise SnPoissonError(f"sn_poisson_solve_mg_batch failed ({rc}): " + sn_poisson_last_error())
    return list(out)


def sn_poisson_solve_mg_batch_host(h, nbatch, rho_ptr, phi_ptr, tol, max_cycles, stream=0):
    """Multigrid variant, nbatch independent solves, HOST addresses; returns a list of sn_poisson_result."""
    out = (sn_poisson_result * int(nbatch))()
    rc = load().sn_poisson_solve_mg_batch_host(h, int(nbatch), rho_ptr, phi_ptr, float(tol), int(max_cycles),
                                               stream or None, out)
    if rc != 0:
        raise SnPoissonError(f"sn_poisson_solve_mg_batch_host failed ({rc}): " + sn_poisson_last_error())
    return list(out)


def sn_poisson_solve_mg_host(h, rho_ptr, phi_ptr, tol, max_cycles, stream=0) -> sn_poisson_result:
    """Multigrid variant (NEXT-4); HOST addresses."""
    return load().sn_poisson_solve_mg_host(h, rho_ptr, phi_ptr, float(tol), int(max_cycles), stream or None)


def sn_poisson_solve_batch(h, nbatch, rho_ptr, phi_ptr, tol, max_sweeps, stream=0):
    out = (sn_poisson_result * int(nbatch))()
    rc = load().sn_poisson_solve_batch(h, int(nbatch), rho_ptr, phi_ptr, float(tol), int(max_sweeps),
                                       stream or None, out)
    if rc != 0:
        raise SnPoissonError(f"sn_poisson_solve_batch failed ({rc}): " + sn_poisson_last_error())
    return list(out)


def sn_poisson_solve_batch_host(h, nbatch, rho_ptr, phi_ptr, tol, max_sweeps, stream=0):
    """rho_ptr / phi_ptr: HOST addresses of nbatch consecutive grids."""
    out = (sn_poisson_result * int(nbatch))()
    rc = load().sn_poisson_solve_batch_host(h, int(nbatch), rho_ptr, phi_ptr, float(tol), int(max_sweeps),
                                            stream or None, out)
    if rc != 0:
        raise SnPoissonError(f"sn_poisson_solve_batch_host failed ({rc}): " + sn_poisson_last_error())
    return list(out)


def sn_poisson_solve_sequence_host(h, nsteps, rho_seq_ptr, phi_ptr, phi_seq_ptr, tol, max_sweeps, stream=0):
    """HOST addresses: rho_seq [nsteps][ncell], phi [ncell] in/out, phi_seq [nsteps][ncell] or 0."""
    out = (sn_poisson_result * int(nsteps))()
    for o in out:
        o.status = -1
    rc = load().sn_poisson_solve_sequence_host(h, int(nsteps), rho_seq_ptr, phi_ptr, phi_seq_ptr or None, float(tol),
                                               int(max_sweeps), stream or None, out)
    if rc != 0:
        raise SnPoissonError(f"sn_poisson_solve_sequence_host failed ({rc}): " + sn_poisson_last_error())
    return list(out)


def sn_poisson_probe_l2(mib=32, stream=0):
    """(copy GB/s, read GB/s) of an L2-resident working set, measured by the library's own probe kernels."""
    c, r = C.c_double(0.0), C.c_double(0.0)
    _check(load().sn_poisson_probe_l2(int(mib), C.byref(c), C.byref(r), stream or None), "sn_poisson_probe_l2")
    return c.value, r.value


def sn_poisson_solve_gravity(h, nbatch, rho_ptr, phi_ptr, gr_ptr, gz_ptr, tol, max_sweeps, stream=0):
    """Solve + fused gravity epilogue; DEVICE addresses of nbatch consecutive grids.  Returns the list of results."""
    out = (sn_poisson_result * int(nbatch))()
    rc = load().sn_poisson_solve_gravity(h, int(nbatch), rho_ptr, phi_ptr, gr_ptr, gz_ptr, float(tol), int(max_sweeps),
                                         stream or None, out)
    if rc != 0:
        raise SnPoissonError(f"sn_poisson_solve_gravity failed ({rc}): " + sn_poisson_last_error())
    return list(out)


def sn_poisson_gravity(h, nbatch, phi_ptr, gr_ptr, gz_ptr, stream=0):
    rc = load().sn_poisson_gravity(h, int(nbatch), phi_ptr, gr_ptr, gz_ptr, stream or None)
    if rc != 0:
        raise SnPoissonError(f"sn_poisson_gravity failed ({rc}): " + sn_poisson_last_error())
    return rc


def sn_poisson_set_stop_rule(h, rule) -> int:
    """0 = residual ratio R_k (R9), 1 = the paper-literal relative change E_k (R16)."""
    return _check(load().sn_poisson_set_stop_rule(h, int(rule)), "sn_poisson_set_stop_rule")


def sn_poisson_set_omega(h, omega) -> int:
    return load().sn_poisson_set_omega(h, float(omega))


def sn_poisson_get_omega(h) -> float:
    return load().sn_poisson_get_omega(h)


def _check(rc, what):
    if rc < 0:
        raise SnPoissonError(f"{what} failed ({rc}): " + sn_poisson_last_error())
    return rc


def sn_poisson_get_moments(h, lmax):
    import numpy as np
    M = np.zeros(lmax + 1)
    _check(load().sn_poisson_get_moments(h, M.ctypes.data_as(_dp)), "sn_poisson_get_moments")
    return M


def sn_poisson_moments_static(rho_ptr, nbatch, nr, nz, dr, dz, symmetry, lmax, m_out_ptr, maxf_out_ptr=0, stream=0) -> int:
    """Multipole moments for hosts that may not allocate device memory (all of it handed to their own pool, or a
    time-step loop that cannot take a cudaMalloc stall): no handle, scratch in an array built into the library.
    DEVICE addresses: rho [nbatch][nz][nr], m_out [nbatch][lmax + 1], maxf_out [nbatch] or 0.  Enqueues on `stream`
    and returns; sizes beyond the fixed scratch raise.  Calls that overlap on the GPU race (include/sn_poisson.h)."""
    return _check(load().sn_poisson_moments_static(rho_ptr, int(nbatch), int(nr), int(nz), float(dr), float(dz),
                                                   int(symmetry), int(lmax), m_out_ptr, maxf_out_ptr or None,
                                                   stream or None), "sn_poisson_moments_static")


def sn_poisson_set_boundary(h, bE, bN, bS=None):
    import numpy as np
    if bE is None:
        return _check(load().sn_poisson_set_boundary(h, None, None, None), "sn_poisson_set_boundary")
    bE = np.ascontiguousarray(bE, dtype=np.float64)
    bN = np.ascontiguousarray(bN, dtype=np.float64)
    bSp = None
    if bS is not None:
        bS = np.ascontiguousarray(bS, dtype=np.float64)
        bSp = bS.ctypes.data_as(_dp)
    return _check(load().sn_poisson_set_boundary(h, bE.ctypes.data_as(_dp), bN.ctypes.data_as(_dp), bSp),
                  "sn_poisson_set_boundary")


def sn_poisson_get_boundary(h, nr, nz, symmetry):
    import numpy as np
    bE, bN, bS = np.zeros(nz), np.zeros(nr), np.zeros(nr)
    _check(load().sn_poisson_get_boundary(h, bE.ctypes.data_as(_dp), bN.ctypes.data_as(_dp),
                                          bS.ctypes.data_as(_dp)), "sn_poisson_get_boundary")
    return bE, bN, (bS if symmetry == 0 else None)


def sn_poisson_get_history(h, n):
    import numpy as np
    R = np.zeros(max(int(n), 1))
    m = _check(load().sn_poisson_get_history(h, R.ctypes.data_as(_dp), int(n)), "sn_poisson_get_history")
    return R[:m]


def sn_poisson_set_option(h, key: str, value: int) -> int:
    return _check(load().sn_poisson_set_option(h, key.encode(), int(value)), f"sn_poisson_set_option({key})")


def sn_poisson_get_stat(h, key: str) -> float:
    out = C.c_double(0.0)
    _check(load().sn_poisson_get_stat(h, key.encode(), C.byref(out)), f"sn_poisson_get_stat({key})")
    return out.value


# ---- NEXT-2: level-set re-initialisation (include/sn_levelset.h) ------------------------------------------------------
def sn_levelset_last_error() -> str:
    return load().sn_levelset_last_error().decode()


def sn_levelset_create(nx, ny, dr, dz, delta):
    h = load().sn_levelset_create(int(nx), int(ny), float(dr), float(dz), float(delta))
    if not h:
        raise SnPoissonError("sn_levelset_create failed: " + sn_levelset_last_error())
    return h


def sn_levelset_destroy(h):
    load().sn_levelset_destroy(h)


def sn_levelset_reinit(h, s_old_ptr, s_new_ptr, dist_ptr=0, stream=0) -> int:
    """DEVICE addresses; returns the number of crossings."""
    n = load().sn_levelset_reinit(h, s_old_ptr, s_new_ptr, dist_ptr or None, stream or None)
    if n < 0:
        raise SnPoissonError(f"sn_levelset_reinit failed ({n}): " + sn_levelset_last_error())
    return n


def sn_levelset_reinit_host(h, s_old_ptr, s_new_ptr, dist_ptr=0, stream=0) -> int:
    """HOST addresses; returns the number of crossings."""
    n = load().sn_levelset_reinit_host(h, s_old_ptr, s_new_ptr, dist_ptr or None, stream or None)
    if n < 0:
        raise SnPoissonError(f"sn_levelset_reinit_host failed ({n}): " + sn_levelset_last_error())
    return n


def sn_levelset_get_stat(h, key: str) -> float:
    out = C.c_double(0.0)
    if load().sn_levelset_get_stat(h, key.encode(), C.byref(out)) != 0:
        raise SnPoissonError("sn_levelset_get_stat: " + sn_levelset_last_error())
    return out.value


# ---- NEXT-3: WENO-5 / global Lax-Friedrichs flux reconstruction (include/sn_weno.h) ------------------------------------
def sn_weno_last_error() -> str:
    return load().sn_weno_last_error().decode()


def _wcheck(rc, what):
    if rc < 0:
        raise SnPoissonError(f"{what} failed ({rc}): " + sn_weno_last_error())
    return rc


def sn_weno_create(nr, nz, dr, dz, gamma, bc):
    h = load().sn_weno_create(int(nr), int(nz), float(dr), float(dz), float(gamma), (C.c_int * 4)(*[int(b) for b in bc]))
    if not h:
        raise SnPoissonError("sn_weno_create failed: " + sn_weno_last_error())
    return h


def sn_weno_destroy(h):
    load().sn_weno_destroy(h)


def sn_weno_max_speeds(h, u_ptr, stream=0):
    a = (C.c_double * 2)()
    _wcheck(load().sn_weno_max_speeds(h, u_ptr, a, stream or None), "sn_weno_max_speeds")
    return a[0], a[1]


def sn_weno_rhs(h, u_ptr, l_ptr, alpha_r=-1.0, alpha_z=-1.0, stream=0) -> int:
    return _wcheck(load().sn_weno_rhs(h, u_ptr, l_ptr, float(alpha_r), float(alpha_z), stream or None), "sn_weno_rhs")


def sn_weno_step(h, u_ptr, cfl, stream=0, want_dt=True):
    dt = C.c_double(0.0)
    _wcheck(load().sn_weno_step(h, u_ptr, float(cfl), C.byref(dt) if want_dt else None, stream or None), "sn_weno_step")
    return dt.value if want_dt else None


def sn_weno_evolve(h, u_ptr, cfl, t_end, max_steps, stream=0) -> int:
    return _wcheck(load().sn_weno_evolve(h, u_ptr, float(cfl), float(t_end), int(max_steps), stream or None),
                   "sn_weno_evolve")


def sn_weno_rhs_host(h, u_host_ptr, l_host_ptr, stream=0) -> int:
    return _wcheck(load().sn_weno_rhs_host(h, u_host_ptr, l_host_ptr, stream or None), "sn_weno_rhs_host")


def sn_weno_get_stat(h, key: str) -> float:
    out = C.c_double(0.0)
    _wcheck(load().sn_weno_get_stat(h, key.encode(), C.byref(out)), f"sn_weno_get_stat({key})")
    return out.value
