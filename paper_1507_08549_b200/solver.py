"""Convenience wrapper: torch tensors in, torch tensors out; pointer / stream marshalling only."""
from __future__ import annotations

from . import binding as B


class PoissonSolver:
    """Owns one sn_poisson handle.  ``rho`` / ``phi`` are float64 CUDA tensors of shape (nz, nr) or (nbatch, nz, nr)."""

    def __init__(self, nr, nz, dr, dz, symmetry, lmax, omega=None):
        self.nr, self.nz, self.dr, self.dz, self.symmetry, self.lmax = nr, nz, dr, dz, symmetry, lmax
        self.h = B.sn_poisson_create(nr, nz, dr, dz, symmetry, lmax)
        if omega is not None:
            if B.sn_poisson_set_omega(self.h, omega) != 0:
                raise B.SnPoissonError(B.sn_poisson_last_error())

    @classmethod
    def for_workload(cls, w):
        return cls(w.nr, w.nz, w.dr, w.dz, w.symmetry, w.lmax, omega=w.omega)

    def close(self):
        if getattr(self, "h", None) and getattr(B, "sn_poisson_destroy", None):     # B is torn down at interpreter exit
            B.sn_poisson_destroy(self.h)
            self.h = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def _check(self, t):
        import torch
        if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
            raise ValueError("expected a contiguous float64 CUDA tensor")

    @staticmethod
    def _raise_if_failed(results, what):
        """Same rule for single solves, batches and sequences: any status < 0 raises; the results ride on the error."""
        bad = [(i, r.status) for i, r in enumerate(results) if r.status < 0]
        if bad:
            e = B.SnPoissonError(f"{what}: status {bad[0][1]} (member/step {bad[0][0]}): {B.sn_poisson_last_error()}")
            e.results = list(results)
            raise e

    def solve(self, rho, phi, tol, max_sweeps):
        """In-place on ``phi``.  Returns sn_poisson_result (or a list for a 3-D batch)."""
        import torch
        self._check(rho)
        self._check(phi)
        stream = torch.cuda.current_stream().cuda_stream
        if rho.dim() == 3:
            if rho.shape != phi.shape or tuple(rho.shape[1:]) != (self.nz, self.nr):
                raise ValueError("shape mismatch")
            res = B.sn_poisson_solve_batch(self.h, rho.shape[0], rho.data_ptr(), phi.data_ptr(), tol, max_sweeps,
                                           stream)
            self._raise_if_failed(res, "sn_poisson_solve_batch")
            return res
        if tuple(rho.shape) != (self.nz, self.nr) or rho.shape != phi.shape:
            raise ValueError("shape mismatch")
        r = B.sn_poisson_solve(self.h, rho.data_ptr(), phi.data_ptr(), tol, max_sweeps, stream)
        self._raise_if_failed([r], "sn_poisson_solve")
        return r

    def solve_mg(self, rho, phi, tol, max_cycles=60):
        """Multigrid variant (NEXT-4): in place on ``phi``; the result's ``sweeps`` counts V-cycles."""
        import torch
        self._check(rho)
        self._check(phi)
        if rho.dim() == 3:
            if rho.shape != phi.shape or tuple(rho.shape[1:]) != (self.nz, self.nr):
                raise ValueError("shape mismatch")
            res = B.sn_poisson_solve_mg_batch(self.h, rho.shape[0], rho.data_ptr(), phi.data_ptr(), tol, max_cycles,
                                              torch.cuda.current_stream().cuda_stream)
            self._raise_if_failed(res, "sn_poisson_solve_mg_batch")
            return res
        if tuple(rho.shape) != (self.nz, self.nr) or rho.shape != phi.shape:
            raise ValueError("shape mismatch")
        r = B.sn_poisson_solve_mg(self.h, rho.data_ptr(), phi.data_ptr(), tol, max_cycles,
                                  torch.cuda.current_stream().cuda_stream)
        self._raise_if_failed([r], "sn_poisson_solve_mg")
        return r

    def solve_mg_host(self, rho_np, phi_np, tol, max_cycles=60):
        """HOST arrays, (nz, nr) -> one result, or (nbatch, nz, nr) -> a list (sn_poisson_solve_mg_batch_host)."""
        import torch
        if getattr(rho_np, "ndim", 0) == 3:
            nb = rho_np.shape[0]
            self._check_host(rho_np, (nb, self.nz, self.nr))
            self._check_host(phi_np, (nb, self.nz, self.nr), writeable=True)
            res = B.sn_poisson_solve_mg_batch_host(self.h, nb, rho_np.ctypes.data, phi_np.ctypes.data, tol, max_cycles,
                                                   torch.cuda.current_stream().cuda_stream)
            self._raise_if_failed(res, "sn_poisson_solve_mg_batch_host")
            return res
        self._check_host(rho_np, (self.nz, self.nr))
        self._check_host(phi_np, (self.nz, self.nr), writeable=True)
        r = B.sn_poisson_solve_mg_host(self.h, rho_np.ctypes.data, phi_np.ctypes.data, tol, max_cycles,
                                       torch.cuda.current_stream().cuda_stream)
        self._raise_if_failed([r], "sn_poisson_solve_mg_host")
        return r

    def _check_host(self, a, shape, writeable=False):
        import numpy as np
        if not isinstance(a, np.ndarray) or a.dtype != np.float64 or not a.flags.c_contiguous or tuple(a.shape) != shape:
            raise ValueError(f"expected a C-contiguous float64 numpy array of shape {shape}")
        if writeable and not a.flags.writeable:
            raise ValueError("output array is read-only")

    def solve_host(self, rho_np, phi_np, tol, max_sweeps):
        """Host numpy arrays (C-contiguous float64, (nz, nr) or (nbatch, nz, nr)); phi_np is updated in place.
        H2D/D2H inside the call (sn_poisson_solve_host / sn_poisson_solve_batch_host)."""
        import torch
        stream = torch.cuda.current_stream().cuda_stream
        if rho_np.ndim == 3:
            shape = (rho_np.shape[0], self.nz, self.nr)
            self._check_host(rho_np, shape)
            self._check_host(phi_np, shape, writeable=True)
            res = B.sn_poisson_solve_batch_host(self.h, shape[0], rho_np.ctypes.data, phi_np.ctypes.data, tol,
                                                max_sweeps, stream)
            self._raise_if_failed(res, "sn_poisson_solve_batch_host")
            return res
        self._check_host(rho_np, (self.nz, self.nr))
        self._check_host(phi_np, (self.nz, self.nr), writeable=True)
        r = B.sn_poisson_solve_host(self.h, rho_np.ctypes.data, phi_np.ctypes.data, tol, max_sweeps, stream)
        self._raise_if_failed([r], "sn_poisson_solve_host")
        return r

    def solve_sequence_host(self, rho_seq_np, phi_np, tol, max_sweeps, phi_seq_np=None):
        """Warm-started sequence ([CFG 3]): rho_seq_np (nsteps, nz, nr); phi_np (nz, nr) initial guess in / last
        potential out; phi_seq_np (nsteps, nz, nr) optional, every step's potential.  Returns the list of results."""
        import torch
        n = rho_seq_np.shape[0]
        self._check_host(rho_seq_np, (n, self.nz, self.nr))
        self._check_host(phi_np, (self.nz, self.nr), writeable=True)
        if phi_seq_np is not None:
            self._check_host(phi_seq_np, (n, self.nz, self.nr), writeable=True)
        res = B.sn_poisson_solve_sequence_host(self.h, n, rho_seq_np.ctypes.data, phi_np.ctypes.data,
                                               0 if phi_seq_np is None else phi_seq_np.ctypes.data, tol, max_sweeps,
                                               torch.cuda.current_stream().cuda_stream)
        self._raise_if_failed(res, "sn_poisson_solve_sequence_host")      # steps after a failed one stay at -1
        return res

    def solve_gravity(self, rho, phi, tol, max_sweeps):
        """Solve in place on ``phi`` and return (results, g_r, g_z) from the fused epilogue (sn_poisson_solve_gravity)."""
        import torch
        self._check(rho)
        self._check(phi)
        if rho.shape != phi.shape or tuple(rho.shape[-2:]) != (self.nz, self.nr):
            raise ValueError("shape mismatch")
        nb = rho.shape[0] if rho.dim() == 3 else 1
        gr, gz = torch.empty_like(phi), torch.empty_like(phi)
        res = B.sn_poisson_solve_gravity(self.h, nb, rho.data_ptr(), phi.data_ptr(), gr.data_ptr(), gz.data_ptr(), tol,
                                         max_sweeps, torch.cuda.current_stream().cuda_stream)
        self._raise_if_failed(res, "sn_poisson_solve_gravity")
        return (res if rho.dim() == 3 else res[0]), gr, gz

    def gravity(self, phi, gr=None, gz=None):
        """(g_r, g_z) = -grad phi with the ghost values of the last solve; enqueued on the current stream."""
        import torch
        self._check(phi)
        gr = torch.empty_like(phi) if gr is None else gr
        gz = torch.empty_like(phi) if gz is None else gz
        self._check(gr)
        self._check(gz)
        nb = phi.shape[0] if phi.dim() == 3 else 1
        if tuple(phi.shape[-2:]) != (self.nz, self.nr) or gr.shape != phi.shape or gz.shape != phi.shape:
            raise ValueError("shape mismatch")
        B.sn_poisson_gravity(self.h, nb, phi.data_ptr(), gr.data_ptr(), gz.data_ptr(),
                             torch.cuda.current_stream().cuda_stream)
        return gr, gz

    def set_stop_rule(self, rule):
        return B.sn_poisson_set_stop_rule(self.h, rule)

    def set_option(self, key, value):
        return B.sn_poisson_set_option(self.h, key, value)

    def stat(self, key):
        return B.sn_poisson_get_stat(self.h, key)

    def moments(self):
        return B.sn_poisson_get_moments(self.h, self.lmax)

    def boundary(self):
        return B.sn_poisson_get_boundary(self.h, self.nr, self.nz, self.symmetry)

    def set_boundary(self, bE, bN, bS=None):
        return B.sn_poisson_set_boundary(self.h, bE, bN, bS)

    def history(self, n):
        return B.sn_poisson_get_history(self.h, n)

    @property
    def omega(self):
        return B.sn_poisson_get_omega(self.h)


class LevelSet:
    """Owns one sn_levelset handle (NEXT-2: level-set re-initialisation).  ``S``: float64 CUDA tensor (ny, nx) of the
    scalar field on the cell corners."""

    def __init__(self, nx, ny, dr, dz, delta=None):
        self.nx, self.ny = nx, ny
        self.h = B.sn_levelset_create(nx, ny, dr, dz, dr if delta is None else delta)

    def close(self):
        if getattr(self, "h", None) and getattr(B, "sn_levelset_destroy", None):
            B.sn_levelset_destroy(self.h)
            self.h = None

    __del__ = close

    def reinit(self, S, want_dist=False):
        """Returns (S_new, dist or None, crossings); enqueued on the current stream, synchronised by the library."""
        import torch
        if not (S.is_cuda and S.dtype == torch.float64 and S.is_contiguous() and tuple(S.shape) == (self.ny, self.nx)):
            raise ValueError("expected a contiguous float64 CUDA tensor of shape (ny, nx)")
        out = torch.empty_like(S)
        dist = torch.empty_like(S) if want_dist else None
        n = B.sn_levelset_reinit(self.h, S.data_ptr(), out.data_ptr(), dist.data_ptr() if want_dist else 0,
                                 torch.cuda.current_stream().cuda_stream)
        return out, dist, n

    def reinit_host(self, S_np, want_dist=False):
        import numpy as np
        import torch
        if S_np.dtype != np.float64 or not S_np.flags.c_contiguous or tuple(S_np.shape) != (self.ny, self.nx):
            raise ValueError("expected a C-contiguous float64 numpy array of shape (ny, nx)")
        out = np.empty_like(S_np)
        dist = np.empty_like(S_np) if want_dist else None
        n = B.sn_levelset_reinit_host(self.h, S_np.ctypes.data, out.ctypes.data, dist.ctypes.data if want_dist else 0,
                                      torch.cuda.current_stream().cuda_stream)
        return out, dist, n

    def stat(self, key):
        return B.sn_levelset_get_stat(self.h, key)


class Weno:
    """Owns one sn_weno handle (NEXT-3: WENO-5 / global Lax-Friedrichs flux reconstruction).  ``U``: float64 CUDA
    tensor (4, nz, nr) of (rho, rho v_r, rho v_z, tau); bc = (r-low, r-high, z-low, z-high), 0 outflow / 1 reflecting /
    2 periodic."""

    def __init__(self, nr, nz, dr, dz, gamma, bc):
        self.nr, self.nz = nr, nz
        self.h = B.sn_weno_create(nr, nz, dr, dz, gamma, bc)

    def close(self):
        if getattr(self, "h", None) and getattr(B, "sn_weno_destroy", None):
            B.sn_weno_destroy(self.h)
            self.h = None

    __del__ = close

    def _check(self, U):
        import torch
        if not (U.is_cuda and U.dtype == torch.float64 and U.is_contiguous() and tuple(U.shape) == (4, self.nz, self.nr)):
            raise ValueError("expected a contiguous float64 CUDA tensor of shape (4, nz, nr)")

    @staticmethod
    def _stream():
        import torch
        return torch.cuda.current_stream().cuda_stream

    def max_speeds(self, U):
        self._check(U)
        return B.sn_weno_max_speeds(self.h, U.data_ptr(), self._stream())

    def rhs(self, U, alpha=None, out=None):
        """L(U); alpha = (alpha_r, alpha_z) or None for the device-computed global maxima.  Asynchronous."""
        import torch
        self._check(U)
        out = torch.empty_like(U) if out is None else out
        self._check(out)
        ar, az = (-1.0, -1.0) if alpha is None else alpha
        B.sn_weno_rhs(self.h, U.data_ptr(), out.data_ptr(), ar, az, self._stream())
        return out

    def step(self, U, cfl, want_dt=True):
        """One SSP-RK3 step in place; returns dt (synchronises) or None."""
        self._check(U)
        return B.sn_weno_step(self.h, U.data_ptr(), cfl, self._stream(), want_dt)

    def evolve(self, U, cfl, t_end, max_steps=1000000):
        self._check(U)
        return B.sn_weno_evolve(self.h, U.data_ptr(), cfl, t_end, max_steps, self._stream())

    def rhs_host(self, U_np):
        import numpy as np
        if U_np.dtype != np.float64 or not U_np.flags.c_contiguous or tuple(U_np.shape) != (4, self.nz, self.nr):
            raise ValueError("expected a C-contiguous float64 numpy array of shape (4, nz, nr)")
        out = np.empty_like(U_np)
        B.sn_weno_rhs_host(self.h, U_np.ctypes.data, out.ctypes.data, self._stream())
        return out

    def stat(self, key):
        return B.sn_weno_get_stat(self.h, key)
