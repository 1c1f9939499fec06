"""GPU parity of the multigrid variant (sn_poisson_solve_mg, readings M1-M8) against
oracle/mg_oracle.cpp through the C ABI on the same seeded inputs.

Bar: with injected ghosts BIT-EXACT iterates, ratios and cycle counts (pinned expression trees, exact maxima); with the
library's own moments (different summation order) <= 1e-11 relative and the same cycle count."""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def P(torch_cuda):
    import paper_1507_08549_b200 as pkg
    from paper_1507_08549_b200 import build
    build.build()
    pkg.load()
    return pkg


@pytest.fixture(scope="module")
def oracle():
    import oracle as O
    O.build()
    return O


def ghosts_of(oracle, w):
    M = oracle.moments(w.rho, w.dr, w.dz, w.symmetry, w.lmax)
    return oracle.boundary(w.nr, w.nz, w.dr, w.dz, w.symmetry, w.lmax, M)


def gpu_mg(P, torch, w, tol, max_cycles, ghosts=None, phi0=None, options=None):
    s = P.PoissonSolver.for_workload(w)
    for k, v in (options or {}).items():
        s.set_option(k, v)
    if ghosts is not None:
        s.set_boundary(*ghosts)
    rho = torch.from_numpy(w.rho).cuda()
    phi = torch.zeros_like(rho) if phi0 is None else torch.from_numpy(phi0).cuda()
    r = s.solve_mg(rho, phi, tol, max_cycles)
    hist = s.history(r.sweeps)
    lev = int(s.stat("mg_levels"))
    s.close()
    return r, phi.cpu().numpy(), hist, lev


CASES = [lambda: W.random_smooth(32, 48, 1, 3), lambda: W.random_smooth(40, 24, 0, 4), lambda: W.cfg1(64),
         lambda: W.cfg3(64).first, lambda: W.random_smooth(6, 10, 1, 8),           # cannot be coarsened: plain Gauss-Seidel
         lambda: W.random_smooth(36, 20, 0, 9), lambda: W.random_smooth(8, 64, 1, 10), lambda: W.cfg1(256)]


@pytest.mark.parametrize("make", CASES)
@pytest.mark.parametrize("ncyc", [1, 3])
def test_fixed_cycles_bit_exact_with_injected_ghosts(P, torch_cuda, oracle, make, ncyc):
    w = make()
    g = ghosts_of(oracle, w)
    ref = oracle.mg_solve(w.rho, np.zeros_like(w.rho), w.dr, w.dz, w.symmetry, w.lmax, 0.0, ncyc, ghosts=g)
    r, phi, hist, lev = gpu_mg(P, torch_cuda, w, 0.0, ncyc, ghosts=g)
    assert lev == oracle.mg_levels(w.nr, w.nz)
    assert r.sweeps == ncyc and r.status == 0
    assert np.array_equal(phi, ref["phi"])
    assert np.array_equal(hist, ref["history"]) and r.residual == ref["residual"]


@pytest.mark.parametrize("nu", [(1, 1), (2, 1), (0, 2), (2, 2)])
def test_to_tolerance_bit_exact_and_options(P, torch_cuda, oracle, nu):
    w = W.cfg3(128).first
    g = ghosts_of(oracle, w)
    ref = oracle.mg_solve(w.rho, np.zeros_like(w.rho), w.dr, w.dz, w.symmetry, w.lmax, w.tol, 40, nu1=nu[0], nu2=nu[1],
                          nc=20, ghosts=g)
    r, phi, hist, _ = gpu_mg(P, torch_cuda, w, w.tol, 40, ghosts=g, options={"mg_nu1": nu[0], "mg_nu2": nu[1], "mg_nc": 20})
    assert r.status == 0 == ref["status"] and r.sweeps == ref["cycles"] and r.residual == ref["residual"]
    assert np.array_equal(phi, ref["phi"]) and np.array_equal(hist, ref["history"])
    # max_cycles one short of the crossing: status 1, same iterates
    r2, phi2, _, _ = gpu_mg(P, torch_cuda, w, w.tol, ref["cycles"] - 1, ghosts=g,
                            options={"mg_nu1": nu[0], "mg_nu2": nu[1], "mg_nc": 20})
    assert r2.status == 1 and r2.sweeps == ref["cycles"] - 1 and r2.residual == ref["history"][-2]


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3"])
def test_full_size_configs_own_moments(P, torch_cuda, oracle, name):
    """The BASELINE.json configs at full size with the library's own moments: same cycle count as the oracle, potential
    within the north_star tolerance, and the same potential as the SOR path's converged answer (same fixed point)."""
    w = {"cfg1": W.cfg1, "cfg2": W.cfg2, "cfg3": lambda: W.cfg3().first}[name]()
    ref = oracle.mg_solve_workload(w)
    r, phi, hist, lev = gpu_mg(P, torch_cuda, w, w.tol, 60)
    assert r.status == 0 and r.sweeps == ref["cycles"] <= 10
    assert np.abs(phi - ref["phi"]).max() <= 1e-11 * np.abs(ref["phi"]).max()
    assert abs(r.residual - ref["residual"]) <= 1e-13
    # SOR on the GPU to the same tolerance: both iterates are within ~1e-8 of the common fixed point
    s = P.PoissonSolver.for_workload(w)
    rho = torch_cuda.from_numpy(w.rho).cuda()
    p2 = torch_cuda.zeros_like(rho)
    s.solve(rho, p2, w.tol, w.max_sweeps)
    s.close()
    assert np.abs(phi - p2.cpu().numpy()).max() <= 5e-8 * np.abs(phi).max()


def test_warm_start_host_entry_and_errors(P, torch_cuda, oracle):
    torch = torch_cuda
    w = W.cfg1(128)
    ref = oracle.mg_solve_workload(w)
    s = P.PoissonSolver.for_workload(w)
    phi = np.zeros_like(w.rho)
    r = s.solve_mg_host(w.rho, phi, w.tol, 60)                       # HOST buffers
    assert r.sweeps == ref["cycles"] and np.abs(phi - ref["phi"]).max() <= 1e-11 * np.abs(phi).max()
    r = s.solve_mg_host(w.rho, phi, w.tol, 60)                       # warm start from the converged iterate
    assert r.sweeps == 1 and r.status == 0
    rho = torch.from_numpy(w.rho).cuda()
    p = torch.zeros_like(rho)
    r0 = s.solve_mg(rho, p, w.tol, 0)
    assert r0.sweeps == 0 and r0.status == 1 and float(p.abs().max()) == 0.0
    rbad = P.sn_poisson_solve_mg(s.h, 0, p.data_ptr(), 1e-10, 5)
    assert rbad.status == -1
    p.fill_(float("nan"))
    with pytest.raises(P.SnPoissonError):
        s.solve_mg(rho, p, w.tol, 5)                                 # status -3
    s.close()


def test_batch_members_equal_single_solves_and_the_oracle(P, torch_cuda, oracle):
    """sn_poisson_solve_mg_batch: members with different convergence histories in one call; each member's result is the
    single-solve result bit for bit, and the oracle's within the north_star tolerance with the same cycle count."""
    torch = torch_cuda
    members = [W.cfg4a_member(b, 128) for b in (0, 1, 2, 3, 4)]
    w0 = members[0]
    rho = torch.from_numpy(np.stack([m.rho for m in members])).cuda()
    phi = torch.zeros_like(rho)
    s = P.PoissonSolver.for_workload(w0)
    res = s.solve_mg(rho, phi, w0.tol, 60)
    got = phi.cpu().numpy()
    for b, m in enumerate(members):
        ref = oracle.mg_solve_workload(m)
        assert res[b].status == 0 and res[b].sweeps == ref["cycles"], (b, res[b], ref["cycles"])
        assert np.abs(got[b] - ref["phi"]).max() <= 1e-11 * np.abs(ref["phi"]).max()
        one = torch.zeros_like(rho[b])
        r1 = s.solve_mg(rho[b].contiguous(), one, w0.tol, 60)
        assert r1.sweeps == res[b].sweeps and r1.residual == res[b].residual
        assert np.array_equal(one.cpu().numpy(), got[b])
    # a member that needs no work next to ones that do: warm start of member 2 only
    phi2 = torch.zeros_like(rho)
    phi2[2] = phi[2]
    res2 = s.solve_mg(rho, phi2, w0.tol, 60)
    assert res2[2].sweeps == 1 and [r.sweeps for i, r in enumerate(res2) if i != 2] == [r.sweeps for i, r in enumerate(res) if i != 2]
    assert np.array_equal(phi2.cpu().numpy()[[0, 1, 3, 4]], got[[0, 1, 3, 4]])
    # fixed cycles, max_cycles reached
    phi3 = torch.zeros_like(rho)
    res3 = s.solve_mg(rho, phi3, w0.tol, 3)
    assert all(r.sweeps == 3 and r.status == 1 for r in res3)
    # the HOST-buffer batch entry (sn_poisson_solve_mg_batch_host, what bench.py's e2e of mg_cfg4a times): same bits,
    # from pageable and from pinned arrays
    rho_h = np.stack([m.rho for m in members])
    for pin in (False, True):
        rho_in = torch.from_numpy(rho_h).pin_memory().numpy() if pin else rho_h
        phi_h = torch.zeros(rho_h.shape, dtype=torch.float64).pin_memory().numpy() if pin else np.zeros_like(rho_h)
        res_h = s.solve_mg_host(rho_in, phi_h, w0.tol, 60)
        assert [(r.sweeps, r.status, r.residual) for r in res_h] == [(r.sweeps, r.status, r.residual) for r in res]
        assert np.array_equal(phi_h, got)
    s.close()


def test_batch_full_size_cfg4a(P, torch_cuda, oracle):
    """All 64 members of [CFG 4a] (512 x 512) in one multigrid call against 64 oracle solves."""
    torch = torch_cuda
    members = W.cfg4a(64)
    w0 = members[0]
    rho = torch.from_numpy(np.stack([m.rho for m in members])).cuda()
    phi = torch.zeros_like(rho)
    s = P.PoissonSolver.for_workload(w0)
    res = s.solve_mg(rho, phi, w0.tol, 60)
    got = phi.cpu().numpy()
    for b, m in enumerate(members):
        ref = oracle.mg_solve_workload(m)
        assert res[b].status == 0 and res[b].sweeps == ref["cycles"], (b, res[b], ref["cycles"])
        assert np.abs(got[b] - ref["phi"]).max() <= 1e-11 * np.abs(ref["phi"]).max()
    s.close()


def test_largest_size_sweep_point_two_cycles_bit_exact(P, torch_cuda, oracle):
    """4096 x 4096 (the largest grid of BASELINE.json's size sweep; 11 levels, 64-bit-free index path, 256 MiB working
    set): two V-cycles with injected ghosts, every element against the oracle."""
    w = W.cfg4b(4096, 2)
    g = ghosts_of(oracle, w)
    ref = oracle.mg_solve(w.rho, np.zeros_like(w.rho), w.dr, w.dz, w.symmetry, w.lmax, 0.0, 2, ghosts=g)
    r, phi, hist, lev = gpu_mg(P, torch_cuda, w, 0.0, 2, ghosts=g)
    assert lev == oracle.mg_levels(4096, 4096) == 11 and r.sweeps == 2
    assert np.array_equal(phi, ref["phi"]) and np.array_equal(hist, ref["history"])
