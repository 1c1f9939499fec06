"""GPU parity of the WENO-5 / global Lax-Friedrichs flux reconstruction (include/sn_weno.h)
against oracle/weno_oracle.cpp, through the C ABI, on the same seeded inputs.

Bar: BIT-EXACT.  Both sides evaluate the pinned expression trees of readings W2-W8 with correctly rounded IEEE fp64
operations and no FMA contraction (-fmad=false / -ffp-contract=off); the global maxima are exact in any order."""
import os

import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu
GAMMA = 1.4


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


def table3():
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_table3_shocktubes.txt")
    return [[float(t) for t in line.split()] for line in open(path) if line.strip() and not line.startswith("#")]


# grids that span several 32 x 8 tiles with ragged tails in both axes, one tile, a single row, a single column
GRIDS = [(70, 37), (32, 8), (33, 9), (100, 1), (1, 50), (5, 3), (257, 66)]
BCS = [[0, 0, 0, 0], [1, 0, 1, 0], [2, 2, 2, 2], [1, 1, 0, 1], [2, 2, 0, 0]]


@pytest.mark.parametrize("nr,nz", GRIDS)
@pytest.mark.parametrize("bc", BCS)
def test_rhs_and_speeds_bit_exact(P, torch_cuda, oracle, nr, nz, bc):
    torch = torch_cuda
    if (bc[0] != 0 or bc[1] != 0) and nr < 3 or (bc[2] != 0 or bc[3] != 0) and nz < 3:
        with pytest.raises(P.SnPoissonError):
            P.Weno(nr, nz, 0.1, 0.1, GAMMA, bc)
        return
    U, dr, dz = W.hydro_blobs(nr, nz, seed=nr + 3 * nz, jump=0.8)
    w = P.Weno(nr, nz, dr, dz, GAMMA, bc)
    Ud = torch.from_numpy(U).cuda()
    assert w.max_speeds(Ud) == oracle.weno_max_speeds(U, dr, dz, GAMMA, bc)
    want = oracle.weno_rhs(U, dr, dz, GAMMA, bc)
    got = w.rhs(Ud).cpu().numpy()                        # alpha computed on the device
    assert np.array_equal(got, want)
    al = (3.7, 2.9)                                      # caller-supplied splitting speeds
    assert np.array_equal(w.rhs(Ud, alpha=al).cpu().numpy(), oracle.weno_rhs(U, dr, dz, GAMMA, bc, alpha=al))
    assert np.array_equal(w.rhs_host(U), want)           # HOST-buffer entry point
    w.close()


def test_rhs_full_size_paper_grid(P, torch_cuda, oracle):
    """500 x 500, reflecting axis / equator, outflow outside: every element against the oracle."""
    torch = torch_cuda
    U, dr, dz = W.hydro_blobs(500, 500, seed=11, jump=0.5)
    bc = [1, 0, 1, 0]
    w = P.Weno(500, 500, dr, dz, GAMMA, bc)
    got = w.rhs(torch.from_numpy(U).cuda()).cpu().numpy()
    assert np.array_equal(got, oracle.weno_rhs(U, dr, dz, GAMMA, bc))
    assert w.stat("rhs_ms") > 0 and w.stat("launches") == 2
    w.close()


@pytest.mark.parametrize("bc", [[0, 0, 0, 0], [1, 0, 1, 0], [2, 2, 2, 2]])
def test_rk3_steps_bit_exact(P, torch_cuda, oracle, bc):
    torch = torch_cuda
    nr, nz = 70, 37
    U, dr, dz = W.hydro_blobs(nr, nz, seed=5, jump=0.6)
    w = P.Weno(nr, nz, dr, dz, GAMMA, bc)
    Ud = torch.from_numpy(U).cuda()
    ref = U
    for _ in range(4):
        ref, dt_ref = oracle.weno_step(ref, dr, dz, GAMMA, bc, 0.5)
        dt = w.step(Ud, 0.5)
        assert dt == dt_ref
        assert np.array_equal(Ud.cpu().numpy(), ref)
    assert w.stat("launches") == 7                        # 3 x (maxima + reconstruction) + the time-step kernel
    w.close()


@pytest.mark.parametrize("test", [1, 2, 3, 4])
def test_paper_shock_tubes_match_the_oracle(P, torch_cuda, oracle, test):
    """PAPER.md:391-398 (Table 3) on 400 cells (one row, dz huge: the paper's 1-D Courant number 0.5): the whole
    evolution bit for bit, same number of steps.  The oracle's own distance to the exact Riemann solution is pinned in
    tests/test_weno_pins.py."""
    torch = torch_cuda
    row = table3()[test - 1]
    t0 = 0.15 if test == 2 else row[1]                   # reading W9
    n = 400
    U, dx = W.shock_tube(*row[3:9], x0=row[2], n=n)
    ref, steps_ref = oracle.weno_evolve(U, dx, 1.0e30, GAMMA, [0, 0, 0, 0], 0.5, t0)
    w = P.Weno(n, 1, dx, 1.0e30, GAMMA, [0, 0, 0, 0])
    Ud = torch.from_numpy(U).cuda()
    steps = w.evolve(Ud, 0.5, t0)
    assert steps == steps_ref
    assert np.array_equal(Ud.cpu().numpy(), ref)
    w.close()


def test_shock_tube_along_z_is_the_transpose(P, torch_cuda, oracle):
    """The z sweep (shared-memory exchange between thread rows) against the r sweep (warp shuffles) on the same tube."""
    torch = torch_cuda
    row = table3()[0]
    n = 200
    Ur, dx = W.shock_tube(*row[3:9], x0=row[2], n=n, rows=3, axis=0)
    Uz, _ = W.shock_tube(*row[3:9], x0=row[2], n=n, rows=3, axis=1)
    wr = P.Weno(n, 3, dx, dx, GAMMA, [0, 0, 0, 0])
    wz = P.Weno(3, n, dx, dx, GAMMA, [0, 0, 0, 0])
    a, b = torch.from_numpy(Ur).cuda(), torch.from_numpy(Uz).cuda()
    for _ in range(25):
        assert wr.step(a, 0.5) == wz.step(b, 0.5)
    a, b = a.cpu().numpy(), b.cpu().numpy()
    assert np.array_equal(a[0], b[0].T) and np.array_equal(a[1], b[2].T) and np.array_equal(a[3], b[3].T)
    ref = Ur
    for _ in range(25):
        ref, _ = oracle.weno_step(ref, dx, dx, GAMMA, [0, 0, 0, 0], 0.5)
    assert np.array_equal(a, ref)
    wr.close()
    wz.close()


def test_weno_argument_errors(P, torch_cuda):
    torch = torch_cuda
    for bad in [(0, 4, .1, .1, 1.4, [0, 0, 0, 0]), (4, 4, -.1, .1, 1.4, [0, 0, 0, 0]), (4, 4, .1, .1, 1.0, [0, 0, 0, 0]),
                (4, 4, .1, .1, 1.4, [3, 0, 0, 0]), (4, 4, .1, .1, 1.4, [2, 0, 0, 0])]:
        with pytest.raises(P.SnPoissonError):
            P.Weno(*bad)
    w = P.Weno(8, 8, .1, .1, 1.4, [0, 0, 0, 0])
    U = torch.ones((4, 8, 8), dtype=torch.float64, device="cuda")
    with pytest.raises(P.SnPoissonError):
        P.sn_weno_rhs(w.h, U.data_ptr(), U.data_ptr())   # aliasing
    with pytest.raises(P.SnPoissonError):
        P.sn_weno_step(w.h, U.data_ptr(), -1.0)
    with pytest.raises(ValueError):
        w.rhs(U[:, :4])
    w.close()


@pytest.mark.parametrize("test", [1, 2, 3, 4])
def test_paper_tubes_at_the_papers_resolution(P, torch_cuda, oracle, test):
    """PAPER.md:402 "2000 computing cells": every test of Table 3 evolved to its t0 on both sides, bit for bit, with the
    same number of steps (tests 3 and 4 are the strong-shock ones; the oracle needs 20-60 s per tube; its distance to the
    exact Riemann solution is pinned in tests/test_weno_pins.py)."""
    torch = torch_cuda
    row = table3()[test - 1]
    t0 = 0.15 if test == 2 else row[1]                   # reading W9
    n = 2000
    U, dx = W.shock_tube(*row[3:9], x0=row[2], n=n)
    ref, steps_ref = oracle.weno_evolve(U, dx, 1.0e30, GAMMA, [0, 0, 0, 0], 0.5, t0)
    w = P.Weno(n, 1, dx, 1.0e30, GAMMA, [0, 0, 0, 0])
    Ud = torch.from_numpy(U).cuda()
    assert w.evolve(Ud, 0.5, t0) == steps_ref
    assert np.array_equal(Ud.cpu().numpy(), ref)
    assert w.stat("launches") == 7 * steps_ref           # no separate maxima pass per step: 3 x (maxima + rhs) + dt
    w.close()
