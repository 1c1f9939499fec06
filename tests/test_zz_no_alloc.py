"""sn_poisson_moments_static: the multipole moments for callers that are not allowed to allocate device memory.

Some hosts of this library cannot call cudaMalloc while they run: a simulation that claimed the whole GPU for its own
grids at start-up, a framework whose device memory all lives in one pool, a time-step loop that cannot afford the
device-wide stall an allocation may cause.  Every handle-based call allocates workspace; this one entry point does not.
Its scratch is a fixed array inside the library, shared by all calls on a GPU and never cleared between them, so what
has to be shown is (1) it gives the moments the ordinary handle path gives, and (2) a second call is not polluted by
what the first one left in the array.  Both calls below go on one stream with no synchronisation in between.

The file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide other tests.
It sets up its own fixtures so it passes alone in a fresh process as well as after the rest of the suite.
"""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

FOUR_PI = 12.566370614359172     # the fp64 constant the kernels multiply rho by
TOL = 1e-13                      # bar of the moment parity tests (tests/test_gpu_parity.py)


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


def handle_moments(P, torch, w):
    """The existing path: a handle (which allocates), one sweep, then the moments it used for the boundary."""
    s = P.PoissonSolver(w.nr, w.nz, w.dr, w.dz, w.symmetry, w.lmax)
    rho = torch.from_numpy(w.rho).cuda()
    phi = torch.zeros_like(rho)
    s.solve(rho, phi, 0.0, 1)
    torch.cuda.synchronize()
    return s.moments()


def static_moments(P, torch, members):
    """Enqueue one sn_poisson_moments_static call for a batch of same-shaped workloads; returns device outputs
    (not synchronised) together with the input tensor, which must stay alive until the stream has run."""
    w = members[0]
    rho = torch.from_numpy(np.stack([m.rho for m in members])).cuda()
    M = torch.full((len(members), w.lmax + 1), float("nan"), dtype=torch.float64, device="cuda")
    mx = torch.full((len(members),), float("nan"), dtype=torch.float64, device="cuda")
    rc = P.sn_poisson_moments_static(rho.data_ptr(), len(members), w.nr, w.nz, w.dr, w.dz, w.symmetry, w.lmax,
                                     M.data_ptr(), mx.data_ptr(), torch.cuda.current_stream().cuda_stream)
    assert rc == 0
    return rho, M, mx


def assert_matches_handle(P, torch, members, M, mx):
    M, mx = M.cpu().numpy(), mx.cpu().numpy()
    for b, w in enumerate(members):
        want = handle_moments(P, torch, w)
        assert np.all(np.isfinite(M[b]))
        assert np.all(np.abs(M[b] - want) <= TOL * np.maximum(np.abs(want), np.abs(want[0]))), (b, M[b], want)
        if w.symmetry == 1:
            assert np.all(M[b][1::2] == 0.0)
        assert mx[b] == np.max(np.abs(FOUR_PI * w.rho))


def test_two_calls_in_a_row_match_the_handle_path(P, torch_cuda):
    torch = torch_cuda
    # first call: three members, many blocks, 17 sums per block, large densities -> fills a lot of the scratch
    first = [W.random_smooth(200, 168, 0, seed=900 + b, lmax=16) for b in range(3)]
    for m in first:
        m.rho *= 50.0
    # second call: one small half-plane grid, 9 sums per block, small densities.  Anything left over from the first
    # call (partial sums of blocks that no longer exist, a larger max|4 pi rho|) would show up here.
    second = [W.random_smooth(36, 50, 1, seed=950, lmax=5)]
    keep1 = static_moments(P, torch, first)
    keep2 = static_moments(P, torch, second)
    keep3 = static_moments(P, torch, first)            # and back again: same bits as the first time
    torch.cuda.synchronize()
    assert_matches_handle(P, torch, first, keep1[1], keep1[2])
    assert_matches_handle(P, torch, second, keep2[1], keep2[2])
    assert torch.equal(keep1[1], keep3[1]) and torch.equal(keep1[2], keep3[2])


def test_sizes_beyond_the_static_scratch_are_refused(P, torch_cuda):
    torch = torch_cuda
    rho = torch.zeros((13, 1024, 1024), dtype=torch.float64, device="cuda")
    M = torch.zeros((65, 9), dtype=torch.float64, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    # 13 members x (4 x SM count) blocks x 9 sums is more than the array holds on any GPU with >= 141 SMs
    with pytest.raises(P.SnPoissonError, match="scratch"):
        P.sn_poisson_moments_static(rho.data_ptr(), 13, 1024, 1024, 1e-3, 1e-3, 1, 8, M.data_ptr(), 0, st)
    with pytest.raises(P.SnPoissonError, match="members"):
        P.sn_poisson_moments_static(rho.data_ptr(), 65, 16, 16, 1e-3, 1e-3, 1, 8, M.data_ptr(), 0, st)
    with pytest.raises(P.SnPoissonError):
        P.sn_poisson_moments_static(rho.data_ptr(), 1, 16, 16, 1e-3, 1e-3, 1, 65, M.data_ptr(), 0, st)
    # the largest single grid of BASELINE.json at the largest lmax still fits, and the refusals left no error state behind
    assert P.sn_poisson_moments_static(rho.data_ptr(), 1, 1024, 2048, 1e-3, 1e-3, 1, 64, M.data_ptr(), 0, st) == 0
    torch.cuda.synchronize()
    assert torch.all(M[0, :9] == 0.0)
