"""Pins of the level-set re-initialisation oracle (oracle/levelset_oracle.cpp) against things the paper and geometry fix
-- not against itself.  PAPER.md:131-141 (section 2.2, eqs. 6-7).  CPU only."""
import math

import numpy as np
import pytest

import workloads as W


def circle(n, R, cx=0.0, cy=0.0, scale=None):
    dr = 1.0 / (n - 1)
    x = np.arange(n) * dr
    X, Y = np.meshgrid(x, x)
    S = R - np.hypot(X - cx, Y - cy)                 # exact signed distance, > 0 inside (ash)
    if scale is not None:
        S = S * scale(X, Y)
    return np.ascontiguousarray(S), dr, X, Y


def test_H_end_points_and_plateau(oracle):
    """eq. (7): H(0) = 1, H(inf) = 0, H = 1/2 + ... at d0 = 3 Delta; S on the three closest grids unchanged."""
    delta = 0.01
    assert oracle.levelset_H(0.0, delta) == 1.0
    assert oracle.levelset_H(1e9, delta) == 0.0
    # typed-out formula at a few points
    for d in (0.3 * delta, 2.0 * delta, 3.0 * delta, 3.5 * delta, 6.0 * delta):
        want = (1 - math.tanh((d - 3 * delta) / (delta / 3))) / (1 - math.tanh(-3 * delta / (delta / 3)))
        assert oracle.levelset_H(d, delta) == pytest.approx(want, rel=1e-14)
    assert oracle.levelset_H(3.0 * delta, delta) == pytest.approx(0.5, rel=1e-7)
    assert 1.0 - oracle.levelset_H(2.0 * delta, delta) < 3e-3        # within 2 Delta: essentially the old value
    assert oracle.levelset_H(4.5 * delta, delta) < 2e-4              # beyond 4.5 Delta: essentially the distance


def test_crossings_match_brute_force_python(oracle):
    """Every grid edge with one end < 0 and the other >= 0, linear interpolation -- enumerated by a
    pure-Python double loop on a small distorted front, compared as sets."""
    S, dr = W.levelset_front(24, seed=3)
    ny, nx = S.shape
    want = []
    for j in range(ny):
        for i in range(nx):
            a = S[j, i]
            if i + 1 < nx and (a < 0) != (S[j, i + 1] < 0):
                want.append((i * dr + dr * a / (a - S[j, i + 1]), j * dr))
            if j + 1 < ny and (a < 0) != (S[j + 1, i] < 0):
                want.append((i * dr, j * dr + dr * a / (a - S[j + 1, i])))
    cx, cy = oracle.levelset_crossings(S, dr, dr)
    assert len(cx) == len(want) > 20
    got = sorted(zip(cx, cy))
    for (gx, gy), (wx, wy) in zip(got, sorted(want)):
        assert gx == pytest.approx(wx, abs=1e-15) and gy == pytest.approx(wy, abs=1e-15)
    # a node with S == 0 is a crossing of its own edges (t = 0)
    Z = np.array([[-1.0, -1.0, -1.0], [-1.0, 0.0, -1.0], [-1.0, -1.0, -1.0]])
    zx, zy = oracle.levelset_crossings(Z, 1.0, 1.0)
    assert sorted(zip(zx, zy)) == [(1.0, 1.0)] * 4                  # its four edges, all at the node itself


def test_circle_distance_and_blend(oracle):
    """A circular front: the exact signed distance is R - s.  The crossings lie within O(Delta^2) of the circle (chord
    interpolation of a smooth S) and are at most ~Delta apart, so the minimum distance to them equals the exact
    distance to within Delta^2 / (8 R) + (Delta / 2)^2 / (2 d) for nodes at distance d >> Delta."""
    n, R = 201, 0.5
    S, dr, X, Y = circle(n, R)
    r = oracle.levelset_reinit(S, dr, dr)
    exact = R - np.hypot(X, Y)
    assert r["crossings"] > 150
    assert np.all(np.sign(r["dist"]) == np.sign(S))                    # ash stays ash, fuel stays fuel
    far = np.abs(exact) > 6 * dr
    err = np.abs(np.abs(r["dist"]) - np.abs(exact))
    assert np.max(err[far]) < dr * dr / (8 * R) + (0.75 * dr) ** 2 / (2 * 6 * dr) + 1e-12
    # far from the front the new value IS the distance (H -> 0); close to it the old value is kept (H -> 1)
    assert np.max(np.abs(r["S"][far] - r["dist"][far])) < 1e-7 * dr
    near = np.abs(exact) < 2 * dr
    assert np.max(np.abs(r["S"][near] - S[near])) < 4e-3 * dr
    # S_old was already a distance function: re-initialisation changes it by no more than the interpolation error
    assert np.max(np.abs(r["S"] - S)) < 0.6 * dr


def test_distorted_field_is_repaired_and_front_is_kept(oracle):
    """re-initialisation restores |grad S| = 1 without moving the front.  S = (R - s)(1 + 0.6 sin..):
    same zero contour, wrong slope.  After the call: far nodes carry the true distance; the crossings of the NEW field
    coincide with the old ones (the three closest grids are unchanged)."""
    n, R = 161, 0.45
    S, dr, X, Y = circle(n, R, scale=lambda x, y: 1.0 + 0.6 * np.sin(7 * x) * np.cos(5 * y))
    r = oracle.levelset_reinit(S, dr, dr)
    exact = R - np.hypot(X, Y)
    far = np.abs(exact) > 6 * dr
    assert np.max(np.abs(S[far] - exact[far])) > 20 * dr * dr            # the input really was off
    assert np.max(np.abs(r["S"][far] - exact[far])) < 6 * dr * dr             # O(Delta^2): chord + interpolation of a curved S
    ox, oy = oracle.levelset_crossings(S, dr, dr)
    nx_, ny_ = oracle.levelset_crossings(r["S"], dr, dr)
    assert len(ox) == len(nx_)
    assert np.max(np.abs(np.sort(ox) - np.sort(nx_))) < 1e-2 * dr and np.max(np.abs(np.sort(oy) - np.sort(ny_))) < 1e-2 * dr
    # gradient norm of the repaired field away from the blend zone and the centre kink
    gy, gx = np.gradient(r["S"], dr)
    band = (np.abs(exact) > 6 * dr) & (np.hypot(X, Y) > 10 * dr) & (X > dr) & (Y > dr) & (X < 1 - dr) & (Y < 1 - dr)
    assert np.max(np.abs(np.hypot(gx, gy)[band] - 1.0)) < 0.02


def test_straight_tilted_line(oracle):
    """S linear in (x, y): linear interpolation is exact, every crossing lies ON the line a x + b y = c, so the minimum
    distance to the crossings can never be smaller than the exact point-line distance, and exceeds it by less than the
    gap between neighbouring crossings."""
    n = 81
    dr = 1.0 / (n - 1)
    x = np.arange(n) * dr
    X, Y = np.meshgrid(x, x)
    a, b, c = math.cos(0.4), math.sin(0.4), 0.55
    S = np.ascontiguousarray(c - (a * X + b * Y))                     # exact signed distance to the line
    r = oracle.levelset_reinit(S, dr, dr)
    cx, cy = oracle.levelset_crossings(S, dr, dr)
    assert np.max(np.abs(a * cx + b * cy - c)) < 1e-14
    d, ex = np.abs(r["dist"]), np.abs(S)
    assert np.all(d >= ex - 1e-14)
    inner = (X > 0.15) & (X < 0.85) & (Y > 0.15) & (Y < 0.85) & (ex < 0.1)
    assert np.max((d - ex)[inner]) < dr                                # nearest crossing is within one cell along the line


def test_no_front_leaves_field_unchanged(oracle):
    S = np.full((9, 7), -0.3)
    r = oracle.levelset_reinit(S, 0.1, 0.1)
    assert r["crossings"] == 0 and np.array_equal(r["S"], S) and np.all(np.isinf(r["dist"])) and np.all(r["dist"] < 0)


def test_three_finger_workload_shape():
    """The seeded stand-in for the paper's c3 three-finger flame: three maxima of the front radius in the
    quadrant, ash inside."""
    S, dr = W.levelset_front(200, seed=7)
    assert S.shape == (201, 201) and S[0, 0] > 0 and S[-1, -1] < 0
    ang = np.linspace(0, np.pi / 2, 721)
    rad = []
    for t in ang:                                                  # radius of the sign change along a ray
        s = np.linspace(0.05, 0.6, 1200)
        i = np.clip(np.rint(s * np.sin(t) / dr).astype(int), 0, 200)
        j = np.clip(np.rint(s * np.cos(t) / dr).astype(int), 0, 200)
        rad.append(s[np.argmax(S[j, i] < 0)])
    rad = np.array(rad)
    peaks = [k for k in range(5, 716) if rad[k] == rad[k - 5:k + 6].max() and rad[k] > 0.33]
    groups = 1 + sum(1 for a, b in zip(peaks, peaks[1:]) if b - a > 20)
    assert groups == 3
