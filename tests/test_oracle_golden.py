"""Oracle regression against tests/golden/oracle_regression.json (written by make_oracle_golden.py, oracle-only)."""
import json
import os

import numpy as np

import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))
SAMPLES = [(0, 0), (0, 5), (3, 0), (17, 9), (31, 40), (63, 63), (40, 2)]


def _check_history(oracle, w, g):
    M = oracle.moments(w.rho, w.dr, w.dz, w.symmetry, w.lmax)
    assert [float(m).hex() for m in M] == g["M"]
    bE, bN, bS = oracle.boundary(w.nr, w.nz, w.dr, w.dz, w.symmetry, w.lmax, M)
    omega = float.fromhex(g["omega"])
    if w.omega is None:
        assert oracle.default_omega(w.nr, w.nz, w.dr, w.dz, w.symmetry) == omega
    for k, it in g["iterates"].items():
        phi, Rabs, P = oracle.sweeps(w.rho, np.zeros_like(w.rho), w.dr, w.dz, w.symmetry, omega, bE, bN, bS, int(k))
        assert [float(phi[j % w.nz, i % w.nr]).hex() for (j, i) in SAMPLES] == it["samples"]
        assert float(Rabs[-1]).hex() == it["Rabs"] and float(P[-1]).hex() == it["P"]


def test_oracle_iteration_history_is_frozen(oracle):
    g = json.load(open(os.path.join(HERE, "golden", "oracle_regression.json")))
    _check_history(oracle, W.cfg0(64), g["cfg0_64"])
    _check_history(oracle, W.cfg1(64), g["cfg1_64"])
    _check_history(oracle, W.random_smooth(24, 40, 0, seed=21, lmax=5), g["full_plane_24x40"])


def test_oracle_converged_counts_are_frozen(oracle):
    g = json.load(open(os.path.join(HERE, "golden", "oracle_regression.json")))["converged"]
    for name, w in (("cfg1_256", W.cfg1()), ("cfg2_128", W.cfg2(128)), ("cfg3_64x128", W.cfg3(64).first)):
        r = oracle.solve_workload(w)
        assert r["sweeps"] == g[name]["sweeps"] and r["status"] == g[name]["status"]
        assert float(r["residual"]).hex() == g[name]["residual"]
        assert float(r["phi"].min()).hex() == g[name]["phi_min"]
