"""Writes tests/golden/oracle_regression.json.  Calls ONLY oracle/ (and the input generators in workloads/).

These are not paper values (the paper prints none for the Poisson solver); they freeze the
oracle's own iteration history so that an unintended change to its arithmetic is caught.  A deliberate change
must cite the DESIGN.md reading that justifies it in its commit message, then re-run this script:

    python tests/golden/make_oracle_golden.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle as O          # noqa: E402
import workloads as W       # noqa: E402

SAMPLES = [(0, 0), (0, 5), (3, 0), (17, 9), (31, 40), (63, 63), (40, 2)]


def history_case(w, sweeps_list):
    M = O.moments(w.rho, w.dr, w.dz, w.symmetry, w.lmax)
    bE, bN, bS = O.boundary(w.nr, w.nz, w.dr, w.dz, w.symmetry, w.lmax, M)
    omega = w.omega if w.omega is not None else O.default_omega(w.nr, w.nz, w.dr, w.dz, w.symmetry)
    out = {"omega": omega.hex() if isinstance(omega, float) else float(omega).hex(),
           "M": [float(m).hex() for m in M], "iterates": {}}
    for k in sweeps_list:
        phi, Rabs, P = O.sweeps(w.rho, np.zeros_like(w.rho), w.dr, w.dz, w.symmetry, omega, bE, bN, bS, k)
        out["iterates"][str(k)] = {
            "samples": [float(phi[j % w.nz, i % w.nr]).hex() for (j, i) in SAMPLES],
            "Rabs": float(Rabs[-1]).hex(), "P": float(P[-1]).hex()}
    return out


def main():
    g = {"_doc": "oracle-only regression values (hex floats); see make_oracle_golden.py"}
    g["cfg0_64"] = history_case(W.cfg0(64), [1, 2, 10, 100, 1000])
    g["cfg1_64"] = history_case(W.cfg1(64), [1, 10, 100])
    g["full_plane_24x40"] = history_case(W.random_smooth(24, 40, 0, seed=21, lmax=5), [1, 3, 50])
    conv = {}
    for name, w in (("cfg1_256", W.cfg1()), ("cfg2_128", W.cfg2(128)), ("cfg3_64x128", W.cfg3(64).first)):
        r = O.solve_workload(w)
        conv[name] = {"sweeps": r["sweeps"], "residual": float(r["residual"]).hex(), "status": r["status"],
                      "phi_min": float(r["phi"].min()).hex()}
    g["converged"] = conv
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_regression.json"), "w") as f:
        json.dump(g, f, indent=1)


if __name__ == "__main__":
    main()
