"""In-kernel SM-clock profile and plan scan of the resident sweep kernel (the library's own "prof" option).

    python -m paper_1507_08549_b200.inkernel_profile CASE [CASE ...]        # one line per case
    python -m paper_1507_08549_b200.inkernel_profile --scan NAME [NAME ...]  # every (shape, mode, m) for a workload

CASE = NAME[:opt=val,...]; NAME in cfg0, cfg1, cfg2, cfg3, sweep<N>, rs<NR>x<NZ> (seeded smooth full-plane grid);
options are sn_poisson_set_option keys (path, shape, tblock, halo, ds, ring, ll, group) plus nsw=<fixed sweeps> (default
600) and prof=0 (timing only).  With prof=1 thread 0 of every CTA accumulates clock64() differences around the phases
of the sweep loop; the columns are SM clocks PER HALF-SWEEP, mean over the CTAs: compute = ring duty + patch update +
publish, xchg = wait for the neighbours' packets / flags, barrier = CTA barrier after it, end = checkpoint + report at
the end of an interval, refill = ring duty alone (halo mode) or margin refill (block mode), wait = wait for the service
warp's decision.  Measurement helper of the library: marshalling and printing only, nothing of the method runs here.
"""
from __future__ import annotations

import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

NAMES = ["total", "compute", "xchg", "barrier", "end", "refill", "wait"]


def workload(name):
    import workloads as W
    if name in ("cfg0", "cfg1", "cfg2"):
        return getattr(W, name)()
    if name == "cfg3":
        return W.cfg3().first
    if name.startswith("sweep"):
        return W.cfg4b(int(name[5:]), 2000)
    if name.startswith("rs"):
        nr, nz = map(int, name[2:].split("x"))
        return W.random_smooth(nr, nz, 0, 5)
    raise SystemExit(f"unknown workload {name}")


def run_case(P, torch, case):
    name, _, opts = case.partition(":")
    w = workload(name)
    s = P.PoissonSolver.for_workload(w)
    nsw, prof = 600, 1
    for kv in filter(None, opts.split(",")):
        k, v = kv.split("=")
        if k == "nsw":
            nsw = int(v)
        elif k == "prof":
            prof = int(v)
        else:
            s.set_option(k, int(v))
    s.set_option("prof", prof)
    rho = torch.from_numpy(w.rho).cuda()
    phi = torch.zeros_like(rho)
    ms = []
    for _ in range(4):
        phi.zero_()
        s.solve(rho, phi, 0.0, nsw)
        ms.append(s.stat("sweep_ms"))
    st = {k: s.stat(k) for k in ("path", "shape", "halo", "ds", "ring", "tblock", "ctas", "tile_w", "tile_h", "redundancy")}
    line = (f"{case:42s} ms/{nsw}={min(ms):.3f} clk/sweep={min(ms) * 1e-3 * 1.965e9 / nsw:.0f} "
            + " ".join(f"{k}={int(v) if v == int(v) else round(v, 2)}" for k, v in st.items()))
    if prof and st["path"] == 2:
        hs = max(1.0, s.stat("prof_mean7"))
        line += " | per half-sweep: " + " ".join(f"{n}={s.stat('prof_mean%d' % i) / hs:.0f}" for i, n in enumerate(NAMES))
    s.close()
    return line


def scan(P, torch, name, nsw=600, top=12):
    w = workload(name)
    rho = torch.from_numpy(w.rho).cuda()
    phi = torch.zeros_like(rho)
    rows = []
    for shape in range(16):
        for mode in ("block", "halo", "ds"):
            for tb in ([1, 2, 3, 4, 6, 8, 10, 12] if mode == "block" else [12]):
                s = P.PoissonSolver.for_workload(w)
                try:
                    s.set_option("path", 2); s.set_option("shape", shape); s.set_option("tblock", tb)
                    s.set_option("halo", 0 if mode == "block" else 1)
                    if mode != "block":
                        s.set_option("ds", 1 if mode == "ds" else 0)
                    ms = []
                    for _ in range(3):
                        phi.zero_()
                        s.solve(rho, phi, 0.0, nsw)
                        ok = (int(s.stat("path")) == 2 and int(s.stat("shape")) == shape
                              and int(s.stat("halo")) == (mode != "block") and int(s.stat("ds")) == (mode == "ds"))
                        if not ok:
                            break
                        ms.append(s.stat("sweep_ms"))
                    if ok:
                        rows.append((min(ms) * 1e-3 * 1.965e9 / nsw, shape, mode, tb, int(s.stat("ctas")),
                                     int(s.stat("tile_w")), int(s.stat("tile_h")), s.stat("redundancy")))
                except P.SnPoissonError:
                    pass
                s.close()
    rows.sort()
    out = [run_case(P, torch, f"{name}:prof=0").replace(name + ":prof=0", name + " (planner's pick)")]
    out += ["  clk/sweep=%.0f shape=%d %s m=%d ctas=%d tile=%dx%d redundancy=%.2f" % r for r in rows[:top]]
    return out


def main(argv):
    import torch
    import paper_1507_08549_b200 as P
    P.load()
    if argv and argv[0] == "--scan":
        for name in argv[1:]:
            print("\n".join(scan(P, torch, name)), flush=True)
        return
    for case in argv:
        print(run_case(P, torch, case), flush=True)


if __name__ == "__main__":
    main(sys.argv[1:])
