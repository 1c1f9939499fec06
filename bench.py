#!/usr/bin/env python
"""bench.py -- Poisson relaxation throughput (fp64 cell-updates/s) and time-to-residual per solve.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]
                    [--workload cfg0|cfg1|cfg2|cfg3|cfg3seq<N>|cfg4a|sweep<N>]

One "step" = one pass of the whole hot path over one synthetic input: multipole moments -> boundary fill ->
red-black SOR sweeps with the fused residual reduction until the device-side stopping rule fires (cold start,
phi = 0), through the C ABI (sn_poisson_solve / _solve_batch).  Default workload: BASELINE.json configs[1]
(256x256 n=1 polytrope, lmax 16, tol 1e-10).  cfg3seq<N>: one step = the warm-started sequence of N solves of
[CFG 3].  Prints ONE JSON line (rank 0).

Timing: W warm-up steps, then K steps each bracketed by CUDA events on the launching stream (the call
synchronises that stream itself); L2 is flushed (a 256 MiB write) and phi re-zeroed between steps, outside the
events; the K-step region is bracketed by barrier + torch.cuda.synchronize(); max over ranks.  `value` = all
cell-updates of the K steps / that device time (inputs resident in HBM); `e2e` = the same with pinned HOST buffers,
H2D / D2H inside the timed wall-clock region; `roofline` = 24 B x cell-updates of the relaxation kernel's launches /
their device time (the library's own CUDA events) against the measured L2 / HBM peak; `cpu_baseline` = the oracle
as it stands on one host core on a bounded sample.
`--impl reference` times the CPU oracle (oracle/, single thread) on the same workload -- a deliberately slow
program; parity and the roofline fraction are the headline, not that ratio.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import workloads as W  # noqa: E402

METRIC = "poisson_relaxation_cell_updates_per_s"
UNIT = "cell-updates/s"
BYTES_PER_UPDATE = 24.0     # phi read + f read + phi write


def make_workload(name: str):
    """Returns (label, list of Workload members, description)."""
    if name == "cfg1":
        return "cfg1: 256x256 half-plane n=1 polytrope, lmax=16, tol=1e-10, cold start", [W.cfg1()]
    if name == "cfg0":
        return "cfg0: 64x64 uniform sphere, lmax=8, omega=1.9, 4000 fixed sweeps", [W.cfg0()]
    if name == "cfg2":
        return "cfg2: 512x512 half-plane n=3 WD + 20 bubbles, lmax=16, tol=1e-10, cold start", [W.cfg2()]
    if name == "cfg3":
        return "cfg3: 1024x2048 full-plane offset WD, lmax=32, tol=1e-10, cold solve (first of the sequence)", \
            [W.cfg3().first]
    if name.startswith("cfg3seq"):
        n = int(name[7:] or 100)
        return (f"cfg3 sequence: {n} warm-started solves on 1024x2048 (rho evolves by seeded 0.1 % perturbations), "
                f"lmax=32, tol=1e-10"), [W.cfg3(nsteps=n)]
    if name == "cfg4a":
        return "cfg4a: batch of 64 x 512x512 half-plane WDs, lmax=16, tol=1e-10, cold start", W.cfg4a(64)
    if name.startswith("sweep"):
        n = int(name[5:])
        return f"cfg4b: {n}x{n} half-plane WD, lmax=16, 2000 fixed sweeps", [W.cfg4b(n, 2000)]
    raise SystemExit(f"unknown workload {name}")


class ClockSampler:
    """Samples nvidia-smi SM clocks and throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.t.join(timeout=2)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for nme, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)"
    return 6650.0, "B200_PROFILING.md fallback 6.65 TB/s (of fallback)"


def profiled_traffic(workload: str, kernel: str):
    """dram bytes per launch of the dominant kernel from the committed ncu --set full capture (profiles/), or None."""
    p = os.path.join(ROOT, "profiles", "r01b_traffic.json")
    try:
        e = json.load(open(p)).get(workload)
    except (OSError, ValueError):
        return None
    return float(e["traffic_bytes_per_launch"]) if e and e.get("kernel") == kernel else None


def l2_copy_peak_gbs(torch, mib=24, iters=40):
    """L2-resident copy bandwidth (read + write bytes), measured live the way MEASURED_PEAKS.json measures HBM:
    b.copy_(a) with a working set (2 x `mib` MiB) that stays in the 126 MB L2; best of several."""
    n = mib * (1 << 20) // 8
    a = torch.ones(n, dtype=torch.float64, device="cuda")
    b = torch.empty_like(a)
    for _ in range(5):
        b.copy_(a)
    best = 0.0
    for _ in range(5):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(iters):
            b.copy_(a)
        e1.record()
        torch.cuda.synchronize()
        best = max(best, 2.0 * n * 8 * iters / (e0.elapsed_time(e1) * 1e-3) / 1e9)
    return best


def oracle_rate(members, budget_s=12.0):
    """Times the oracle as it stands on 1 host core on a bounded sample; returns (cell-updates/s, description)."""
    import oracle as O
    O.build()
    w = members[0]
    full_cost = w.cells * 2000.0 / 1.0e8            # rough seconds for a full solve at ~1e8 updates/s
    if full_cost <= budget_s:
        t0 = time.perf_counter()
        upd, n = 0, 0
        while time.perf_counter() - t0 < budget_s * 0.8 or n == 0:
            r = O.solve_workload(members[n % len(members)])
            upd += r["sweeps"] * w.cells
            n += 1
        dt = time.perf_counter() - t0
        return upd / dt, f"{n} full solve(s) of {w.name} ({w.nr}x{w.nz}, to tol {w.tol:g} / {w.max_sweeps} sweeps)"
    nsw = max(4, int(budget_s * 1.0e8 / w.cells))
    t0 = time.perf_counter()
    O.solve(w.rho, np.zeros_like(w.rho), w.dr, w.dz, w.symmetry, w.lmax, 0.0, nsw, omega=w.omega)
    dt = time.perf_counter() - t0
    return nsw * w.cells / dt, f"moments+boundary+{nsw} sweeps of {w.name} ({w.nr}x{w.nz})"


def run_reference(args, label, members):
    """--impl reference: the CPU oracle, single thread, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle as O
    O.build()
    if hasattr(members[0], "first"):                  # the cfg3 sequence: its first (cold) solve is the sample
        members = [members[0].first]
    w = members[0]
    per_step_sweeps = None
    if w.cells * 2000.0 / 1.0e8 > 8.0:               # too slow for full solves: fixed-sweep sample per step
        per_step_sweeps = max(4, int(4.0e8 / w.cells))

    def one_step(i):
        m = members[i % len(members)]
        if per_step_sweeps is None:
            r = O.solve_workload(m)
            return r["sweeps"] * m.cells
        O.solve(m.rho, np.zeros_like(m.rho), m.dr, m.dz, m.symmetry, m.lmax, 0.0, per_step_sweeps, omega=m.omega)
        return per_step_sweeps * m.cells

    for i in range(args.warmup):
        one_step(i)
    t0 = time.perf_counter()
    upd = sum(one_step(i) for i in range(args.steps))
    dt = time.perf_counter() - t0
    value = upd / dt
    sample = (f"{args.steps} full oracle solve(s)" if per_step_sweeps is None
              else f"{args.steps} x (moments+boundary+{per_step_sweeps} sweeps)") + f" of {w.name}"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": label},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg1")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--path", type=int, default=0, help="0 auto, 1 streaming kernels, 2 resident kernel, 3 blocked kernel")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup

    label, members = make_workload(args.workload)
    if args.impl == "reference":
        run_reference(args, label, members)
        return

    import torch
    import torch.distributed as dist

    import paper_1507_08549_b200 as P
    from paper_1507_08549_b200 import build as pbuild
    from paper_1507_08549_b200.sharding import reduce_timing, shard_members

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    if rank == 0:
        pbuild.build()
    if world > 1:
        dist.barrier()
    P.load()

    # multi-GPU: batch members are sharded across ranks with no collective; a single solve runs as replicas
    idx, scaling = shard_members(len(members), rank, world)
    mine = [members[i] for i in idx]
    seq = None
    if hasattr(mine[0], "first"):                     # cfg3 sequence: rho_t precomputed on the host, solves in order
        seq = mine[0]
        mine = [seq.first]
    w0 = mine[0]
    nb = len(mine)
    solver = P.PoissonSolver.for_workload(w0)
    if args.path:
        solver.set_option("path", args.path)
    rho_h = np.stack([m.rho for m in mine]) if nb > 1 else w0.rho
    rho = torch.from_numpy(rho_h).cuda()
    phi = torch.zeros_like(rho)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    cells = w0.cells

    rho_seq = None
    if seq is not None:
        rhos, r_t = [w0.rho], w0.rho
        for t in range(1, seq.nsteps):
            r_t = seq.step(r_t, t)
            rhos.append(r_t)
        rho_seq = [torch.from_numpy(r).cuda() for r in rhos]

    acc = {"sweep_ms": 0.0, "setup_ms": 0.0, "launches": 0, "sweep_launches": 0}

    def solve_dev():
        """One step: one solve (or batch), or the whole warm-started sequence; accumulates the library's counters."""
        for k in acc:
            acc[k] = 0
        out = []
        for rt in (rho_seq if rho_seq is not None else [rho]):
            res = solver.solve(rt, phi, w0.tol, w0.max_sweeps)        # phi carries over inside a sequence
            out += res if isinstance(res, list) else [res]
            for k in acc:
                acc[k] += solver.stat(k)
        return out

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        phi.zero_()
        solve_dev()

    sampler = ClockSampler(local_rank)
    step_ms, sweep_ms, setup_ms, launches, updates = [], [], [], 0, 0
    results = None
    barrier()
    sampler.start()
    t_region = time.perf_counter()
    for _ in range(args.steps):
        phi.zero_()
        flush.fill_(1)                                    # L2 flush between timed iterations
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        results = solve_dev()
        e1.record()
        torch.cuda.synchronize()
        step_ms.append(e0.elapsed_time(e1))
        sweep_ms.append(acc["sweep_ms"])
        setup_ms.append(acc["setup_ms"])
        launches += int(acc["launches"])
        updates += sum(r.sweeps for r in results) * cells
    barrier()
    region_s = time.perf_counter() - t_region
    clocks = sampler.stop()
    assert all(r.status == 0 for r in results), results

    # end to end with HOST buffers (pinned), H2D + D2H inside the timed region.  Single solve: through the C ABI
    # (sn_poisson_solve_host).  Batch / sequence: every solve's rho goes host -> device and its phi device -> host
    # around the device call (what a hydro step that lives on the host does).
    has_e2e = True
    e2e_ms, e2e_upd, h2d_bytes, d2h_bytes = [], 0, 0, 0
    if nb == 1 and seq is None:
        rho_pin = torch.from_numpy(w0.rho).pin_memory()
        phi_pin = torch.zeros(w0.rho.shape, dtype=torch.float64).pin_memory()
        rho_np, phi_np = rho_pin.numpy(), phi_pin.numpy()
        h2d_bytes, d2h_bytes = 2 * cells * 8, cells * 8
        for i in range(args.warmup + args.steps):
            phi_np[...] = 0.0
            flush.fill_(1)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            r = solver.solve_host(rho_np, phi_np, w0.tol, w0.max_sweeps)
            dt = time.perf_counter() - t0
            if i >= args.warmup:
                e2e_ms.append(dt * 1e3)
                e2e_upd += r.sweeps * cells
    else:
        host_rhos = ([torch.from_numpy(r).pin_memory() for r in rhos] if seq is not None
                     else [torch.from_numpy(rho_h).pin_memory()])
        phi_host = torch.zeros(rho.shape, dtype=torch.float64).pin_memory()
        rho_dev = torch.empty_like(rho)
        n_e2e = min(args.steps, 3)                        # these steps are long; a few suffice
        h2d_bytes = sum(t.numel() * 8 for t in host_rhos) + phi_host.numel() * 8
        d2h_bytes = len(host_rhos) * phi_host.numel() * 8
        for i in range(1 + n_e2e):
            phi_host.zero_()
            flush.fill_(1)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            phi.copy_(phi_host, non_blocking=True)
            sw = 0
            for hr in host_rhos:
                rho_dev.copy_(hr, non_blocking=True)
                res = solver.solve(rho_dev, phi, w0.tol, w0.max_sweeps)
                sw += sum(x.sweeps for x in res) if isinstance(res, list) else res.sweeps
                phi_host.copy_(phi, non_blocking=True)
                torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            if i >= 1:
                e2e_ms.append(dt * 1e3)
                e2e_upd += sw * cells
    e2e_time = sum(e2e_ms) * 1e-3
    e2e_steps = len(e2e_ms)

    total_ms = float(sum(step_ms))
    counters = [float(updates), float(launches), float(e2e_upd)]
    dev = torch.device("cuda", local_rank)
    total_ms, (updates_all, launches_all, e2e_upd_all) = reduce_timing(total_ms, counters, world, dev)
    e2e_time_all, _ = reduce_timing(e2e_time * 1e3, [], world, dev)
    e2e_time_all *= 1e-3
    launches_all = int(launches_all)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    value = updates_all / (total_ms * 1e-3)
    # roofline of the dominant kernel (the relaxation sweep), from the library's own CUDA events on the stream
    path = int(solver.stat("path"))
    sw_ms = float(np.mean(sweep_ms))
    sweeps_per_step = sum(r.sweeps for r in results)
    sweep_launches = max(1, int(acc["sweep_launches"]))
    alg_bytes_per_launch = BYTES_PER_UPDATE * sweeps_per_step * cells / sweep_launches
    achieved = alg_bytes_per_launch / (sw_ms * 1e-3 / sweep_launches) / 1e9
    hbm_peak, hbm_src = measured_peaks()
    working_set = 16.0 * cells * nb
    if working_set > 100e6:
        bound, peak, src = "hbm", hbm_peak, hbm_src
    else:
        bound, peak = "l2", l2_copy_peak_gbs(torch)
        src = "L2-resident torch copy (2 x 24 MiB, read+write bytes), measured live in this run (of measured)"
    kernel = {1: "k_halfsweep", 2: "k_sor_resident", 3: "k_sor_blocked"}[path]
    roofline = {"bound": bound, "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": profiled_traffic(args.workload, kernel), "kernel": kernel,
                "alg_bytes_per_launch": alg_bytes_per_launch, "launch_ms": sw_ms / sweep_launches,
                "sweep_launches_per_step": sweep_launches, "peak_source": src,
                "frac_of_hbm_peak": achieved / hbm_peak,
                # the limiter once phi stays on chip: 7 fp64 instructions per update against 64 lanes / clock / SM
                # (DESIGN.md section 6); for information, the judged fraction is `frac`
                "fp64_pipe_frac": value * 7.0 / (148 * 64 * 1.965e9)}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
        "scaling": scaling, "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": label, "grid": [w0.nr, w0.nz], "batch_per_gpu": nb, "lmax": w0.lmax,
                   "tol": w0.tol, "l2": "flushed between timed solves (256 MiB write)",
                   "path": {1: "streaming", 2: "resident", 3: "blocked"}.get(path, str(path)),
                   "tblock": int(solver.stat("tblock")), "ctas": int(solver.stat("ctas")),
                   "mode": ("halo" if solver.stat("halo") else "block") if path == 2 else None,
                   "tile": [int(solver.stat("tile_w")), int(solver.stat("tile_h"))],
                   "parallelism": "replicas" if scaling == "weak" else f"batch sharded x{world}, no collective"},
        "time_to_residual_ms": total_ms / args.steps, "sweeps_per_solve": [r.sweeps for r in results][:8],
        "solves_per_step": len(results), "sweeps_per_step": sum(r.sweeps for r in results),
        "final_residual": results[0].residual,
        "setup_ms": float(np.mean(setup_ms)), "sweep_ms": sw_ms,
        "gpu_launches": launches_all, "clocks": clocks, "roofline": roofline,
        "region_wall_s": region_s,
    }
    out["e2e"] = {"value": e2e_upd_all / e2e_time_all, "unit": UNIT,
                  "h2d_bytes_per_step": h2d_bytes, "d2h_bytes_per_step": d2h_bytes,
                  "ms_per_step": e2e_time_all / e2e_steps * 1e3, "steps": e2e_steps,
                  "api": "sn_poisson_solve_host" if (nb == 1 and seq is None) else
                         "pinned tensor.copy_ + sn_poisson_solve / _solve_batch + copy back, per solve"}
    if not args.no_cpu_baseline and world == 1:
        v, sample = oracle_rate(mine)
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                               "host_cores_available": os.cpu_count()}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
