#!/usr/bin/env python
"""bench.py -- headline measurement of the B200 multigrid pressure solver.

Step  = one pass of the whole hot path on one batch of synthetic
        input: mg_set_density(rho) + mg_solve(rhs, p0 = 0) to rtol on the 512^3 drop-film
        workload (BASELINE.json configs[3], "config 4": the paper's per-device load,
        PAPER.md:196/218), V(3,3), 8 levels.
value = fine-grid smoother cell updates per second, N * (nu1+nu2) * cycles / t_step
        [Gcell-updates/s], inputs resident in HBM, whole-step time in the denominator
        (norm passes, coefficient setup and mean removal included).
Also on the line: time-to-rtol, the time of one bare V-cycle (graph replay) with its
Gcell-updates/s and fraction of the B_sched HBM roofline, the roofline of the dominant
kernel (level-0 sweep) timed with CUDA events, the same metric end to end from host
buffers (mg_solve_host), and the CPU oracle on a bounded sample.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload config4]

N > 1 (torchrun): the path does not shard (replicas only); every rank solves
its own replica, value = total units / max-over-ranks time ("scaling": "weak").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "V-cycle Gcell-updates/s (time-to-rtol 1e-8 at 512^3 fp64; % HBM roofline alongside)"
UNIT = "Gcell-updates/s"

# algorithmic HBM bytes: level-0 sweep pass 32 B/cell
# (p read+write, f, a); coarse-level pass 48 B/cell; whole V(3,3) cycle per fine cell:
B_SWEEP_L0 = 32.0


def b_sched_per_fine_cell(nu1, nu2):
    """SURVEY §8(d) B_sched: nu1 sweeps in one pass + residual/restrict + prolong/correct/
    first post-sweep + remaining post-sweeps in one pass; coarse levels 5 arrays."""
    l0 = 32.0 + 25.0 + 33.0 + (32.0 if nu2 > 1 else 0.0)
    lc = 48.0 + 41.0 + 49.0 + (48.0 if nu2 > 1 else 0.0)
    return l0 + lc / 7.0


def b_sweep_per_fine_cell(nu1, nu2):
    l0 = 32.0 * (nu1 + nu2) + 25.0 + 17.0
    lc = 48.0 * (nu1 + nu2) + 41.0 + 17.0
    return l0 + lc / 7.0


def parse_workload(name: str):
    name = name.lower()
    if not name.startswith("config"):
        raise SystemExit("--workload must look like config4 or config3@128")
    body = name[len("config"):]
    if "@" in body:
        c, n = body.split("@")
        return int(c), int(n)
    return int(body), None


def workload_config(w, wname):
    """The keys of `config` that identify the workload: the same in both arms."""
    return {"workload": wname, "cells": list(w.n), "bc": list(w.bc), "cycle": f"V({w.nu1},{w.nu2})",
            "rtol": w.rtol, "step": "mg_set_density + mg_solve from p=0", "parallelism": "replicas only"}


def peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self._stop, self._t = index, [], threading.Event(), None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True,
                                     timeout=5).stdout.strip()
                if out:
                    self.rows.append([t.strip() for t in out.split(",")])
            except Exception:
                pass
            self._stop.wait(0.2)

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=6)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for nm, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle as it stands, on the host cores
# ------------------------------------------------------------------------------------
def oracle_sample(w, repeats=1, min_seconds=0.0):
    """Bounded sample of the workload on the CPU oracle: set_density + `repeats` x
    (one V(nu1,nu2) cycle + residual norm).  Returns (seconds per repeat, threads)."""
    from oracle import mgo
    from oracle.mgo import Oracle

    o = Oracle(w.n, w.h, w.bc, w.nu1, w.nu2)
    o.set_density(w.rho)
    p = np.zeros(o.shape)
    times = []
    while len(times) < repeats or (min_seconds and sum(times) < min_seconds and len(times) < 40):
        t0 = time.perf_counter()
        o.vcycle(w.rhs, p)
        o.residual(w.rhs, p)
        times.append(time.perf_counter() - t0)
    o.close()
    return times, mgo.threads()


def run_reference(args, w, wname):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # warm-up + timed steps; each step = one V-cycle + norm on the full workload
    times, thr = oracle_sample(w, repeats=args.warmup + args.steps)
    t = times[args.warmup:]
    per = float(np.mean(t))
    val = w.ncells * (w.nu1 + w.nu2) / per / 1e9
    sample = (f"1 V({w.nu1},{w.nu2}) cycle + 1 residual norm per step on {wname} "
              "(a bounded sample of the step: the solve is 17 such cycles at 512^3)")
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": per * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(w, wname),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": thr, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    if args.full_solve:
        # the oracle's whole solve (time-to-rtol, cycle count), once
        from oracle.mgo import Oracle
        o = Oracle(w.n, w.h, w.bc, w.nu1, w.nu2)
        o.set_density(w.rho)
        p = np.zeros(o.shape)
        t0 = time.perf_counter()
        st, cyc, rel, _ = o.solve(w.rhs, p, w.rtol, 60)
        line["full_solve"] = {"seconds": time.perf_counter() - t0, "cycles": cyc, "relres": rel, "status": st}
        o.close()
    try:
        import platform
        cpu = [l.split(":", 1)[1].strip() for l in open("/proc/cpuinfo") if l.startswith("model name")]
        line["host"] = {"nproc": os.cpu_count(), "cpu": cpu[0] if cpu else platform.processor()}
    except OSError:
        pass
    print(json.dumps(line))


# ------------------------------------------------------------------------------------
# CUDA arm
# ------------------------------------------------------------------------------------
def aggregate_replicas(times_ms, counts, dist, device):
    """Replicas only: every rank times its own independent solves.  The job's
    time is the MAX over ranks, its work the SUM over ranks; no other collective touches the
    data path.  `dist` is torch.distributed or None (single process)."""
    import torch

    t = torch.tensor(list(times_ms), dtype=torch.float64, device=device)
    c = torch.tensor(list(counts), dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return t.tolist(), c.tolist()


def free_port():
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        return sk.getsockname()[1]


def spawn_command(args, argv, environ):
    """`--gpus N` without a launcher: the command that runs this script as N ranks (one per GPU),
    or None when a launcher already did (WORLD_SIZE set) or one GPU is asked for."""
    if args.gpus <= 1 or "WORLD_SIZE" in environ:
        return None
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
            "--master-addr", "127.0.0.1", "--master-port", str(free_port()), str(ROOT / "bench.py"), *argv]


def measure_rank(args, w, wname, rank, local, dist):
    """Everything one rank measures on its own GPU (CUDA events on the solver's stream)."""
    import torch

    import paper_2605_30082_b200 as mgpkg
    from paper_2605_30082_b200 import binding as B

    torch.cuda.set_device(local)
    devname = f"cuda:{local}"
    N = w.ncells
    stream = torch.cuda.Stream(device=devname)
    m = {}

    with torch.cuda.stream(stream):
        g = mgpkg.Multigrid(w.n, w.h, w.bc, w.nu1, w.nu2, stream=stream, device=devname)
        rho_d = torch.from_numpy(w.rho).to(devname)
        rhs_d = torch.from_numpy(w.rhs).to(devname)
        p_d = torch.zeros(g.shape, dtype=torch.float64, device=devname)
        max_cycles = 60
        m["levels"] = g.num_levels

        def barrier():
            torch.cuda.synchronize()
            if dist is not None:
                dist.barrier()
            torch.cuda.synchronize()

        def step():
            g.set_density(rho_d)
            p_d.zero_()
            return g.solve(rhs_d, p_d, w.rtol, max_cycles)

        for _ in range(args.warmup):
            res = step()
        barrier()
        l0 = g.stat(B.MG_STAT_KERNEL_LAUNCHES)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with ClockSampler(local) as clocks:
            ev0.record(stream)
            cycles_total = 0
            for _ in range(args.steps):
                res = step()
                cycles_total += res[1]
            ev1.record(stream)
            barrier()
        m["t_ms"] = ev0.elapsed_time(ev1)
        m["cycles_total"] = cycles_total
        m["launches"] = g.stat(B.MG_STAT_KERNEL_LAUNCHES) - l0
        m["status"], m["cycles"], m["relres"], _ = res
        m["clocks"] = clocks.summary()

        def timed(fn, reps, warm=2):
            for _ in range(warm):
                fn()
            torch.cuda.synchronize()
            lk = g.stat(B.MG_STAT_KERNEL_LAUNCHES)
            ev0.record(stream)
            for _ in range(reps):
                fn()
            ev1.record(stream)
            torch.cuda.synchronize()
            return ev0.elapsed_time(ev1) / reps, (g.stat(B.MG_STAT_KERNEL_LAUNCHES) - lk) / reps

        # time-to-rtol: mg_solve alone, with the V-cycle of the config and with the F-cycle
        def solve_once():
            p_d.zero_()
            return g.solve(rhs_d, p_d, w.rtol, max_cycles)

        def median_solve(reps=5):
            ts = sorted(timed(solve_once, 1, warm=0)[0] for _ in range(reps))
            return ts[len(ts) // 2], ts

        g.set_density(rho_d)
        m["t_solve_ms"], m["t_solve_samples"] = median_solve()
        g.set_cycle_type(B.MG_CYCLE_F)
        solve_once()
        t_f, t_f_all = median_solve()
        rf = solve_once()
        p_d.zero_()
        t_fc, _ = timed(lambda: g.vcycle(rhs_d, p_d), 10, warm=3)
        m["f_cycle"] = {"time_to_rtol_ms": t_f, "cycles": rf[1], "relres": rf[2], "ms_per_cycle": t_fc,
                        "time_to_rtol_samples_ms": t_f_all,
                        "what": "the same solve with mg_set_cycle_type(MG_CYCLE_F): F(nu1,nu2) cycles"}
        g.set_cycle_type(B.MG_CYCLE_V)

        # bare V-cycle (graph replay), 20 launches after 3 warm-ups
        p_d.zero_()
        m["t_vc_ms"], _ = timed(lambda: g.vcycle(rhs_d, p_d), 20, warm=3)
        m["launches_per_vcycle"] = g.stat(B.MG_STAT_LAUNCHES_PER_VCYCLE)

        # the kernels of level 0, one by one (CUDA events on the launching stream; every call
        # below is one or two launches of the named kernel, counted by the library)
        kern = {}
        p_d.zero_()
        g.set_option(B.MG_OPT_SWEEP_FUSE, 3)
        t, nl = timed(lambda: g.level_smooth(0, 4, rhs_d, p_d), 10)
        kern["k_rbt<NS=2> two sweeps per pass"] = {"ms": t / nl, "bytes_per_cell": 32.0, "sweeps_per_launch": 2}
        g.set_option(B.MG_OPT_SWEEP_FUSE, 1)
        t, nl = timed(lambda: g.level_smooth(0, 2, rhs_d, p_d), 10)
        kern["k_rbt<NS=1> one sweep per pass"] = {"ms": t / nl, "bytes_per_cell": 32.0, "sweeps_per_launch": 1}
        g.set_option(B.MG_OPT_SWEEP_FUSE, 2)
        e1_d = torch.zeros(g.level_shape(1), dtype=torch.float64, device=devname)
        t, nl = timed(lambda: g.level_prolong_add(0, e1_d, p_d), 10)
        kern["k_prolong_stream"] = {"ms": t / nl, "bytes_per_cell": 17.0}
        t, nl = timed(lambda: g.residual(rhs_d, p_d), 10)
        kern["mg_residual call: k_resid_stream<NORM> + k_final_sum + host fetch"] = {"ms": t, "bytes_per_cell": 24.0}
        # the same streaming kernel alone (restriction variant: one launch, no host fetch)
        t, nl = timed(lambda: g.level_residual_restrict(0, rhs_d, p_d), 10)
        kern["k_resid_stream<RESTRICT>"] = {"ms": t / nl, "bytes_per_cell": 25.0}
        # two sweeps with the restriction tail = k_rbt<1> (p -> q) + k_rbt<1,RESTRICT> (q -> p): no copy back;
        # the tail pass is the call minus the one-sweep pass timed above
        g.set_option(B.MG_OPT_SWEEP_FUSE, 1)
        t, nl = timed(lambda: g.level_smooth_restrict(0, 2, rhs_d, p_d), 10)
        g.set_option(B.MG_OPT_SWEEP_FUSE, 2)
        if nl == 2:
            kern["k_rbt<NS=1,RESTRICT> sweep + residual + restriction"] = {
                "ms": t - kern["k_rbt<NS=1> one sweep per pass"]["ms"], "bytes_per_cell": 33.0, "sweeps_per_launch": 1,
                "how": "2-launch call minus the one-sweep pass"}
        del e1_d
        # level 1 (stored faces: p, bx, by, bz, f in, p out = 48 B per level-1 cell and pass)
        if g.num_levels > 2 and g.level_shape(1)[0] * g.level_shape(1)[1] * g.level_shape(1)[2] >= (1 << 24):
            n1 = g.level_shape(1)[0] * g.level_shape(1)[1] * g.level_shape(1)[2]
            f1 = torch.randn(g.level_shape(1), dtype=torch.float64, device=devname)
            p1 = torch.zeros(g.level_shape(1), dtype=torch.float64, device=devname)
            e2_d = torch.zeros(g.level_shape(2), dtype=torch.float64, device=devname)
            t, nl = timed(lambda: g.level_smooth(1, 4, f1, p1), 10)
            kern["level 1: k_rbt<NS=2,FACES> two sweeps per pass"] = {"ms": t / nl, "bytes_per_cell": 48.0, "cells": n1, "sweeps_per_launch": 2}
            g.set_option(B.MG_OPT_SWEEP_FUSE, 1)
            t, nl = timed(lambda: g.level_smooth(1, 2, f1, p1), 10)
            kern["level 1: k_rbt<NS=1,FACES> one sweep per pass"] = {"ms": t / nl, "bytes_per_cell": 48.0, "cells": n1, "sweeps_per_launch": 1}
            g.set_option(B.MG_OPT_SWEEP_FUSE, 2)
            t, nl = timed(lambda: g.level_residual_restrict(1, f1, p1), 10)
            kern["level 1: k_resid_stream<RESTRICT,FACES>"] = {"ms": t / nl, "bytes_per_cell": 41.0, "cells": n1}
            t, nl = timed(lambda: g.level_prolong_add(1, e2_d, p1), 10)
            kern["level 1: k_prolong_stream"] = {"ms": t / nl, "bytes_per_cell": 17.0, "cells": n1}
            del f1, p1, e2_d
        m["kernels"] = kern

        # set_density alone
        torch.cuda.synchronize()
        ev0.record(stream)
        g.set_density(rho_d)
        ev1.record(stream)
        torch.cuda.synchronize()
        m["t_setrho_ms"] = ev0.elapsed_time(ev1)

        # the projection step around the solve: rhs = div(u*)/dt,
        # solve, u -= dt beta grad p, on the 16-mode staggered velocity behind the workload's rhs
        proj = None
        if args.projection and getattr(w, "seed", None) is not None and tuple(w.bc) == (0, 0, 1):
            from workloads import velocity_field
            uh, vh, wh = velocity_field(w.n, w.h, w.seed)
            u0, v0, w0 = (torch.from_numpy(a).to(devname) for a in (uh, vh, wh))
            del uh, vh, wh
            ud, vd, wd = u0.clone(), v0.clone(), w0.clone()
            fd = torch.empty_like(p_d)
            dtp = 1.0
            for _ in range(2):
                g.project_rhs(ud, vd, wd, dtp, fd)
                g.project_correct(p_d, dtp, ud, vd, wd)
            torch.cuda.synchronize()
            ev0.record(stream)
            for _ in range(10):
                g.project_rhs(ud, vd, wd, dtp, fd)
            ev1.record(stream)
            torch.cuda.synchronize()
            t_rhs = ev0.elapsed_time(ev1) / 10
            ev0.record(stream)
            for _ in range(10):
                g.project_correct(p_d, dtp, ud, vd, wd)
            ev1.record(stream)
            torch.cuda.synchronize()
            t_cor = ev0.elapsed_time(ev1) / 10
            ud.copy_(u0); vd.copy_(v0); wd.copy_(w0)
            p_d.zero_()
            torch.cuda.synchronize()
            ev0.record(stream)
            pst, pcyc, prel = g.project(ud, vd, wd, dtp, p_d, fd, w.rtol, max_cycles)
            ev1.record(stream)
            torch.cuda.synchronize()
            t_proj = ev0.elapsed_time(ev1)
            g.project_rhs(ud, vd, wd, dtp, fd)
            div_after = float(torch.linalg.vector_norm(fd))
            g.project_rhs(u0, v0, w0, dtp, fd)
            div_before = float(torch.linalg.vector_norm(fd))
            proj = {"ms_per_step": t_proj, "cycles": pcyc, "relres": prel, "status": pst,
                    "rhs_ms": t_rhs, "rhs_gbs": 32.0 * N / (t_rhs * 1e-3) / 1e9,
                    "correct_ms": t_cor, "correct_gbs": 64.0 * N / (t_cor * 1e-3) / 1e9,
                    "div_after_over_before": div_after / div_before,
                    "what": "mg_project = rhs (32 B/cell) + mg_solve + correct (64 B/cell), dt = 1"}
            del u0, v0, w0, ud, vd, wd, fd

        # the paper's box: symmetry planes x-, y-, no-slip base z-,
        # outflow planes x+, y+, z+ as Dirichlet walls; same densities and rhs (no compatibility
        # condition there), V- and F-cycles
        box = None
        if args.projection and tuple(w.bc) == (0, 0, 1):
            gb = mgpkg.Multigrid(w.n, w.h, (1, 2, 1, 2, 1, 2), w.nu1, w.nu2, stream=stream, device=devname)
            gb.set_density(rho_d)
            box = {"bc6": [1, 2, 1, 2, 1, 2], "what": "mg_create6: Neumann x-, y-, z-; Dirichlet x+, y+, z+"}
            for ct, name in ((B.MG_CYCLE_V, "V"), (B.MG_CYCLE_F, "F")):
                gb.set_cycle_type(ct)
                p_d.zero_()
                gb.solve(rhs_d, p_d, w.rtol, max_cycles)
                torch.cuda.synchronize()
                p_d.zero_()
                ev0.record(stream)
                rb = gb.solve(rhs_d, p_d, w.rtol, max_cycles)
                ev1.record(stream)
                torch.cuda.synchronize()
                box[name] = {"cycles": rb[1], "relres": rb[2], "status": rb[0], "time_to_rtol_ms": ev0.elapsed_time(ev1)}
            gb.close()
            del gb

        # optional: a time sequence: the drop falls onto the film, the density
        # changes every step (set_density), the solve is warm-started from the previous pressure
        seq = None
        if args.sequence > 0 and tuple(w.bc) == (0, 0, 1):
            from workloads import sequence_density
            cfg_id, n_over = parse_workload(args.workload)
            rows = []
            p_d.zero_()
            for sidx in range(args.sequence):
                rho_s = torch.from_numpy(sequence_density(cfg_id, n_over, sidx, args.sequence)).to(devname)
                torch.cuda.synchronize()
                ev0.record(stream)
                g.set_density(rho_s)
                ev1.record(stream)
                torch.cuda.synchronize()
                t_sd = ev0.elapsed_time(ev1)
                ev0.record(stream)
                st_s, cyc_s, rel_s, _ = g.solve(rhs_d, p_d, w.rtol, max_cycles)      # warm start
                ev1.record(stream)
                torch.cuda.synchronize()
                rows.append({"step": sidx, "set_density_ms": t_sd, "solve_ms": ev0.elapsed_time(ev1),
                             "cycles": cyc_s, "status": st_s})
                del rho_s
            seq = {"steps": rows, "what": "drop centre falls 0.8 r onto its config position in equal steps; "
                   "rhs fixed; p warm-started from the previous step (step 0 from p = 0)"}
            g.set_density(rho_d)

        # end to end from pinned host buffers through mg_solve_host
        rho_h = torch.from_numpy(w.rho).pin_memory()
        rhs_h = torch.from_numpy(w.rhs).pin_memory()
        p_h = torch.empty(g.shape, dtype=torch.float64).pin_memory()
        e2e_steps = max(1, min(args.steps, 3))
        g.solve_host(rho_h, rhs_h, p_h, w.rtol, max_cycles)          # warm-up (allocates staging)
        barrier()
        ev0.record(stream)
        e2e_cycles = 0
        for _ in range(e2e_steps):
            e2e_cycles += g.solve_host(rho_h, rhs_h, p_h, w.rtol, max_cycles)[1]
        ev1.record(stream)
        barrier()
        m["t_e2e_ms"] = ev0.elapsed_time(ev1)
        m["e2e_cycles"], m["e2e_steps"] = e2e_cycles, e2e_steps
    m["proj"], m["seq"], m["box"] = proj, seq, box
    return m


# dram__bytes_read.sum + dram__bytes_write.sum of one launch of the dominant kernel at 512^3, from the
# `ncu --set full` capture summarised in the named file (bench.py itself never runs under ncu)
NCU_TRAFFIC_512 = {"bytes": 4.279e9 + 1.145e9, "source": "profiles/r2b_cycle.md (k_rbt<2,NONE,CELL>, 512^3: dram read + write)"}


def assemble_line(args, w, wname, world, m, t_ms, t_e2e_ms, cycles_all, e2e_cycles_all):
    """The JSON line from rank 0's measurements and the aggregated (max time, summed units)."""
    N = w.ncells
    upd = w.nu1 + w.nu2
    value = N * upd * cycles_all / (t_ms * 1e-3) / 1e9
    e2e_value = N * upd * e2e_cycles_all / (t_e2e_ms * 1e-3) / 1e9
    peak, peak_src = peaks()
    bs = b_sched_per_fine_cell(w.nu1, w.nu2) * N
    bw = b_sweep_per_fine_cell(w.nu1, w.nu2) * N
    t_vc_ms = m["t_vc_ms"]
    # per-kernel HBM roofline: algorithmic bytes of one launch / event-timed launch duration
    kernels = {}
    for name, k in m.get("kernels", {}).items():
        ach = k["bytes_per_cell"] * k.get("cells", N) / (k["ms"] * 1e-3) / 1e9
        kernels[name] = dict(k, achieved_gbs=ach, frac=ach / peak)
    # the cycle uses the two-sweep pass on level 0 from 2^26 cells (mg.cu use_fuse2), the one-sweep pass below
    fused = N >= (1 << 26)
    dom_name = "k_rbt<NS=2> two sweeps per pass" if fused else "k_rbt<NS=1> one sweep per pass"
    dom = kernels.get(dom_name)
    roof = {"bound": "hbm", "kernel": dom_name + " (level 0, p_in -> p_out: 32 B/cell per launch)",
            "achieved": dom["achieved_gbs"] if dom else None, "peak": peak, "unit": "GB/s",
            "frac": dom["frac"] if dom else None, "traffic": None, "peak_source": peak_src,
            "bytes_per_launch": 32.0 * N, "ms_per_launch": dom["ms"] if dom else None,
            "note": ("dominant by share of the V-cycle (2 launches); two red-black sweeps per HBM pass, so "
                     "its bytes per second are lower than the one-sweep pass's although each sweep is faster: "
                     "the fused pass is bound by shared-memory bandwidth and latency, not by HBM (DESIGN.md 4.1)")
                    if fused else "dominant by share of the V-cycle; one red-black sweep per HBM pass at this size",
            "sweeps_per_pass_times_frac": ((2 if fused else 1) * dom["frac"]) if dom else None,
            "sweeps_per_pass_times_frac_note": "not a roofline fraction: the 32 B/cell of one pass counted once per fused sweep",
            "kernels": kernels}
    if list(w.n) == [512, 512, 512]:
        roof["traffic"] = NCU_TRAFFIC_512["bytes"]
        roof["traffic_source"] = NCU_TRAFFIC_512["source"]
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": t_ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(w, wname),
        "solve": {"levels": m["levels"], "cycles_per_solve": m["cycles"], "relres": m["relres"],
                  "l2": f"inputs larger than L2 ({3 * N * 8 / 1e6:.0f} MB resident vs 126 MB)"},
        "time_to_rtol_ms": m["t_solve_ms"], "time_to_rtol_samples_ms": m.get("t_solve_samples"),
        "time_to_rtol_stat": "median of 5 solves", "set_density_ms": m["t_setrho_ms"],
        "f_cycle": m.get("f_cycle"),
        "time_to_rtol_best": (lambda fc: {"ms": min(m["t_solve_ms"], fc["time_to_rtol_ms"]),
                                          "cycle": "F" if fc["time_to_rtol_ms"] < m["t_solve_ms"] else "V"})(m["f_cycle"])
                             if m.get("f_cycle") else None,
        "vcycle": {"ms": t_vc_ms, "gcell_updates_per_s": N * upd / (t_vc_ms * 1e-3) / 1e9,
                   "launches": m["launches_per_vcycle"],
                   "frac_of_B_sched_roofline": (bs / (peak * 1e9)) / (t_vc_ms * 1e-3),
                   "frac_of_B_sweep_roofline": (bw / (peak * 1e9)) / (t_vc_ms * 1e-3),
                   "frac_of_B_sched_roofline_at_8000_GBs": (bs / 8000e9) / (t_vc_ms * 1e-3),
                   "B_sched_bytes": bs, "B_sweep_bytes": bw},
        "roofline": roof,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 2 * N * 8, "d2h_bytes_per_step": N * 8,
                "ms_per_step": t_e2e_ms / m["e2e_steps"], "steps": m["e2e_steps"],
                "api": "mg_solve_host (pinned host buffers)"},
        "gpu_launches": int(m["launches"]),
        "clocks": m["clocks"],
    }
    if m.get("proj") is not None:
        line["projection_step"] = m["proj"]
    if m.get("seq") is not None:
        line["time_sequence"] = m["seq"]
    if m.get("box") is not None:
        line["paper_box"] = m["box"]
    return line


def run_cuda(args, w, wname, measure=measure_rank, backend="nccl"):
    """One process per GPU: every rank measures its own replica (`measure`), the job's time is the
    MAX over ranks and its work the SUM (aggregate_replicas), rank 0 prints the line."""
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    device = "cpu"
    if world > 1:
        import torch.distributed as dist
        if backend == "nccl":
            import torch
            dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
        else:
            dist.init_process_group(backend)
    if backend == "nccl":
        device = f"cuda:{local}"
    m = measure(args, w, wname, rank, local, dist)
    (t_ms, t_e2e_ms), (cycles_all, e2e_cycles_all) = aggregate_replicas(
        [m["t_ms"], m["t_e2e_ms"]], [float(m["cycles_total"]), float(m["e2e_cycles"])], dist, device)
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    line = assemble_line(args, w, wname, world, m, t_ms, t_e2e_ms, cycles_all, e2e_cycles_all)
    if world == 1 and not args.no_cpu_baseline:
        N, upd, cycles = w.ncells, w.nu1 + w.nu2, m["cycles"]
        times_o, thr = oracle_sample(w, repeats=1, min_seconds=10.0)
        line["cpu_baseline"] = {
            "value": N * upd * len(times_o) / sum(times_o) / 1e9, "unit": UNIT, "cores": thr, "kind": "oracle",
            "sample": f"{len(times_o)} x (1 V({w.nu1},{w.nu2}) cycle + 1 residual norm) of {wname} "
                      f"({sum(times_o):.1f} s in total; a solve is {cycles} cycles)"}
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


ONLY_STEPS = ("sweep4", "sweep2", "sweep1", "sweep_restrict", "sweep_norm", "head", "residual", "resid_restrict",
              "prolong", "vcycle", "fcycle", "solve", "set_density", "box_vcycle", "box_fcycle")


def run_only(args, w):
    """`--only STEP`: launch one step of the cycle `--reps` times on the workload and print its
    CUDA-event time; the command ncu wraps for the captures under profiles/ (nothing else runs,
    no JSON line).  `--level L` selects the grid level of the single-step calls, `--kernels`,
    `--graph`, `--fuse`, `--face-log2` the library options of the same name."""
    import torch

    import paper_2605_30082_b200 as mgpkg
    from paper_2605_30082_b200 import binding as B

    step, lev = args.only, args.level
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        bc = (1, 2, 1, 2, 1, 2) if step.startswith("box_") else w.bc
        g = mgpkg.Multigrid(w.n, w.h, bc, w.nu1, w.nu2, stream=st)
        g.set_option(B.MG_OPT_KERNELS, args.kernels)
        g.set_option(B.MG_OPT_GRAPH, args.graph)
        g.set_option(B.MG_OPT_SWEEP_FUSE, args.fuse)
        if args.face_log2 is not None:
            g.set_option(B.MG_OPT_FACE_STREAM_LOG2, args.face_log2)
        if step in ("fcycle", "box_fcycle"):
            g.set_cycle_type(B.MG_CYCLE_F)
        rho = torch.from_numpy(w.rho).cuda()
        g.set_density(rho)
        shp = g.level_shape(lev)
        f = torch.from_numpy(w.rhs).cuda() if lev == 0 else torch.randn(shp, dtype=torch.float64, device="cuda")
        p = torch.zeros(shp, dtype=torch.float64, device="cuda")
        e = torch.zeros(g.level_shape(lev + 1), dtype=torch.float64, device="cuda") if lev + 1 < g.num_levels else None
        calls = {
            "sweep4": lambda: g.level_smooth(lev, 4, f, p),
            "sweep2": lambda: g.level_smooth(lev, 2, f, p),
            "sweep1": lambda: g.level_smooth(lev, 1, f, p),
            "sweep_restrict": lambda: g.level_smooth_restrict(lev, 1, f, p),
            "sweep_norm": lambda: g.level_smooth_norm(1, f, p),
            "head": lambda: g.level_prolong_smooth(lev, 1, e, f, p),
            "residual": lambda: g.residual(f, p),
            "resid_restrict": lambda: g.level_residual_restrict(lev, f, p),
            "prolong": lambda: g.level_prolong_add(lev, e, p),
            "vcycle": lambda: g.vcycle(f, p),
            "fcycle": lambda: g.vcycle(f, p),
            "box_vcycle": lambda: g.vcycle(f, p),
            "box_fcycle": lambda: g.vcycle(f, p),
            "solve": lambda: (p.zero_(), g.solve(f, p, w.rtol, 60)),
            "set_density": lambda: g.set_density(rho),
        }
        if step == "head":
            g.set_option(B.MG_OPT_PROLONG_FUSE, 1)
        run = calls[step]
        for _ in range(2):
            run()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        for _ in range(args.reps):
            run()
        e1.record(st)
        torch.cuda.synchronize()
        print(f"{step} level {lev} {w.name}: {e0.elapsed_time(e1) / args.reps:.4f} ms per rep")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="config4", help="config<k>[@n], k = 1..5 (BASELINE.json configs)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--full-solve", action="store_true",
                    help="reference arm only: also time the oracle's whole solve once")
    ap.add_argument("--sequence", type=int, default=4,
                    help="also run a K-step falling-drop sequence (set_density + warm-started solve per step)")
    ap.add_argument("--no-projection", dest="projection", action="store_false",
                    help="skip the projection-step timing (rhs + solve + correct)")
    ap.add_argument("--only", choices=ONLY_STEPS, default=None,
                    help="profiling aid: run just this step --reps times (see run_only); prints no JSON line")
    ap.add_argument("--level", type=int, default=0)
    ap.add_argument("--reps", type=int, default=5)
    ap.add_argument("--kernels", type=int, default=1)
    ap.add_argument("--graph", type=int, default=1)
    ap.add_argument("--fuse", type=int, default=2)
    ap.add_argument("--face-log2", type=int, default=None)
    args = ap.parse_args()
    if args.only:
        from workloads import make_workload
        cfg, n = parse_workload(args.workload)
        return run_only(args, make_workload(cfg, n))
    if args.warmup < 3 and args.impl == "cuda":
        args.warmup = 3
    cmd = spawn_command(args, sys.argv[1:], os.environ) if args.impl == "cuda" else None
    if cmd is not None:                 # --gpus N without a launcher: run N ranks, one per GPU
        raise SystemExit(subprocess.run(cmd).returncode)
    from workloads import make_workload

    cfg, n = parse_workload(args.workload)
    rank = int(os.environ.get("RANK", "0"))
    if args.impl == "reference" and rank != 0:
        return
    w = make_workload(cfg, n)
    wname = f"config{cfg}: {w.n[0]}^3 " + w.note
    if args.impl == "reference":
        run_reference(args, w, wname)
    else:
        run_cuda(args, w, wname)


if __name__ == "__main__":
    main()
