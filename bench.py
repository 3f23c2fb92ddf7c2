#!/usr/bin/env python
"""Benchmark of the CHFPE hot path (arXiv 2509.25840) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg4]

A "step" is one pass of the whole hot path over one batch: one fourth-order Runge-Kutta step of the whole
hierarchy (steps a1-a3 of DESIGN.md: Liouvillian stencil + hierarchy couplings + stage combine, 4 fused stage
kernels) followed by the phase-space expectation <C> of element 0 (step a5), i.e. one sample of the linear
response protocol of section IV.C.1.  Metric (BASELINE.json): phase-space cell-updates/s in
fp64 = cells * steps / time; one cell-update advances all K hierarchy elements of one grid cell by one step.

Workload at N = 1: BASELINE.json configs[3] ("cfg4": 3 modes, 16^6 grid, depth 3 -> 20 elements), the
configuration the north-star target is quoted on.  Inputs are synthetic (chfpe_inputs.py): the state is the
analytic equilibrium kicked by mu = q1+q2+q3.  One state array (2.7 GB) exceeds the 126 MB L2, so every timed
iteration streams from HBM ("inputs larger than L2").

N > 1 (torchrun): a single propagation does not shard ("replicas only"); every rank propagates its
own replica, no data-path collective, scaling = weak; time = max over ranks.

--impl reference times the CPU oracle (oracle/, test infrastructure) as it stands on the host cores, rank 0 only.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import chfpe_inputs as ci  # noqa: E402

METRIC = "phase-space cell-updates/s (fp64)"
UNIT = "cell-updates/s"
BYTES_PER_VALUE_STEP_SURVEY = 128.0        # classical RK4, 4 arrays, 9R + 7W per value per step
HBM_NOMINAL_GBS = 8000.0                   # "about 8 TB/s", BASELINE.json north_star


def profiled_traffic(pattern="r*_stage_kernel_ncu_full.txt", key="dram_bytes_per_launch"):
    """A `key=value` figure of the stage kernel from the latest committed ncu --set full summary (profiles/), or None
    (DRAM bytes per launch by default).  ncu cannot run inside a timed benchmark, so these come from the committed
    capture of the same command; `roofline.traffic_source` names the file."""
    import glob
    import re
    best = None
    for f in sorted(glob.glob(os.path.join(ROOT, "profiles", pattern))):
        m = re.search(r"^%s=([0-9.eE+]+)" % key, open(f).read(), flags=re.M)
        if m:
            best = float(m.group(1))
    return best


def profile_file(pattern="r*_stage_kernel_ncu_full.txt"):
    import glob
    fs = sorted(glob.glob(os.path.join(ROOT, "profiles", pattern)))
    return os.path.relpath(fs[-1], ROOT) if fs else None


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index = index
        self.rows = []
        self.proc = None

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.rows.append([x.strip() for x in line.split(",")])
        except Exception:
            pass

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()          # exact PID of the child we started
        self.join(timeout=2.0)
        sm, mx, reasons = [], 0.0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = max(mx, float(r[1]))
            except Exception:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        med = sm[len(sm) // 2] if sm else None
        return {"sm_mhz": med, "sm_max_mhz": mx or None, "reasons": sorted(reasons), "samples": len(sm)}


def obs(mod, kind, M):
    d = ci.observable(kind, M)
    return mod.make_observable(d["c0"], d["lin_q"], d["quad"], d["lin_p"])


def cpu_oracle_time(cfg, steps, warmup=0, threads=0):
    """Time the oracle as it stands: equilibrium, kick(mu), then `steps` x (RK4 step + <mu>).  Returns
    (seconds, threads, K, cells).  threads = 0: all cores (the OpenMP default), else that many."""
    import oracle
    all_threads = oracle.set_threads(0)
    if threads:
        oracle.set_threads(threads)
    o = oracle.RefCHFPE(cfg)
    mu = obs(oracle, "mu", cfg["n_modes"])
    o.equilibrate()
    o.kick(mu)
    for _ in range(warmup):
        o.step(1, cfg["dt"]); o.expect(mu)
    t0 = time.perf_counter()
    for _ in range(steps):
        o.step(1, cfg["dt"]); o.expect(mu)
    dt = time.perf_counter() - t0
    K, cells = o.K, o.cells
    o.close()
    used = oracle.set_threads(0)
    oracle.set_threads(all_threads)
    return dt, used, K, cells


def cpu_baseline_record(workload):
    """SURVEY 8(d) "timing the oracle beside it": all-core time on the full workload (one RK4 step + <mu>, about 6 s at
    config 4) and single-core time on the 12^6 shrink of the same model (a full-size single-core step would take
    90 s), both as cell-updates/s, with the core count and the CPU model."""
    cfg_c, sample = pick_cpu_sample(workload)
    tc, threads, Kc, cells_c = cpu_oracle_time(cfg_c, 1, 0)
    rec = {"value": cells_c / tc, "unit": UNIT, "cores": threads, "kind": "oracle",
           "sample": "%s, 1 RK4 step + <mu> (%.1f s)" % (sample, tc), "nproc": os.cpu_count(), "cpu_model": cpu_model()}
    small = {"cfg4": "cfg4s12", "cfg5": "cfg4s12", "cfg3": "cfg3s"}.get(workload)
    if small:
        c1 = ci.config(small)
        t1, th1, K1, cells1 = cpu_oracle_time(c1, 1, 0, threads=1)
        rec["value_1core"] = cells1 / t1
        rec["sample_1core"] = "%s (%s grid, same model), 1 RK4 step + <mu> on 1 core (%.1f s)" % (
            small, "x".join(str(x) for x in ci.grid_shape(c1)), t1)
    return rec


def pick_cpu_sample(workload):
    """Bounded sample of the workload for the oracle: the full grid if the host has the RAM (4 state-sized
    arrays + scratch), else the 12^6 shrink of the same model (stated in `sample`)."""
    cfg = ci.config(workload)
    cells = 1
    for s in range(cfg["n_modes"]):
        cells *= cfg["nq"][s] * cfg["np"][s]
    K = {1: cfg["depth"] + 1, 2: (cfg["depth"] + 1) * (cfg["depth"] + 2) // 2,
         3: (cfg["depth"] + 1) * (cfg["depth"] + 2) * (cfg["depth"] + 3) // 6}[cfg["n_modes"]]
    need = 5 * K * cells * 8
    try:
        import psutil
        avail = psutil.virtual_memory().available
    except Exception:
        avail = 0
    if workload == "cfg4" and avail < need + (8 << 30):
        return ci.config("cfg4s12"), "cfg4 model on a 12^6 grid (host RAM too small for 16^6)"
    return cfg, "%s at full size" % workload


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    if args.protocol == "2d":
        return run_2d_reference(args)
    cfg, sample = pick_cpu_sample(args.workload)
    steps = max(1, args.steps)
    # keep the whole run within a few minutes: the oracle does ~1e7 value-updates/s on 8 cores
    t_probe, threads, K, cells = cpu_oracle_time(cfg, 1, 0)
    budget = 150.0
    max_steps = max(1, int(budget / max(t_probe, 1e-3)) - 1)
    warm = min(args.warmup, max(0, max_steps // 4))
    steps = min(steps, max(1, max_steps - warm))
    dt, threads, K, cells = cpu_oracle_time(cfg, steps, warm)
    val = cells * steps / dt
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": warm, "ms_per_step": 1e3 * dt / steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "sample": sample, "K": K, "cells": cells,
                       "note": "CPU oracle (oracle/chfpe_ref.c, OpenMP) on the host cores; a deliberately plain program"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle",
                             "sample": "%s, %d RK4 steps + <mu> each" % (sample, steps), "nproc": os.cpu_count(),
                             "cpu_model": cpu_model()},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def run_ours(args):
    import numpy as np
    import torch
    import paper_2509_25840_b200 as P

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: a CUDA device is required (the CHFPE path has no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = ci.config(args.workload, scheme=args.scheme)
    cfg4 = args.workload == "cfg4" and args.scheme == "central4"
    M = cfg["n_modes"]
    g = P.CHFPE(cfg, batch=1, device="cuda:%d" % local)
    mu = obs(P, "mu", M)
    dt = cfg["dt"]
    K, cells = g.K, g.cells
    values = K * cells
    steps, warm = args.steps, max(args.warmup, 3)

    # ---- device-resident arm: equilibrium, kick(mu), W warm-up steps, then exactly K x (step + <mu>) ----
    g.equilibrate(residual=False)
    g.kick(mu)
    g.response_1d(None, mu, warm + 1, 1, dt)
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
        time.sleep(0.3)
    n0 = g.launch_count()
    g.profile_enable(True)
    g.profile_read()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    R = g.response_1d(None, mu, steps + 1, 1, dt)        # K steps, K+1 expectation samples, one D2H of K+1 doubles
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    stage_ms, stage_n = g.profile_read()
    g.profile_enable(False)
    launches = g.launch_count() - n0
    clocks = sampler.stop() if sampler else None
    if not np.all(np.isfinite(R)):
        raise SystemExit("bench.py: non-finite response")

    # ---- end-to-end arm: host state in pinned memory -> import (H2D) -> kick, K x (step + <mu>) -> R on host ----
    X0 = g.export_state_device().cpu().pin_memory()       # canonical layout, K*cells doubles, pinned
    R_host_bytes = 8 * (steps + 1)
    barrier()
    e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e2.record()
    g.import_state(X0.numpy())
    g.response_1d(None, mu, steps + 1, 1, dt)
    e3.record()
    barrier()
    ms_e2e = e2.elapsed_time(e3)

    t = torch.tensor([ms, ms_e2e], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms, ms_e2e = float(t[0]), float(t[1])

    if rank == 0:
        peak, peak_src = measured_peaks()
        value = world * cells * steps / (ms * 1e-3)
        e2e = world * cells * steps / (ms_e2e * 1e-3)
        # dominant kernel: the fused RK-stage kernel.  Algorithmic (compulsory) bytes per launch, DESIGN.md section 5:
        # stage 1 reads y and writes v (16 B/value), stages 2-4 read v, read y, write the next v (24 B/value);
        # averaged over the four launches of a step: 22 B/value/launch = 88 B/value/step.
        # Reported two ways: `achieved` / `frac` use the survey's fixed F_alg accounting, 128 B per value
        # per step = 32 B per value per launch (classical four-array RK4), so traffic the implementation saves shows;
        # `frac_compulsory_88B` uses the 22 B per value per launch this three-array Horner form must move.
        alg_bytes_launch = values * (BYTES_PER_VALUE_STEP_SURVEY / 4.0)
        compulsory_bytes_launch = values * 22.0
        kern_ms = stage_ms / max(stage_n, 1)
        achieved = alg_bytes_launch / (kern_ms * 1e-3) / 1e9
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warm,
            "ms_per_step": ms / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "modes": M, "grid": "x".join(str(x) for x in g.shape), "K": K,
                       "cells": cells, "depth": cfg["depth"], "dt": dt, "scheme": cfg["scheme"], "gauge": cfg["gauge"],
                       "integrator": "RK4 (Horner form)", "l2": "inputs larger than L2 (state array 2.7 GB vs 126 MB)",
                       "parallelism": "replicas x%d" % world if world > 1 else "single GPU"},
            "value_updates_per_s": value * K,
            "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": values * 8.0 / steps,
                    "d2h_bytes_per_step": R_host_bytes / steps,
                    "note": "one chfpe_import_state of the pinned host state (H2D, whole state once per job) + "
                            "chfpe_response_1d returning R on the host, all inside the timed region"},
            "gpu_launches": int(launches),
            "clocks": clocks,
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "accounting": "achieved/frac: SURVEY 8(d) F_alg, 128 B per value per step = 32 B per value per "
                                       "launch, against the measured copy peak; frac_compulsory_88B: the 22 B per value "
                                       "per launch of the three-array Horner form",
                         "frac_compulsory_88B": compulsory_bytes_launch / (kern_ms * 1e-3) / 1e9 / peak,
                         "frac_of_8TBs": achieved / HBM_NOMINAL_GBS,
                         "traffic": profiled_traffic() if cfg4 else None,
                         "fp64_pipe_pct": profiled_traffic(key="fp64_pipe_pct") if cfg4 else None,
                         "l2_hit_pct": profiled_traffic(key="l2_hit_pct") if cfg4 else None,
                         "traffic_source": ("ncu --set full capture of the same command, %s" % profile_file()) if cfg4 else None,
                         "peak_source": peak_src, "kernel": "RK stage (%s)" % g.stage_kernel_name(),
                         "kernel_ms": kern_ms, "kernel_launches_timed": int(stage_n),
                         "kernel_share_of_step": stage_ms / ms,
                         "algorithmic_bytes_per_launch": alg_bytes_launch,
                         "compulsory_bytes_per_launch": compulsory_bytes_launch,
                         "frac_survey_128B_of_8TBs": values * BYTES_PER_VALUE_STEP_SURVEY * steps
                         / (ms * 1e-3) / 1e9 / HBM_NOMINAL_GBS},
        }
        if world == 1 and not args.no_cpu:
            line["cpu_baseline"] = cpu_baseline_record(args.workload)
    g.close()
    del X0
    torch.cuda.empty_cache()
    if rank == 0:
        if world == 1 and not args.no_2d:                 # third part of the metric: 2D THz-Raman wall time (config 5)
            try:
                line["two_d"] = two_d_record(P, batch=5, n1=4, n2=8)
            except Exception as exc:                      # e.g. not enough device memory for five replica slots
                line["two_d"] = {"unavailable": str(exc)[:200]}
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


FULL_2D_REPLICA_STEPS = 63 + 64 * 255                    # BASELINE configs[4]: 64 t1 x 256 t2 delays, stride 1


def two_d_record(P, batch=5, n1=4, n2=8, workload="cfg5"):
    """Third part of BASELINE.json's metric, "2D THz-Raman wall time": chfpe_response_2d (A = mu, B = C = alpha) on
    config 5 (20^6 grid, 20 elements, t1 replicas batched into HBM) timed end to end on a bounded n1 x n2 sample of
    the delay grid -- trajectory steps, replica copies, kicks, batched propagation, expectations, D2H of R -- and
    extrapolated linearly in replica-steps to the full 64 x 256 grid (labelled as such)."""
    import numpy as np
    import torch
    cfg = ci.config(workload)
    M = cfg["n_modes"]
    g = P.CHFPE(cfg, batch=batch)
    try:
        mu, al = obs(P, "mu", M), obs(P, "alpha", M)
        g.equilibrate(residual=False)
        g.response_2d(mu, al, al, [0, 1], [0, 1], cfg["dt"])          # warm-up
        g.equilibrate(residual=False)
        t1, t2 = list(range(n1)), list(range(n2))
        n0 = g.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        R = g.response_2d(mu, al, al, t1, t2, cfg["dt"])
        e1.record()
        torch.cuda.synchronize()
        sec = e0.elapsed_time(e1) * 1e-3
        rsteps = (n1 - 1) + n1 * (n2 - 1)                           # trajectory steps + replica steps
        rec = {"metric": "2D THz-Raman wall time", "workload": workload + " chfpe_response_2d, A=mu B=alpha C=alpha",
               "grid": "x".join(str(x) for x in g.shape), "K": g.K, "batch_slots": batch,
               "workspace_GB": P.workspace_bytes(cfg, batch) / 1e9, "stage_kernel": g.stage_kernel_name(),
               "timed_sample": "%d t1 x %d t2 delays, stride 1" % (n1, n2), "sample_seconds": sec,
               "replica_steps_timed": rsteps, "ms_per_replica_step": 1e3 * sec / rsteps,
               "wall_time_s_64x256_extrapolated": sec * FULL_2D_REPLICA_STEPS / rsteps, "extrapolated": True,
               "full_protocol": "64 t1 x 256 t2 = %d replica-steps, linear in replica-steps" % FULL_2D_REPLICA_STEPS,
               "cell_updates_per_s": g.cells * rsteps / sec, "gpu_launches": int(g.launch_count() - n0),
               "finite": bool(np.all(np.isfinite(R)))}
    finally:
        g.close()
        torch.cuda.empty_cache()
    return rec


def run_2d(args):
    """Secondary metric of BASELINE.json: wall time of the 2D THz-Raman response R2(t2, t1) (configs[4]: 20^6 grid,
    64 t1 x 256 t2 delays, t1 replicas batched into HBM).  Times chfpe_response_2d end to end (replica copies, kicks,
    batched propagation, expectations, D2H of R) on a bounded sample of the delay grid and extrapolates linearly in
    replica-steps to the full grid; says so."""
    import numpy as np
    import torch
    import paper_2509_25840_b200 as P
    from paper_2509_25840_b200 import sharding
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    # the t1 rows of R2 shard over the ranks (round-robin), every rank advances its own copy of the t1
    # trajectory, one NCCL all_gather of n1 x n2 doubles at the end; --sharded runs the same path with one rank
    dist = None
    if world > 1 or args.sharded:
        import torch.distributed as dist
        if world == 1:
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29517")
            os.environ.setdefault("RANK", "0")
            os.environ.setdefault("WORLD_SIZE", "1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    herm = args.representation == "hermite"             # row f1: the same protocol on the Hermite representation (cfg4h)
    wl = args.workload if args.workload != "cfg4" else ("cfg4h" if herm else "cfg5")
    cfg = ci.config(wl, scheme=args.scheme) if herm else ci.config(wl)
    M = cfg["n_modes"]
    dev = "cuda:%d" % local
    g = P.Hermite(cfg, batch=args.batch, device=dev) if herm else P.CHFPE(cfg, batch=args.batch, device=dev)
    mu, al = obs(P, "mu", M), obs(P, "alpha", M)
    g.equilibrate(residual=False)
    n1, n2 = args.n1, args.n2
    t1, t2 = list(range(n1)), list(range(n2))
    g.response_2d(mu, al, al, t1[:2], t2[:2], cfg["dt"])            # warm-up
    g.equilibrate(residual=False)
    n0 = g.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    e0.record()
    if dist is not None:
        R = sharding.response_2d_sharded(g, mu, al, al, t1, t2, cfg["dt"], device=dev)
    else:
        R = g.response_2d(mu, al, al, t1, t2, cfg["dt"])
    e1.record()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    tms = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(tms, op=dist.ReduceOp.MAX)              # time = max over ranks
    sec = float(tms[0]) * 1e-3
    rsteps = (n1 - 1) + n1 * (n2 - 1)                               # trajectory steps + replica steps (whole job)
    full = FULL_2D_REPLICA_STEPS
    if rank != 0:
        g.close()
        if dist is not None:
            dist.destroy_process_group()
        return 0
    line = {"metric": "2D THz-Raman wall time", "value": sec * full / rsteps, "unit": "s", "higher_is_better": False,
            "n_gpus": world, "dtype": "f64", "data": "synthetic", "extrapolated": True,
            "scaling": "strong" if world > 1 else "weak",
            "parallelism": ("t1 rows round-robin over %d ranks, one NCCL all_gather of %d doubles" % (world, n1 * n2))
            if dist is not None else "single GPU",
            "config": {"workload": wl + (" chfpe_hermite_response_2d" if herm else " response_2d"),
                       "grid": "x".join(str(x) for x in g.shape), "K": g.K, "batch_slots": args.batch,
                       "workspace_GB": (P.hermite_workspace_bytes(cfg, args.batch) if herm
                                        else P.workspace_bytes(cfg, args.batch)) / 1e9,
                       "timed_sample": "%d t1 x %d t2 delays, stride 1, A=mu B=alpha C=alpha" % (n1, n2),
                       "full_protocol": "64 t1 x 256 t2 (16383 replica-steps), linear extrapolation in replica-steps"},
            "sample_seconds": sec, "replica_steps_timed": rsteps, "ms_per_replica_step": 1e3 * sec / rsteps,
            ("value_updates_per_s" if herm else "cell_updates_per_s"): (g.values if herm else g.cells) * rsteps / sec,
            "gpu_launches": int(g.launch_count() - n0), "finite": bool(np.all(np.isfinite(R)))}
    print(json.dumps(line))
    g.close()
    if dist is not None:
        dist.destroy_process_group()
    return 0


def run_slab(args):
    """Row f4: ONE propagation of --workload cut along q_1 into WORLD_SIZE slabs (sharding.SlabPropagator): every rank
    steps its slab with chfpe_rk4_stage and refreshes two halo planes per inner face of the stage input over NCCL
    point-to-point before every stage.  value = global cell-updates/s (strong scaling; time = max over ranks).  With one
    rank it measures the stage-by-stage path without exchange."""
    import torch
    import torch.distributed as dist
    import paper_2509_25840_b200 as P
    from paper_2509_25840_b200 import sharding
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world == 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29519")
        os.environ.setdefault("RANK", "0")
        os.environ.setdefault("WORLD_SIZE", "1")
    dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cfg = ci.config(args.workload)
    loc, geo = sharding.slab_config(cfg, rank, world)
    g = P.CHFPE(loc, batch=1, device="cuda:%d" % local)
    g.equilibrate(residual=False)                           # (slab-local normalisation: a timing state, not a physical one)
    g.kick(obs(P, "mu", cfg["n_modes"]))
    prop = sharding.SlabPropagator(g, geo, sharding.DistExchange())
    steps, warm = args.steps, max(args.warmup, 3)
    prop.step(warm, cfg["dt"])
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    dist.barrier(); torch.cuda.synchronize()
    e0.record()
    prop.step(steps, cfg["dt"])
    e1.record()
    dist.barrier(); torch.cuda.synchronize()
    t = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device="cuda")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms = float(t[0])
    cells = 1
    for s_ in range(cfg["n_modes"]):
        cells *= cfg["nq"][s_] * cfg["np"][s_]
    if rank == 0:
        plane = g.cells // loc["nq"][0]
        print(json.dumps({"metric": METRIC, "value": cells * steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
                          "steps": steps, "warmup": warm, "ms_per_step": ms / steps, "higher_is_better": True,
                          "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                          "config": {"workload": args.workload + " single propagation, slab-decomposed along q_1",
                                     "parallelism": "%d slabs, halo 2 planes x %d elements per inner face and stage "
                                                    "(%.0f MB), NCCL point-to-point" % (world, g.K, 2 * g.K * plane * 8 / 1e6),
                                     "local_grid": "x".join(str(x) for x in g.shape), "stage_kernel": g.stage_kernel_name()},
                          "gpu_launches": int(g.launch_count())}))
    g.close()
    dist.destroy_process_group()
    return 0


def run_2d_reference(args):
    """Reference arm of --protocol 2d: the CPU oracle's response_2d as it stands, on the 12^6 shrink of config 5's model
    (a full 20^6 replica-step takes 20 s on 16 cores), scaled by the cell count and extrapolated to 64 x 256 delays."""
    import oracle
    cfg = ci.config("cfg4s12")
    o = oracle.RefCHFPE(cfg)
    M = cfg["n_modes"]
    mu, al = obs(oracle, "mu", M), obs(oracle, "alpha", M)
    o.equilibrate()
    n1, n2 = 2, 3
    t0 = time.perf_counter()
    o.response_2d(mu, al, al, list(range(n1)), list(range(n2)), cfg["dt"])
    sec = time.perf_counter() - t0
    rsteps = (n1 - 1) + n1 * (n2 - 1)
    scale = 20.0 ** 6 / o.cells
    val = sec / rsteps * scale * FULL_2D_REPLICA_STEPS
    line = {"impl": "reference", "metric": "2D THz-Raman wall time", "value": val, "unit": "s", "higher_is_better": False,
            "n_gpus": args.gpus, "dtype": "f64", "data": "synthetic", "extrapolated": True,
            "config": {"workload": "cfg5 response_2d", "sample": "CPU oracle on the 12^6 grid of the same model, %d t1 x %d t2 "
                       "delays (%.1f s), scaled by cells (x%.1f) and to 16383 replica-steps" % (n1, n2, sec, scale)},
            "cpu_baseline": {"value": val, "unit": "s", "cores": oracle.set_threads(0), "kind": "oracle",
                             "sample": "12^6 proxy, scaled", "nproc": os.cpu_count(), "cpu_model": cpu_model()},
            "e2e": {"value": val, "unit": "s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    o.close()
    print(json.dumps(line))
    return 0


def run_3d(args):
    """Row f2: third-order response R3(t3, t2, t1) of Eq. (17) at one waiting time t2 -- the scan behind
    the 2D IR spectrum of Eq. (21) -- on config 4's model.  Times chfpe_response_3d end to end (trajectory, replica
    copies, three kicks, batched propagation of batch-1 replicas, expectations, D2H of R) on an n1 x 1 x n2 sample
    of delays (--n2 is the number of t3 delays here) and reports replica-steps per second; not a BASELINE metric."""
    import numpy as np
    import torch
    import paper_2509_25840_b200 as P
    herm = args.representation == "hermite"             # row f1: chfpe_hermite_response_3d on cfg4h
    wl = args.workload if not (herm and args.workload == "cfg4") else "cfg4h"
    cfg = ci.config(wl, scheme=args.scheme) if herm else ci.config(wl)
    M = cfg["n_modes"]
    g = P.Hermite(cfg, batch=args.batch) if herm else P.CHFPE(cfg, batch=args.batch)
    mu = obs(P, "mu_nl", M)
    g.equilibrate(residual=False)
    n1, n3, wait = args.n1, args.n2, 4
    t1, t3 = list(range(n1)), list(range(n3))
    g.response_3d(mu, mu, mu, mu, t1[:2], [wait], t3[:2], cfg["dt"])   # warm-up
    g.equilibrate(residual=False)
    n0 = g.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    R = g.response_3d(mu, mu, mu, mu, t1, [wait], t3, cfg["dt"])
    e1.record()
    torch.cuda.synchronize()
    sec = e0.elapsed_time(e1) * 1e-3
    rsteps = (n1 - 1) + n1 * wait + n1 * (n3 - 1)                   # t1 trajectory + waiting time + t3 scans
    line = {"metric": "third-order response replica-steps/s", "value": rsteps / sec, "unit": "replica-steps/s",
            "higher_is_better": True, "n_gpus": 1, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl + " response_3d", "grid": "x".join(str(x) for x in g.shape), "K": g.K,
                       "batch_slots": args.batch,
                       "workspace_GB": (P.hermite_workspace_bytes(cfg, args.batch) if herm
                                        else P.workspace_bytes(cfg, args.batch)) / 1e9,
                       "timed_sample": "%d t1 x 1 t2 (%d steps) x %d t3 delays, stride 1, A=B=C=D=mu (nonlinear)"
                                       % (n1, wait, n3)},
            "sample_seconds": sec, "replica_steps_timed": rsteps, "ms_per_replica_step": 1e3 * sec / rsteps,
            ("value_updates_per_s" if herm else "cell_updates_per_s"): (g.values if herm else g.cells) * rsteps / sec,
            "gpu_launches": int(g.launch_count() - n0), "finite": bool(np.all(np.isfinite(R)))}
    print(json.dumps(line))
    g.close()
    return 0


def run_hermite(args):
    """Row f1: the Hermite-in-momentum representation (the paper's production scheme, Eq. 22-23 and A1-A4)
    on config 4's model: 32^3 q mesh x 8^3 Hermite functions x 20 elements = 3.36e8 values (the value count of
    config 4).  A step = one RK4 step of the whole hierarchy (4 launches of k_hermite_stage) + <mu>.  Not a BASELINE
    metric (there are no phase-space cells here): value-updates/s, with the same roofline accounting as the grid
    path (22 compulsory bytes per value per launch)."""
    import numpy as np
    import torch
    import paper_2509_25840_b200 as P
    wl = args.workload if args.workload != "cfg4" else "cfg4h"
    cfg = ci.config(wl, scheme=args.scheme)
    M = cfg["n_modes"]
    g = P.Hermite(cfg, batch=1)
    # launches per RK stage: 1 (explicit stencils) | 2 (COMPACT6, march kernel + q_1 line pass) | 1 + M (COMPACT6 otherwise)
    per_stage = {"compact": 1 + M, "compact_tma": 2}.get(g.stage_kernel(), 1)
    mu = obs(P, "mu", M)
    dt = cfg["dt"]
    steps, warm = args.steps, max(args.warmup, 3)
    g.equilibrate(residual=False)
    g.kick(mu)
    g.response_1d(None, mu, warm + 1, 1, dt)
    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.3)
    n0 = g.launch_count()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    torch.cuda.synchronize()
    ev[0].record()
    R = g.response_1d(None, mu, steps + 1, 1, dt)
    ev[1].record()
    torch.cuda.synchronize()
    launches = g.launch_count() - n0
    ev[2].record()
    g.step(steps, dt)                                    # stage kernels only: 4 * steps launches
    ev[3].record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms, ms_stage = ev[0].elapsed_time(ev[1]), ev[2].elapsed_time(ev[3])
    if not np.all(np.isfinite(R)):
        raise SystemExit("bench.py: non-finite response")
    X0 = torch.from_numpy(g.export_state()).pin_memory()
    e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e2.record()
    g.import_state(X0.numpy())
    g.response_1d(None, mu, steps + 1, 1, dt)
    e3.record()
    torch.cuda.synchronize()
    ms_e2e = e2.elapsed_time(e3)
    peak, peak_src = measured_peaks()
    values = g.values
    kern_ms = ms_stage / (4 * steps)                     # one RK stage (per_stage launches)
    achieved = values * 22.0 / (kern_ms * 1e-3) / 1e9
    kname = g.stage_kernel_name()
    line = {"metric": "Hermite-representation value-updates/s (fp64)", "value": values * steps / (ms * 1e-3),
            "unit": "value-updates/s", "n_gpus": 1, "steps": steps, "warmup": warm, "ms_per_step": ms / steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl + " (Hermite representation, row f1)", "modes": M,
                       "shape": "x".join(str(x) for x in g.shape), "values": values, "depth": cfg["depth"], "dt": dt,
                       "scheme": cfg["scheme"], "integrator": "RK4 (Horner form)",
                       "l2": "inputs larger than L2 (state array %.1f GB vs 126 MB)" % (values * 8 / 1e9)},
            "e2e": {"value": values * steps / (ms_e2e * 1e-3), "unit": "value-updates/s",
                    "h2d_bytes_per_step": values * 8.0 / steps, "d2h_bytes_per_step": 8.0 * (steps + 1) / steps},
            "gpu_launches": int(launches), "clocks": clocks,
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": profiled_traffic("r*_hermite_stage_ncu_full.txt", "dram_bytes_per_launch_hermite")
                         if (wl == "cfg4h" and per_stage == 1) else None, "peak_source": peak_src, "kernel": kname, "kernel_ms": kern_ms,
                         "kernel_launches_timed": 4 * steps * per_stage,
                         "kernel_share_of_step": min(1.0, 4 * kern_ms / (ms / steps)),
                         "algorithmic_bytes_per_launch": values * 22.0}}
    if not args.no_cpu:
        from oracle import hermite
        sub = ci.config(wl, nq=[12] * M, scheme=args.scheme) if M == 3 else cfg
        o = hermite.RefHermite(sub)
        o.equilibrate()
        d = ci.observable("mu", M)
        o.kick(d)
        t0 = time.perf_counter()
        o.step(1, dt); o.expect(d)
        tc = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": float(np.prod(o.shape)) / tc, "unit": "value-updates/s",
                                "cores": os.cpu_count(), "kind": "oracle",
                                "sample": "oracle/hermite.py (numpy) on %s with a %s q mesh, 1 RK4 step + <mu> (%.1f s)"
                                          % (wl, "x".join(str(x) for x in o.nq), tc)}
    print(json.dumps(line))
    g.close()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg (profiling runs)")
    ap.add_argument("--no-2d", action="store_true", help="skip the two_d sub-record (config 5, 154 GB of device memory)")
    ap.add_argument("--sharded", action="store_true",
                    help="--protocol 2d: go through sharding.response_2d_sharded + NCCL even with one rank")
    ap.add_argument("--protocol", default="step", choices=["step", "2d", "3d", "slab"],
                    help="'2d': time chfpe_response_2d on config 5 (secondary metric: 2D THz-Raman wall time); "
                         "'3d': time chfpe_response_3d (row f2) on --workload")
    ap.add_argument("--representation", default="grid", choices=["grid", "hermite"],
                    help="'hermite': row f1, the Hermite-in-momentum representation on cfg4h (not a BASELINE metric)")
    ap.add_argument("--scheme", default="central4", choices=["central4", "central2", "compact6"],
                    help="derivative scheme (compact6 = the paper's Pade scheme, step a9 / row f1)")
    ap.add_argument("--batch", type=int, default=5, help="replica slots for --protocol 2d (trajectory + t1 replicas)")
    ap.add_argument("--n1", type=int, default=8)
    ap.add_argument("--n2", type=int, default=16)
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.protocol == "2d":
        return run_2d(args)
    if args.protocol == "slab":
        return run_slab(args)
    if args.protocol == "3d":
        return run_3d(args)
    if args.representation == "hermite":
        return run_hermite(args)
    if args.protocol == "3d":
        return run_3d(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
