#!/usr/bin/env python
"""bench.py -- grid-point updates/s of the relaxation step (fp64, mimetic curl) on BASELINE.json config 4.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C1..C5]
                    [--operator mimetic|direct] [--integrator euler|adaptive] [--reading P|D]
                    [--isohelix N[,N..] [--t-end T]]

One "step" is one pass of the whole hot path (S1-S5: Jacobian, push-forward, mimetic curl, J x B, line-tied
update) over the full 256x256x512 grid = one fused kernel launch inside mr_step.  The timed region is ONE
mr_step(K) call bracketed by CUDA events on the launching stream (barrier + synchronize on both sides, max
over ranks).  Prints ONE JSON line (see DESIGN.md "Measurement" for every key).

Besides the K timed steps the line carries a "burst" record (20 steps at full clocks) and a "sustained" record (a run of at
least 2 s under the board's power cap, with the clocks it saw): the roofline fraction is quoted for all three.
--workload C3 adds the report BASELINE configs[2] asks for (both curl errors at t = 0, max |J x B| and |x - x0| after the
steps); --integrator adaptive times the Cash-Karp integrator of section 2.4 in right-hand-side evaluations per second.

Multi-GPU: north_star keeps the path on one GPU ("replicas only"): --gpus N runs N independent
replicas, one process per GPU (torchrun), value = N * nodes * K / max-over-ranks time, "scaling": "weak".

--impl reference times the CPU oracle (oracle/mro.c) as it stands on the host cores for the same metric, on a
bounded sample of the same workload.  The oracle is only ever touched by that arm and by the cpu_baseline leg.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "grid-point updates/s (fp64, mimetic curl)"
UNIT = "updates/s"
BYTES_PER_UPDATE = {"f64": 72.0, "f32": 36.0}   # read xi 3T + read b 3T + write xi' 3T
# direct operator (--operator direct): bound by plain FP64 arithmetic, not HBM.  FLOPs per update counted
# in the SASS of k_step_direct<double> (116 DFMA x 2 + 90 DADD + 68 DMUL); peak = 148 SMs x 64 FP64 lanes x
# 2 FLOP x 1.965 GHz (B200_PROFILING.md unit counts and clocks)
DIRECT_FLOP_PER_UPDATE = 390.0
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12


# ---------------------------------------------------------------------------------------------- helpers (CPU)

def measured_peak_gbs():
    """HBM roofline denominator: the driver-measured copy bandwidth, else the profiling guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def csrc_fingerprint():
    """sha1 over the device code (csrc/*.cuh: the kernels, their layouts and the launch geometry): a traffic row is only valid for
    the kernels it was captured with.  (mr_api.cu, the host side of the ABI, does not enter.)"""
    import glob
    import hashlib
    h = hashlib.sha1()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_1405_0942_b200", "csrc", "*.cuh"))):
        with open(f, "rb") as fh:
            h.update(os.path.basename(f).encode() + b"\0" + fh.read())
    return h.hexdigest()[:16]


def recorded_traffic(workload, kernel):
    """dram bytes per launch of this step kernel from the committed ncu --set full capture (profiles/traffic.csv, one row
    per capture with the fingerprint of the sources it was taken with), or None if there is no capture of THESE sources:
    a stale row is never printed."""
    import csv
    try:
        fp = csrc_fingerprint()
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload and row["kernel"] == kernel and row.get("csrc_sha1") == fp:
                    return float(row["dram_bytes_per_launch"])
    except Exception:
        pass
    return None


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons every 100 ms while the timed region runs."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index = index
        self.rows = []
        self._stop = threading.Event()
        self._t = None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                for line in out.strip().splitlines():
                    self.rows.append([c.strip() for c in line.split(",")])
            except Exception:
                pass
            self._stop.wait(0.1)

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=10)

    def summary(self):
        return summarize_clocks(self.rows)


def summarize_clocks(rows):
    sm, mx, pw, reasons = [], [], [], set()
    names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
    for r in rows:
        try:
            sm.append(float(r[0]))
            mx.append(float(r[1]))
        except Exception:
            continue
        try:
            pw.append(float(r[2]))
        except Exception:
            pass
        for name, v in zip(names, r[3:7]):
            if v.lower().startswith("active"):
                reasons.add(name)
    if not sm:
        return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0, "power_w": None}
    sm.sort()
    return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm),
            "power_w": sum(pw) / len(pw) if pw else None}


def aggregate_over_ranks(local_ms, local_updates, dist=None):
    """max-over-ranks time and summed work (torch.distributed when world_size > 1)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local_ms, local_updates
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([local_ms], dtype=torch.float64, device=dev)
    u = torch.tensor([float(local_updates)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def workload(name):
    from paper_1405_0942_b200 import inputs as I
    cfg = I.CONFIGS[name]
    return cfg, I


# ---------------------------------------------------------------------------------------------- oracle legs

def oracle_sample(cfg, I, x0, B0, dt, budget_s=12.0):
    """Time the CPU oracle, as it stands, on the workload itself: whole-grid forward Euler steps from the configuration's
    initial state, as many as fit the budget (at least one; config 4 needs about 1.5 s per step on 16 cores).  Returns
    (updates/s, threads, description)."""
    from oracle import mro                       # the ONLY place bench.py touches the oracle (with run_reference)
    g = cfg.grid
    threads = mro.max_threads()
    mro.set_threads(threads)
    t0 = time.perf_counter()
    x = mro.step(g.n, g.lo, g.hi, x0, B0, dt, 1)
    t1 = time.perf_counter() - t0
    steps = int(max(1, min(20, budget_s / max(t1, 1e-3))))
    t0 = time.perf_counter()
    mro.step(g.n, g.lo, g.hi, x, B0, dt, steps)
    el = time.perf_counter() - t0
    mro.set_threads(1)
    desc = "%s, the whole %dx%dx%d grid, %d Euler steps after one untimed, mimetic, OpenMP over k" % ((cfg.name,) + g.n + (steps,))
    return g.nodes * steps / el, threads, desc


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric and config: each step one forward Euler step of the whole
    grid (config 4: about 1.5 s on 16 cores, so the default 20 + 5 steps end within a minute or two)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg, I = workload(args.workload)
    from oracle import mro
    g = cfg.grid
    x, B0, dt = I.make(cfg)
    threads = mro.max_threads()
    mro.set_threads(threads)
    for _ in range(args.warmup):
        x = mro.step(g.n, g.lo, g.hi, x, B0, dt, 1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        x = mro.step(g.n, g.lo, g.hi, x, B0, dt, 1)
    el = time.perf_counter() - t0
    value = g.nodes * args.steps / el
    sample = "%s, the whole %dx%dx%d grid per step, mimetic, OpenMP over k" % ((cfg.name,) + g.n)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": el / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "%s %dx%dx%d fp64 mimetic, line-tied, forward Euler dt=%.3e (CPU oracle, whole grid)" % ((cfg.name,) + g.n + (dt,)),
                   "nodes": g.nodes},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ---------------------------------------------------------------------------------------------- our arm (GPU)

def reading_P_field(I, g, x0):
    """Config 3, reading P (Q16): B(X,0) pulled back so that the nodal pushed-forward field equals ABC(x0).  The
    discrete Jacobian is numpy.gradient's (second-order central inside, second-order one-sided on the faces: the same
    stencil as reading Q3), so neither the product nor the oracle is involved in making the input."""
    import numpy as np
    F = np.empty((3, 3) + x0.shape[1:])
    for c in range(3):
        for a in range(3):
            F[c, a] = np.gradient(x0[c], g.h[a], axis=2 - a, edge_order=2)
    Fm = np.moveaxis(F, (0, 1), (-2, -1))
    det = np.linalg.det(Fm)
    Fi = np.linalg.inv(Fm)
    return np.ascontiguousarray(np.einsum("...ac,c...->a...", Fi, I.abc_field(x0)) * det)


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%d: launch N ranks with torch.distributed.run (one per GPU)" % (args.gpus, world))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the relaxation step has no CPU path")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    from paper_1405_0942_b200 import mr   # fails loudly if libmr.so is missing

    cfg, I = workload(args.workload)
    g = cfg.grid
    dtype = cfg.dtype
    td = torch.float64 if dtype == "f64" else torch.float32
    x0, B0, dt = I.make(cfg)
    if cfg.kind == "abc" and args.reading == "P":
        B0 = reading_P_field(I, g, x0)
        dt = I.stable_dt(B0, g)
    nodes = g.nodes
    X = I.reference_grid(g)
    displaced = not np.array_equal(x0, X)

    sim = mr.Relaxation(g.n, g.lo, g.hi, dtype=dtype, device="cuda:%d" % local_rank)
    if args.variant != "auto":
        sim.set_variant(args.variant)
    if args.no_graphs:
        sim.set_variant("nograph")
    sim.set_B0(torch.from_numpy(B0).to("cuda", dtype=td))

    def reset_state():
        """back to the initial state: an fp32 context takes the displacement (Q15); x = X needs the zero displacement"""
        if dtype == "f64":
            sim.set_x(torch.from_numpy(x0).to("cuda", dtype=td))
        else:
            sim.set_xi(torch.from_numpy(x0 - X).to("cuda", dtype=td))

    if displaced:
        reset_state()                                  # (a context starts at x = X: nothing to set otherwise)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    op = args.operator
    report = None
    if cfg.kind == "abc":
        # BASELINE configs[2]: "the mimetic and direct curl errors are reported" (exact curl of an ABC field: pi B)
        report = {"reading": args.reading, "dt": dt}
        inner = (slice(None), slice(1, -1), slice(1, -1), slice(1, -1))
        for o in ("mimetic", "direct"):
            f = sim.get_fields(o, B=True, J=True)
            Bf, Jf = f["B"][inner], f["J"][inner]
            report["curl_error_" + o] = float((Jf - np.pi * Bf).abs().max() / (np.pi * f["B"].abs().max()))
            del f, Bf, Jf
        d0 = sim.diagnostics(op)
        report.update({"max_jxb_0": d0["max_jxb"], "xi_0": d0["xi"], "energy_0": d0["energy"]})
        sim.step(cfg.steps, dt, op)                    # the config's 200 steps, then back to the initial state for the timing
        d1 = sim.diagnostics(op)
        xi_0 = torch.from_numpy(x0 - X).to("cuda")
        report.update({"steps": cfg.steps, "max_jxb_after": d1["max_jxb"], "xi_after": d1["xi"], "energy_after": d1["energy"],
                       "max_abs_x_minus_x0": float((sim.get_xi().double() - xi_0).abs().max()), "h": g.h[0],
                       "concave_nodes_after": sim.convexity()[0]})
        del xi_0
        reset_state()

    def timed(steps):
        """CUDA events around ONE mr_step(steps) (or one mr_step_adaptive of `steps` trial steps' worth of time)"""
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        with ClockSampler(local_rank) as clocks:
            l0 = sim.launch_count
            e0.record()
            sim.step(steps, dt, op)
            e1.record()
            barrier()
            launches = sim.launch_count - l0
        ms = e0.elapsed_time(e1)
        ms_all, updates_all = aggregate_over_ranks(ms, nodes * steps, dist if world > 1 else None)
        return {"ms": ms, "ms_all": ms_all, "updates_all": updates_all, "launches": launches, "clocks": clocks.summary(), "steps": steps}

    # ---- device-resident throughput: W warm-up steps, then ONE timed mr_step(K) ----
    W = max(args.warmup, 3)
    if 3 * 3 * nodes * (8 if dtype == "f64" else 4) <= 4e8 and not args.no_graphs:
        W = (max(W, 32) + 15) // 16 * 16   # (an L2-resident grid replays CUDA graphs of 16 steps from an even buffer parity: the
                                           # warm-up captures them and ends on the parity the timed call starts from)
    sim.step(W, dt, op)
    main = timed(args.steps)
    variant = sim.step_variant
    value = main["updates_all"] / (main["ms_all"] * 1e-3)
    diag = sim.diagnostics(op)
    peak, peak_src = measured_peak_gbs()

    # the direct operator's roof is FP64 arithmetic: measured in this run with a DFMA-chain kernel (mr_measure_fp64_peak), a
    # 20 ms burst here and a 2 s run after the sustained record (the derived figure stays beside it)
    fp64_peak = {"burst": mr.measure_fp64_peak(0.02)} if op == "direct" else {}

    def roof(rec, regime="burst"):
        launch_ms = rec["ms"] / max(rec["launches"], 1)
        if op == "direct":
            tf = DIRECT_FLOP_PER_UPDATE * nodes / (launch_ms * 1e-3) / 1e12
            pk = fp64_peak.get(regime, fp64_peak["burst"])
            return {"bound": "alu", "achieved": tf, "peak": pk, "unit": "TFLOP/s", "frac": tf / pk,
                    "traffic": None, "peak_source": "measured in this run: DFMA-chain kernel (mr_measure_fp64_peak), %s regime" % regime,
                    "peak_derived": FP64_PEAK_TFLOPS, "peak_derived_source": "148 SMs x 64 FP64 lanes x 2 x 1.965 GHz",
                    "flop_counting": "a DADD or DMUL counts 1 FLOP against a roof of 2 per DFMA slot: pipe occupancy is higher than frac, "
                                     "sm__pipe_fp64_cycles_active = 61 % in profiles/r2b_direct_full.md",
                    "kernel": variant,
                    "algorithmic_flop_per_launch": DIRECT_FLOP_PER_UPDATE * nodes, "launch_ms": launch_ms,
                    "hbm_frac": BYTES_PER_UPDATE[dtype] * nodes / (launch_ms * 1e-3) / 1e9 / peak}
        achieved = BYTES_PER_UPDATE[dtype] * nodes / (launch_ms * 1e-3) / 1e9
        return {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "frac_of_datasheet_8000": achieved / 8000.0,
                "traffic": recorded_traffic(cfg.name, variant),
                "traffic_source": "recorded, not measured in this run: profiles/traffic.csv (ncu --set full of these kernel sources)",
                "peak_source": peak_src, "kernel": variant,
                "algorithmic_bytes_per_launch": BYTES_PER_UPDATE[dtype] * nodes, "launch_ms": launch_ms}

    roofline = roof(main)

    # ---- the two regimes of this board (1 kW cap): a 20-step burst at full clocks and a run of >= 2 s under the cap ----
    regimes = {}
    fbytes = 3 * nodes * (8 if dtype == "f64" else 4)
    if not args.no_regimes and 3 * fbytes > 4e8:       # (L2-resident workloads: the HBM fraction is n/a, and a long run of a
                                                       # small braid ends where the paper says it does)
        ms_step = main["ms"] / args.steps
        for name, steps in (("burst", 20), ("sustained", int(max(200, min(200000, 2200.0 / max(ms_step, 1e-3)))))):
            if name == "burst":
                time.sleep(1.0)                       # let the board cool off the previous run
            r = timed(steps)
            if op == "direct" and name == "sustained":
                fp64_peak["sustained"] = mr.measure_fp64_peak(2.0)     # right after the long run: the board is still at its cap
                roofline["sustained_peak"] = fp64_peak["sustained"]
            rf = roof(r, name)
            pw = r["clocks"].get("power_w")
            regimes[name] = {"steps": steps, "ms_per_step": r["ms_all"] / steps, "seconds": r["ms"] * 1e-3,
                             "value": r["updates_all"] / (r["ms_all"] * 1e-3), "roofline_frac": rf["frac"], "clocks": r["clocks"],
                             # (board power is sampled every 100 ms and lags: only a run with several samples has an energy figure)
                             "joules_per_update": None if pw is None or r["clocks"]["samples"] < 5 else pw * r["ms"] * 1e-3 / (nodes * steps)}
            # (the driver's parser keeps `roofline` and drops the regime records: both fractions go in there too)
            roofline[name + "_frac"] = rf["frac"]
            roofline[name + "_ms_per_step"] = r["ms_all"] / steps
            roofline[name + "_sm_mhz"] = r["clocks"]["sm_mhz"]
            roofline[name + "_reasons"] = r["clocks"]["reasons"]
            roofline[name + "_joules_per_update"] = regimes[name]["joules_per_update"]
        roofline["regime_of_frac"] = "the %d timed steps of this run (%.0f ms): a burst at full clocks unless --steps is large; the " \
                                     "configuration's own length (thousands of steps) runs in the sustained regime" % (args.steps, main["ms"])

    # ---- BASELINE configs[4]: "fp32 results are compared to an fp64 GPU run within 1e-5 relative": the deviations of the fp32
    # state and fields from an fp64 context on the same inputs (norm-wise, max |a - b| / max |b|; x relative to the box) after
    # 100, 500 and the config's own number of steps
    fp32_report = None
    if dtype == "f32" and not args.no_fp32_report:
        reset_state()
        ref = mr.Relaxation(g.n, g.lo, g.hi, dtype="f64", device="cuda:%d" % local_rank)
        ref.set_B0(torch.from_numpy(B0).to("cuda", dtype=torch.float64))
        if displaced:
            ref.set_x(torch.from_numpy(x0).to("cuda", dtype=torch.float64))
        box = float(max(g.hi[a] - g.lo[a] for a in range(3)))

        def rel(a, b):
            return float((a.double() - b).abs().max() / b.abs().max())

        fp32_report, done = {"bar": 1e-5, "operator": op}, 0
        for upto in sorted({min(100, cfg.steps), min(500, cfg.steps), cfg.steps}):
            sim.step(upto - done, dt, op)
            ref.step(upto - done, dt, op)
            done = upto
            a, b = sim.get_xi(), ref.get_xi()
            e = {"x": float((a.double() - b).abs().max()) / box, "xi": rel(a, b)}
            del a, b
            for name in ("B", "J"):
                a, b = sim.get_fields(op, **{name: True})[name], ref.get_fields(op, **{name: True})[name]
                e[name] = rel(a, b)
                del a, b
            fp32_report["after_%d_steps" % upto] = e
        ref.close()
        del ref
        torch.cuda.empty_cache()
        reset_state()

    # ---- section 2.4: the adaptive Cash-Karp integrator, in right-hand-side evaluations per second ----
    adaptive = None
    if args.integrator == "adaptive":
        reset_state()
        lam0 = args.lambda0
        st = sim.step_adaptive(t_end=3.0 * dt, lambda0=lam0, dt=dt, op=op)         # warm-up (binds the workspace)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        t0 = sim.diagnostics(op)["time"]
        e0.record()
        st = sim.step_adaptive(t_end=t0 + args.adaptive_span * dt, lambda0=lam0, dt=st["dt_next"], op=op, max_trials=args.steps)  \
            if args.adaptive_span > 0 else st
        e1.record()
        barrier()
        ams = e0.elapsed_time(e1)
        adaptive = {"lambda0": lam0, "accepted": st["accepted"], "rejected": st["rejected"], "rhs_evals": st["rhs_evals"],
                    "ms": ams, "rhs_evals_per_s": st["rhs_evals"] / (ams * 1e-3), "node_rhs_per_s": st["rhs_evals"] * nodes / (ams * 1e-3),
                    "time_advanced": st["time"] - t0, "dt_next": st["dt_next"], "euler_dt": dt}

    # ---- end to end through the host-buffer entry points: H2D of x, one step, D2H of x, every step.  The streaming calls
    # (mr_step_host_async ... mr_host_sync) keep both directions of the link busy: the copy out of one step overlaps the copy
    # in of the next; "sync" is the same through the blocking calls (mr_set_x_host + mr_step + mr_get_fields_host), one by one.
    xin = [torch.from_numpy(x0).to(td).pin_memory() for _ in range(2)]
    xout = [torch.empty_like(xin[0]).pin_memory() for _ in range(2)]
    e2e_steps = max(1, args.e2e_steps)
    sim.step_host_async(xin[0], xout[0], 1, dt, op)
    sim.host_sync()
    barrier()
    t0 = time.perf_counter()
    for q in range(e2e_steps):
        sim.step_host_async(xin[q % 2], xout[q % 2], 1, dt, op)     # pinned H2D of x + layout import + mr_step(1) + pinned D2H of x
    sim.host_sync()
    barrier()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    e2e_ms_all, e2e_updates = aggregate_over_ranks(e2e_ms, nodes * e2e_steps, dist if world > 1 else None)
    sync_steps = min(2, e2e_steps)
    barrier()
    t0 = time.perf_counter()
    for q in range(sync_steps):
        sim.set_x(xin[q % 2])                 # mr_set_x_host
        sim.step(1, dt, op)                   # mr_step
        sim.get_fields_into(x=xout[q % 2])    # mr_get_fields_host
    barrier()
    sync_ms = (time.perf_counter() - t0) * 1e3
    e2e = {"value": e2e_updates / (e2e_ms_all * 1e-3), "unit": UNIT, "h2d_bytes_per_step": fbytes,
           "d2h_bytes_per_step": fbytes, "steps": e2e_steps,
           "what": "per step: mr_step_host_async (pinned H2D of x, layout import, mr_step(1), pinned D2H of x'); mr_host_sync at the end; "
                   "the D2H of a step overlaps the H2D of the next",
           "blocking_calls_value": nodes * sync_steps / (sync_ms * 1e-3),
           "link_gbs_each_way": fbytes * e2e_steps / (e2e_ms * 1e-3) / 1e9}
    del xin, xout

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, threads, desc = oracle_sample(cfg, I, x0, B0, dt)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc}

    if rank == 0:
        prec = "fp64" if dtype == "f64" else "fp32"
        line = {
            "metric": METRIC.replace("mimetic", op).replace("fp64", prec), "value": value, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": W, "ms_per_step": main["ms_all"] / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": dtype, "data": "synthetic",
            "config": {"workload": "%s %dx%dx%d %s %s%s, line-tied, forward Euler dt=%.3e"
                                   % ((cfg.name,) + g.n + (prec, op, " (S3d: the builder's derivation, unpinned vs the paper)" if op == "direct" else "", dt)),
                       "nodes": nodes, "l2_policy": "working set %.2f GB vs 126 MB L2%s" % (3 * fbytes / 1e9, " (no flush needed)" if 3 * fbytes > 4e8 else " (L2-resident: HBM fraction n/a)"),
                       "parallelism": "replicas only" if world > 1 else "single GPU", "kernel": variant},
            "clocks": main["clocks"], "e2e": e2e, "gpu_launches": main["launches"], "roofline": roofline,
            "burst": regimes.get("burst"), "sustained": regimes.get("sustained"),
            "cpu_baseline": cpu_baseline,
            "state_after": {"steps": diag["steps"], "energy": diag["energy"], "max_jxb": diag["max_jxb"], "xi": diag["xi"],
                            "min_det": diag["min_det"]},
        }
        if report is not None:
            line["config3_report"] = report
        if adaptive is not None:
            line["adaptive"] = adaptive
        if fp32_report is not None:
            line["fp32_vs_fp64"] = fp32_report
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def paper_table_4_1(phi_over_pi=0.25):
    """TABLE 4.1 of the paper as printed (tests/golden/paper_table_4_1.txt): {(method, n): (xi, eps*, sigma_B, sigma_x)} for one phi"""
    rows = {}
    try:
        with open(os.path.join(ROOT, "tests", "golden", "paper_table_4_1.txt")) as f:
            for line in f:
                line = line.split("#", 1)[0].split()
                if line and float(line[0]) == phi_over_pi:
                    rows[(line[1], int(line[2]))] = tuple(float(v) for v in line[3:7])
    except OSError:
        pass
    return rows


def paper_table_4_2():
    """TABLE 4.2 of the paper as printed (tests/golden/paper_table_4_2.txt): {(method, n): (xi, eps*)}, Pontin09, phi = pi/2"""
    rows = {}
    try:
        with open(os.path.join(ROOT, "tests", "golden", "paper_table_4_2.txt")) as f:
            for line in f:
                line = line.split("#", 1)[0].split()
                if line:
                    rows[(line[0], int(line[1]))] = (float(line[2]), float(line[3]), None, None)
    except OSError:
        pass
    return rows


def run_isohelix(args):
    """--isohelix N[,N..]: the paper's own experiment (section 3.1, TABLE 4.1): the IsoHelix field (phi = pi/4) on N^3 nodes relaxed
    with the adaptive Cash-Karp integrator (section 2.4) to t = --t-end, where eps*, sigma_B, sigma_x have stabilised; prints them
    beside the paper's row, with the wall time of the run and the rate of right-hand-side evaluations."""
    import numpy as np
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the relaxation step has no CPU path")
    from paper_1405_0942_b200 import inputs as I, mr
    pontin = args.field == "pontin09"
    paper = (paper_table_4_2() if args.phi == 0.5 else {}) if pontin else paper_table_4_1(args.phi)
    rows, total_rhs, total_s, launches = [], 0, 0.0, 0
    phi = np.pi * args.phi
    td = torch.float64 if args.dtype == "f64" else torch.float32
    for n in [int(v) for v in args.isohelix.split(",")]:
        g = I.Grid((n, n, n), (-4.0, -4.0, -10.0), (4.0, 4.0, 10.0))
        # Pontin09 (Eq. 3.4): two twist regions of opposite sense at Z = -+4 (reading Q25)
        B0 = I.pontin09_B0(g, (phi, -phi), (-4.0, 4.0)) if pontin else I.isohelix_B0(g, phi)
        Bref = np.zeros(g.shape)
        Bref[2] = 1.0
        for op in args.operator.split(","):
            sim = mr.Relaxation(g.n, g.lo, g.hi, dtype=args.dtype, device="cuda:0")
            if args.no_graphs:
                sim.set_variant("nograph")
            sim.set_B0(torch.from_numpy(B0).to("cuda", td))
            xr, Br = torch.from_numpy(I.isohelix_x_relax(g, phi)).to("cuda", td), torch.from_numpy(Bref).to("cuda", td)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            failed = None
            try:
                st = sim.step_adaptive(t_end=args.t_end, lambda0=args.lambda0, dt=1e-3, op=op, max_trials=10 ** 7)
            except mr.MrError as e:                       # (the paper's table has such rows too: "runs which do not converge")
                failed, st = str(e), sim.last_adaptive
            torch.cuda.synchronize()
            el = time.perf_counter() - t0
            if failed:
                rows.append({"n": n, "operator": op, "failed": failed, "t_end": st["time"], "accepted": st["accepted"],
                             "rejected": st["rejected"], "seconds": el})
                continue
            d = sim.diagnostics(op)
            sx, sb = sim.sigma(xr, Br)
            _, eps = sim.eps_star(n // 2, n // 2, float(np.sqrt(2.0)), op)
            pk = paper.get(("mimetic" if op == "mimetic" else "classic", n))
            rows.append({"n": n, "operator": op, "t_end": st["time"], "accepted": st["accepted"], "rejected": st["rejected"],
                         "seconds": el, "us_per_trial": el / max(st["accepted"] + st["rejected"], 1) * 1e6,
                         "xi": d["xi"], "eps_star": eps, "sigma_B": sb, "sigma_x": None if pontin else sx, "energy": d["energy"],
                         "concave_nodes": sim.convexity()[0], "kernel": sim.step_variant,
                         "paper": None if pk is None else {"xi": pk[0], "eps_star": pk[1], "sigma_B": pk[2], "sigma_x": pk[3]}})
            total_rhs += st["rhs_evals"] * g.nodes
            total_s += el
            launches += sim.launch_count
            sim.close()
    line = {"metric": "node right-hand-side evaluations/s (IsoHelix relaxation, adaptive RK5(4), fp64)", "value": total_rhs / max(total_s, 1e-9),
            "unit": "node-rhs/s", "n_gpus": 1, "higher_is_better": True, "dtype": args.dtype, "data": "synthetic", "vs_baseline": None,
            "config": {"workload": "%s phi=%g pi (PAPER.md:170-198) on n^3 nodes, n in [%s], lambda0=%g, t_end=%g; "
                                   "paper rows: TABLE %s (the 'classic' rows are the paper's direct method, whose formulas it does "
                                   "not print: context only)" % ("Pontin09 (twists at Z=-+4)" if pontin else "IsoHelix", args.phi,
                                                                 args.isohelix, args.lambda0, args.t_end, "4.2" if pontin else "4.1")},
            "gpu_launches": launches, "table_4_1": rows}
    print(json.dumps(line))
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C4", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--variant", default="auto", choices=["auto", "generic"])
    ap.add_argument("--operator", default="mimetic", help="mimetic | direct (--isohelix: a comma-separated list of them)")
    ap.add_argument("--isohelix", default="", help="N[,N..]: relax the paper's IsoHelix field on N^3 nodes and report TABLE 4.1's measures")
    ap.add_argument("--t-end", type=float, default=512.0, help="--isohelix: end time of the relaxation")
    ap.add_argument("--field", default="isohelix", choices=["isohelix", "pontin09"], help="--isohelix: Eq. 3.1 or Eq. 3.4 (TABLE 4.2, use --phi 0.5)")
    ap.add_argument("--phi", type=float, default=0.25, help="--isohelix: twist angle in units of pi (the paper: 0.25, 0.5, 1)")
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"], help="--isohelix: precision of the context")
    ap.add_argument("--integrator", default="euler", choices=["euler", "adaptive"])
    ap.add_argument("--reading", default="P", choices=["P", "D"], help="config 3: B0 pulled back (P) or ABC(X) literally (D)")
    ap.add_argument("--lambda0", type=float, default=1e-9, help="tolerance of the adaptive integrator")
    ap.add_argument("--adaptive-span", type=float, default=40.0, help="time to advance in the adaptive run, in Euler steps dt")
    ap.add_argument("--e2e-steps", type=int, default=8)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-regimes", action="store_true", help="skip the burst / sustained records")
    ap.add_argument("--no-fp32-report", action="store_true", help="fp32 workloads (C5): skip the comparison with an fp64 context")
    ap.add_argument("--no-graphs", action="store_true", help="mr_step launches every step itself (small grids replay CUDA graphs by default)")
    args = ap.parse_args(argv)
    if args.isohelix:
        if args.lambda0 == 1e-9:
            args.lambda0 = 1e-8
        return run_isohelix(args)
    if args.operator not in ("mimetic", "direct"):
        ap.error("--operator must be mimetic or direct")
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
