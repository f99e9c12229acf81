#!/usr/bin/env python
"""bench.py -- MPR site-updates/s at L = 16384 (BASELINE.json metric, configs[4]) on N B200s.

A step = one pass of the whole hot path over one synthetic problem: mpr_create (R1 map, sample
energy, mask bitmaps, R8 chain reset), mpr_estimate_temperature (energy matching, ~10 trials of
200 + 50 hybrid sweeps) and mpr_run(n_eq, n_meas) (Metropolis + over-relaxation sweeps, energy
reduction, accumulation of phi, back-map) in the headline precision mode.  One site-update = one
attempted single-site move, Metropolis or over-relaxation, at a prediction site (R11):
a hybrid sweep is 2 P site-updates.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

N > 1 (torchrun): every rank runs its own problem (another field / mask seed), no data-path
collective; value = site-updates of all ranks / max-over-ranks device time ("scaling": "weak").
--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "mpr_site_updates_per_s"
UNIT = "site-updates/s"
# ---- CPU legs (the oracle as it stands).  One temperature per config for BOTH cpu legs (cpu_baseline and --impl
# reference), close to the T_hat the GPU path infers, so that the two report the same quantity.
CPU_T = {1: 0.07, 2: 0.03, 3: 1.5e-3, 4: 1.5e-3, 5: 1.1e-3}
CPU_FULL_WARM, CPU_FULL_SWEEPS = 2, 3          # all host threads, the FULL grid: 2 warm-up + 3 timed hybrid sweeps
CPU_ONE_CROP, CPU_ONE_SWEEPS = 2048, 3         # one thread: top-left 2048^2 window, 1 warm-up + 3 timed sweeps

# ---- ceilings of the dominant kernel.  Algorithmic work of ONE unit (the two sites of one colour in
# one row that a lane owns) in ONE hybrid sweep = one Metropolis + one over-relaxation move per site, in this ISA's
# instructions, priced on the pipe that carries most of them, the FMA-heavy pipe (IMAD, IMAD.WIDE, packed f32x2):
#   Metropolis  Philox4x32-10 block shared by 4 sites (R9): 10 IMAD.WIDE per unit; local field 6 FADD2;
#               proposal 1 FFMA2; rotation / energy 13 packed (ts, nts, ps2, ns2, c2m1, 2 x (FMUL2 + FFMA2) for
#               (dc, ds), cn, sn, FMUL2 + FFMA2 for -dE); acceptance 1 FFMA2                    = 10 W + 21 P
#   over-relax. local field 6 FADD2; reflection 13 packed                                       = 19 P
# measured cost per warp instruction and scheduler (tests/helpers/pipe_microbench.cu, profiles/r02_microbench.md):
#   IMAD.WIDE.U32 4.27 cycles (inside a Philox block), FADD2 / FMUL2 2.03, FFMA2 2.34 -> packed average 2.1
ALG_FMA_CYCLES_PER_UNIT_SWEEP = 10 * 4.27 + (21 + 19) * 2.1       # = 126.7 scheduler cycles
# Double-arithmetic modes (DP, SP): the FP64 pipe carries the moves.  Per unit (two sites) and sweep 160 FP64-pipe
# instructions at the temperatures of configs 3-5 (DFMA / DMUL / DADD / DSETP / conversions; per site: Metropolis 37 -- local
# field 6, proposal from two Philox words 5, sin / cos of the half-angle with the 4 + 4 Taylor coefficients that delta needs
# there 11 (19 with all 8 + 8 at T > 0.04), rotation, difference and energy 12, decision filter 2, range test 1; the double
# exponential is only evaluated when the float filter cannot decide, ~3e-5 of the moves -- and over-relaxation 43 with its
# one division), at the measured 3.28 cycles per warp instruction and scheduler (DFMA 1.22 per clock and SM,
# profiles/r02_microbench.md).  Until the decision filter the count was 210.
ALG_FP64_CYCLES_PER_UNIT_SWEEP = 160 * 3.28
SMS, SCHEDULERS = 148, 4
# dram__bytes_read.sum + dram__bytes_write.sum of one launch at L = 16384 from the committed `ncu --set full` captures
# (profiles/); None for configurations not captured.
NCU_TRAFFIC_BYTES = {("SP_INTRINSIC", "R4", 1): 2.671e9 + 2.116e9,           # profiles/r02v_ncu_full.md
                     ("SP_INTRINSIC", "SITE_FUSED", 2): 2.678e9 + 2.119e9,   # profiles/r02s_ncu_full_strip.md
                     ("DP", "R4", 1): 4.330e9 + 4.246e9}                     # profiles/r02w_ncu_dp.md


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json configs index (1-based); 5 = L 16384")
    ap.add_argument("--mode", default="SP_INTRINSIC")
    ap.add_argument("--n-eq", type=int, default=None)
    ap.add_argument("--n-meas", type=int, default=None)
    ap.add_argument("--fused", type=int, default=0,
                    help="hybrid sweeps per launch; 0 = the library's choice (several on small grids, 1 at the headline size)")
    ap.add_argument("--path", default="AUTO", choices=["AUTO", "STRIP", "TILED", "PLAIN", "LIST"])
    ap.add_argument("--schedule", default="R4", choices=["R4", "SITE_FUSED"],
                    help="pass order of a hybrid sweep (DESIGN.md R4 / R4b); the headline is R4")
    ap.add_argument("--temperature", type=float, default=None,
                    help="profiling only: fix T and skip the temperature estimate (not the benchmark step)")
    ap.add_argument("--skip-cpu-baseline", action="store_true")
    ap.add_argument("--skip-modes", action="store_true")
    ap.add_argument("--skip-e2e", action="store_true")
    ap.add_argument("--skip-fused-leg", action="store_true", help="do not time the same step under the site-fused schedule")
    ap.add_argument("--matrix", action="store_true",
                    help="the paper's experiment shape (PAPER.md:35-57): R_X = t_DDD / t_X for the eight (X_S X_E X_F) settings "
                         "at L = 2^5 .. 2^12, f = 0.9, kappa = 0.2, and Delta MAAE_X over M mask realisations; one JSON line")
    ap.add_argument("--matrix-masks", type=int, default=10, help="M, mask realisations per data set for Delta MAAE (paper: 100)")
    ap.add_argument("--matrix-L", type=int, default=512, help="grid size of the Delta MAAE study")
    ap.add_argument("--slabs", type=int, default=0,
                    help="opt-in, SURVEY 8(e): ONE problem cut into row slabs (strong scaling).  Under torchrun: one slab per "
                         "rank, halo rows over NCCL.  On one GPU: --slabs G works the G slabs off in turn (what the exchange "
                         "schedule and the redundant halo rows cost; checked against the single-context run)")
    ap.add_argument("--halo", type=int, default=8, help="halo rows of a slab (a multiple of 4; exchange every halo / 4 sweeps)")
    ap.add_argument("--peer", action="store_true",
                    help="with --slabs on one GPU: peer mode (mpr_set_peers) -- every strip launch writes its edge rows straight "
                         "into the neighbours' halos, no copy launches; halo 4")
    ap.add_argument("--microbench", action="store_true",
                    help="build and run tests/helpers/pipe_microbench.cu (pipe throughputs, L2 / HBM copy) and exit")
    return ap.parse_args()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "200"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 6:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out = {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                   "samples": len(sm)}
        return out


def cpu_legs(values, mask, T, seed, full_sweeps=CPU_FULL_SWEEPS):
    """The oracle, as it stands, on the host cores: (a) all threads on the FULL grid, CPU_FULL_WARM warm-up +
    `full_sweeps` timed hybrid sweeps after an R8 start with 2 quench double passes; (b) one thread on the top-left
    CPU_ONE_CROP^2 window.  Returns (all-thread dict, one-thread dict)."""
    from oracle import mpr_oracle
    L = values.shape[0]
    cores = mpr_oracle.threads_available()
    t0 = time.perf_counter()
    o = mpr_oracle.Oracle(values=values, mask=mask, seed=seed, threads=cores, n_quench=2)
    o.set_temperature(T)
    t_init = time.perf_counter() - t0
    o.hybrid_sweeps(CPU_FULL_WARM)
    t0 = time.perf_counter()
    o.hybrid_sweeps(full_sweeps)
    dt = time.perf_counter() - t0
    n_free = int(mask.sum())
    full = {"value": 2.0 * n_free * full_sweeps / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "full %dx%d grid, %d warm-up + %d timed hybrid sweeps, T=%g, %.1f s (+ %.1f s set-up)" %
                      (L, L, CPU_FULL_WARM, full_sweeps, T, dt, t_init)}
    del o
    n = min(CPU_ONE_CROP, L)
    v1, m1 = np.ascontiguousarray(values[:n, :n]), np.ascontiguousarray(mask[:n, :n])
    o1 = mpr_oracle.Oracle(values=v1, mask=m1, seed=seed, threads=1, n_quench=2)
    o1.set_temperature(T)
    o1.hybrid_sweeps(1)
    t0 = time.perf_counter()
    o1.hybrid_sweeps(CPU_ONE_SWEEPS)
    dt1 = time.perf_counter() - t0
    one = {"value": 2.0 * int(m1.sum()) * CPU_ONE_SWEEPS / dt1, "unit": UNIT, "cores": 1, "kind": "oracle",
           "sample": "top-left %dx%d window, 1 warm-up + %d timed hybrid sweeps, T=%g, %.1f s" %
                     (n, n, CPU_ONE_SWEEPS, T, dt1)}
    return full, one


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle on the box's host cores; a step = CPU_FULL_SWEEPS hybrid sweeps of the
    full grid of the config (the same bounded sample cpu_baseline times)."""
    if rank != 0:
        return
    from oracle import mpr_oracle
    from paper_1910_08448_b200 import inputs
    c = inputs.CONFIGS[args.config]
    values, mask, _ = inputs.make_problem(c.L, c.xi, c.field_seed, c.f, c.lognormal)
    T = CPU_T[args.config]
    cores = mpr_oracle.threads_available()
    o = mpr_oracle.Oracle(values=values, mask=mask, seed=c.mpr_seed, threads=cores, n_quench=2)
    o.set_temperature(T)
    n_free = int(mask.sum())
    for _ in range(args.warmup):
        o.hybrid_sweeps(1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.hybrid_sweeps(CPU_FULL_SWEEPS)
    dt = time.perf_counter() - t0
    val = 2.0 * n_free * CPU_FULL_SWEEPS * args.steps / dt
    sample = "full %dx%d grid, %d hybrid sweeps per step (%d warm-up sweeps), T=%g" % (c.L, c.L, CPU_FULL_SWEEPS,
                                                                                    args.warmup, T)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": c.name, "L": c.L, "masked_fraction": c.f, "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def run_ours(args, rank, world, local_rank):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    from paper_1910_08448_b200 import inputs, mpr, sharding
    import torch.distributed as dist
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    c = inputs.CONFIGS[args.config]
    n_eq = c.n_eq if args.n_eq is None else args.n_eq
    n_meas = c.n_meas if args.n_meas is None else args.n_meas
    mode = args.mode
    # every rank its own problem of the same recipe (weak scaling; rank 0 = BASELINE.json's seed)
    t_gen = time.perf_counter()
    rp = sharding.rank_problem(c.field_seed, c.mpr_seed, rank, world)
    values, mask, truth = inputs.make_problem(c.L, c.xi, rp.field_seed, c.f, c.lognormal)
    t_gen = time.perf_counter() - t_gen
    L, N = c.L, c.L * c.L
    d_values = torch.from_numpy(values).to(dev)
    d_mask = torch.from_numpy(mask).to(dev)
    d_truth = torch.from_numpy(truth).to(dev)
    seed = rp.mpr_seed

    state = {"launches": 0, "sweeps": 0, "n_free": int(mask.sum()), "T": None, "trials": None, "pred": None,
             "e": None, "se": None, "eq_ms": 0.0, "eq_launches": 0}

    def step():
        g = mpr.Mpr(d_values, d_mask, mode=mode, seed=seed, device=dev)
        g.set_path(args.path)
        g.set_schedule(args.schedule)
        g.set_fused_sweeps(args.fused)
        if args.temperature is not None:
            g.set_temperature(args.temperature)
            T, es, nt = args.temperature, None, 0
        else:
            T, es, nt = g.estimate_temperature()
        pred, e, se = g.run(n_eq, n_meas)
        # the equilibration phase of run() = back-to-back launches of the dominant kernel alone, timed by
        # CUDA events on the library's stream INSIDE this step (mpr_get_run_timing)
        eq_ms, eq_l, _ = g.run_timing()
        state["eq_ms"] += eq_ms
        state["eq_launches"] += eq_l
        state["launches"] += g.launches()
        sw = nt * 250 + n_eq + n_meas
        state["sweeps"] += sw
        state.update(T=T, trials=nt, pred=pred, e=e, se=se, e_sample=es)
        g.close()
        return sw

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()

    for _ in range(args.warmup):
        step()
    state["launches"] = 0
    state["sweeps"] = 0
    state["eq_ms"] = 0.0
    state["eq_launches"] = 0
    barrier()
    clocks = ClockSampler(local_rank)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    clk = clocks.stop()
    ms_max, units_total, launches_total = sharding.aggregate(
        ms, 2.0 * state["n_free"] * state["sweeps"], state["launches"], world, device=dev)
    value = sharding.throughput(units_total, ms_max)
    path_used_early = args.path if args.path != "AUTO" else ("STRIP" if (mode in ("SP_INTRINSIC", "HP") and c.L >= 4096) else "OTHER")

    # ---- the same step in two other launch configurations, reported beside the headline (which stays R4, one sweep per
    # launch): the site-fused schedule (R4b) and R4 with two sweeps per launch (slower alone, but not clocked down by the
    # power cap in a long run: DESIGN.md 4.4).  Same work, same timing rules, SM clock sampled during each leg.
    def other_leg(schedule, k):
        def leg_step():
            gf = mpr.Mpr(d_values, d_mask, mode=mode, seed=seed, device=dev)
            gf.set_schedule(schedule)
            gf.set_fused_sweeps(k)
            if args.temperature is not None:
                gf.set_temperature(args.temperature)
                nt = 0
            else:
                _, _, nt = gf.estimate_temperature()
            pf, ef, sef = gf.run(n_eq, n_meas)
            ms_eq, n_l, n_sw = gf.run_timing()
            gf.close()
            return nt * 250 + n_eq + n_meas, pf, ef, sef, ms_eq, n_sw
        leg_step()
        barrier()
        leg_clocks = ClockSampler(local_rank)
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        f0.record()
        sw_f, eq_ms_f, eq_sw_f = 0, 0.0, 0
        for _ in range(args.steps):
            n_sw_step, pred_f, e_f, se_f, ms_eq, n_sw = leg_step()
            sw_f += n_sw_step
            eq_ms_f += ms_eq
            eq_sw_f += n_sw
        f1.record()
        barrier()
        leg_clk = leg_clocks.stop()
        msf_max, units_f, _ = sharding.aggregate(f0.elapsed_time(f1), 2.0 * state["n_free"] * sw_f, 0, world, device=dev)
        dfz = (pred_f - d_truth)[d_mask.bool()]
        return {"value": sharding.throughput(units_f, msf_max), "unit": UNIT, "ms_per_step": msf_max / args.steps,
                "schedule": schedule, "sweeps_per_launch": k, "ms_per_sweep_in_step": eq_ms_f / max(eq_sw_f, 1),
                "sm_mhz": leg_clk.get("sm_mhz"), "e_mean": e_f, "e_stderr": se_f, "mae": float(dfz.abs().mean().item())}

    fused_leg, k2_leg = None, None
    if args.schedule == "R4" and not args.skip_fused_leg and mode in ("SP_INTRINSIC", "HP"):
        fused_leg = other_leg("SITE_FUSED", 2)
        if path_used_early == "STRIP" and (args.fused or 1) == 1:
            k2_leg = other_leg("R4", 2)

    # prediction error of the last step (metric of PAPER.md Eq. 4; post-processing, not the path)
    m1 = d_mask.bool()
    diff = (state["pred"] - d_truth)[m1]
    mae, rmse = float(diff.abs().mean().item()), float(diff.pow(2).mean().sqrt().item())
    base_mae = float((d_truth[m1] - d_values[~m1].mean()).abs().mean().item())
    T_hat = state["T"]

    # ---- ceilings of the dominant kernel (the sweep launch without measurement), timed live ------------------
    def time_sweeps(md, path, schedule, k, n_launch, warm=6):
        gk = mpr.Mpr(d_values, d_mask, mode=md, seed=seed, device=dev)
        gk.set_path(path)
        gk.set_schedule(schedule)
        gk.set_fused_sweeps(k)
        gk.set_temperature(T_hat)
        gk.sweep(warm * k)
        torch.cuda.synchronize(dev)
        k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        k0.record()
        gk.sweep(n_launch * k)
        k1.record()
        torch.cuda.synchronize(dev)
        ms_launch = k0.elapsed_time(k1) / n_launch
        gk.run(0, 2, want_pred=False)      # first use of the measuring kernel (lazy module load) stays outside
        torch.cuda.synchronize(dev)
        k0.record()
        gk.run(0, 10, want_pred=False)
        k1.record()
        torch.cuda.synchronize(dev)
        gk.close()
        return ms_launch, k0.elapsed_time(k1) / 10

    # what MPR_PATH_AUTO resolves to (csrc/mpr.cu, eff_path)
    def auto_path(md, schedule):
        if schedule == "SITE_FUSED" and md != "HP":
            return "LIST" if (c.f < 0.5 and L <= 4096) else "STRIP"
        if md == "HP":
            return "STRIP" if L >= 4096 else "PLAIN"
        return "STRIP" if (md == "SP_INTRINSIC" and L >= 4096) else "TILED"
    path_used = auto_path(mode, args.schedule) if args.path == "AUTO" else args.path

    # what mpr_set_fused_sweeps(0) resolves to (csrc/mpr.cu, auto_fused)
    def auto_fused(md, path, sched=None):
        if path != "TILED":
            return 1
        if md in ("DP", "SP"):
            return 4 if L <= 256 else 2 if L <= 512 else 1
        return 4 if L <= 512 else 2 if L <= 1536 else 1
    k_lib = args.fused or auto_fused(mode, path_used)
    k_eff = min(k_lib, 2) if path_used == "STRIP" else k_lib
    kern_ms_burst, _ = time_sweeps(mode, args.path, args.schedule, k_lib, 50)   # the kernel timed alone, after the steps
    # the in-step figure (sustained clocks) is the one the ceilings use; the burst leg stands in only when the steps had
    # no equilibration sweeps
    in_step = state["eq_launches"] > 0
    kern_ms = state["eq_ms"] / state["eq_launches"] if in_step else kern_ms_burst
    peak, peak_src = peaks()
    sm_mhz = clk.get("sm_mhz") or 1965.0

    def ceilings(md, ms_launch, k, sm_mhz_used):
        """Ceilings of one sweep launch of k hybrid sweeps.  Bytes per SURVEY.md 8(d): every spin read once and written
        once per LAUNCH at the paper's storage width w (4 B in the float-storage modes: one 32-bit angle; 8 B in DP),
        plus the mask bits; `state_bytes` is what this library's layout moves (a unit vector per spin: 2 w)."""
        w = 8 if md == "DP" else 2 if md == "HP" else 4
        alg_bytes = 2.0 * N * w + N / 8.0
        state_bytes = 2.0 * N * 2 * w + N / 8.0
        # one unit = 2 sites of one colour and row; the method's arithmetic is owed at the PREDICTION sites only
        units = state["n_free"] / 2.0
        fma_cycles = units / 32.0 * k * ALG_FMA_CYCLES_PER_UNIT_SWEEP   # scheduler cycles on the FMA-heavy pipe
        fma_peak = SMS * SCHEDULERS * sm_mhz_used * 1e6             # scheduler cycles per second at the sampled clock
        t = ms_launch * 1e-3
        out = {
            "hbm_algorithmic": {"bytes_per_launch": alg_bytes, "achieved_gb_s": alg_bytes / t / 1e9,
                                "frac": alg_bytes / t / 1e9 / peak, "lower_bound_ms": alg_bytes / (peak * 1e9) * 1e3},
            "hbm_state_layout": {"bytes_per_launch": state_bytes, "achieved_gb_s": state_bytes / t / 1e9,
                                 "frac": state_bytes / t / 1e9 / peak, "lower_bound_ms": state_bytes / (peak * 1e9) * 1e3},
        }
        if md in ("DP", "SP"):
            cyc = units / 32.0 * k * ALG_FP64_CYCLES_PER_UNIT_SWEEP
            out["fp64_pipe"] = {"cycles_per_launch": cyc, "achieved_cycles_per_s": cyc / t, "peak_cycles_per_s": fma_peak,
                                "frac": cyc / t / fma_peak, "lower_bound_ms": cyc / fma_peak * 1e3, "sm_mhz": sm_mhz_used,
                                "cycles_per_unit_sweep": ALG_FP64_CYCLES_PER_UNIT_SWEEP}
        if md in ("SP_INTRINSIC", "SP_PRECISE", "HP"):
            out["fma_pipe"] = {"cycles_per_launch": fma_cycles, "achieved_cycles_per_s": fma_cycles / t,
                               "peak_cycles_per_s": fma_peak, "frac": fma_cycles / t / fma_peak,
                               "lower_bound_ms": fma_cycles / fma_peak * 1e3, "sm_mhz": sm_mhz_used,
                               "cycles_per_unit_sweep": ALG_FMA_CYCLES_PER_UNIT_SWEEP}
        return out

    ceil = ceilings(mode, kern_ms, k_eff, sm_mhz)
    # the binding ceiling = the one with the largest lower-bound time among those computed from ALGORITHMIC work
    pipe_key = "fma_pipe" if "fma_pipe" in ceil else "fp64_pipe" if "fp64_pipe" in ceil else None
    binding = "alu" if pipe_key and ceil[pipe_key]["lower_bound_ms"] > ceil["hbm_algorithmic"]["lower_bound_ms"] else "hbm"
    if binding == "alu":
        fp = ceil[pipe_key]
        roofline = {"bound": "alu", "achieved": fp["achieved_cycles_per_s"], "peak": fp["peak_cycles_per_s"],
                    "unit": ("FMA-pipe" if pipe_key == "fma_pipe" else "FP64-pipe") + " scheduler cycles/s", "frac": fp["frac"],
                    "peak_source": "148 SMs x 4 schedulers x SM clock sampled during the timed steps (%.0f MHz); "
                                   "instruction costs measured by tests/helpers/pipe_microbench.cu "
                                   "(profiles/r02_microbench.md)" % sm_mhz,
                    "binding_evidence": "ncu sm__pipe_fmaheavy_cycles_active is the busiest pipe (profiles/r02*_ncu_full*.md)"}
    else:
        ha = ceil["hbm_algorithmic"]
        roofline = {"bound": "hbm", "achieved": ha["achieved_gb_s"], "peak": peak, "unit": "GB/s", "frac": ha["frac"],
                    "peak_source": peak_src}
    roofline.update({
        "traffic": NCU_TRAFFIC_BYTES.get((mode, args.schedule, k_eff)) if L == 16384 else None,
        "kernel": "strip_kernel<%s, %s, k=%d, 0>" % (mode, args.schedule, k_eff) if path_used == "STRIP"
                  else "tiled_sweep_kernel<%s,0>" % mode,
        "kernel_ms": kern_ms,
        "kernel_ms_source": ("CUDA events around the %d equilibration launches inside the timed steps "
                             "(mpr_get_run_timing)" % state["eq_launches"]) if in_step else "burst leg",
        "kernel_ms_burst": kern_ms_burst, "sweeps_per_launch": k_eff,
        "kernel_ms_per_sweep": kern_ms / k_eff, "kernel_ms_burst_per_sweep": kern_ms_burst / k_eff,
        # the same fraction against the peak at the MAXIMUM SM clock: a launch that draws less power is clocked higher
        # under the cap, which raises the sampled-clock peak it is measured against (and lowers `frac`) while it runs faster
        "frac_at_max_clock": (roofline["frac"] * sm_mhz / (clk.get("sm_max_mhz") or sm_mhz)) if roofline["bound"] == "alu" else None,
        "algorithmic_bytes_per_launch": ceil["hbm_algorithmic"]["bytes_per_launch"],
        "state_bytes_per_launch": ceil["hbm_state_layout"]["bytes_per_launch"],
        "hbm_peak_gb_s": peak, "hbm_peak_source": peak_src,
        "ceilings": ceil,
        "kernel_site_updates_per_s": 2.0 * state["n_free"] * k_eff / (kern_ms * 1e-3),
    })

    # ---- per-mode sweep rates (BASELINE.json: "per precision mode"), both schedules --------------------------------
    modes = {}
    if not args.skip_modes:
        for md, n_sw in (("DP", 10), ("SP", 10), ("SP_PRECISE", 30), ("SP_INTRINSIC", 30), ("HP", 30)):
            if md not in c.modes and not (md == "HP" and "SP_INTRINSIC" in c.modes):     # HP: the paper's outlook, beside SSS
                continue
            entry = {}
            for sched, k in (("R4", auto_fused(md, auto_path(md, "R4"), "R4")), ("SITE_FUSED", 2)):
                t_l, t_meas = time_sweeps(md, "AUTO", sched, k, n_sw, warm=3)
                cl = ceilings(md, t_l, k, sm_mhz)
                entry[sched] = {"path": auto_path(md, sched), "sweeps_per_launch": k, "ms_per_sweep": t_l / k,
                                "site_updates_per_s": 2.0 * state["n_free"] * k / (t_l * 1e-3),
                                "ms_per_measurement_sweep": t_meas,
                                "frac_hbm_algorithmic": cl["hbm_algorithmic"]["frac"],
                                "frac_hbm_state_layout": cl["hbm_state_layout"]["frac"],
                                "frac_fma_pipe": cl.get("fma_pipe", {}).get("frac"),
                                "frac_fp64_pipe": cl.get("fp64_pipe", {}).get("frac")}
            modes[md] = entry

    # ---- end to end through the C ABI with HOST buffers (mpr_predict_host) ---------------------
    e2e = None
    if not args.skip_e2e:
        h_values = torch.from_numpy(values).pin_memory()
        h_mask = torch.from_numpy(mask).pin_memory()
        h_pred = torch.empty((L, L), dtype=torch.float64).pin_memory()
        ws = torch.empty(mpr.workspace_bytes(L, host=True) + 256, dtype=torch.uint8, device=dev)
        sweeps_e2e = 0

        def e2e_step():
            _, e, se, T, nl = mpr.predict_host(h_values.numpy(), h_mask.numpy(), mode=mode, seed=seed,
                                               T=-1.0 if args.temperature is None else args.temperature,
                                               n_eq=n_eq, n_meas=n_meas, workspace=ws, pred_out=h_pred.numpy(),
                                               device=dev)
            return nl

        e2e_step()
        barrier()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(args.steps):
            e2e_step()
        b.record()
        barrier()
        # same problem, seed and mode => same number of T trials as the device-resident steps
        sweeps_e2e = state["sweeps"]
        te_max, ue_total, _ = sharding.aggregate(a.elapsed_time(b), 2.0 * state["n_free"] * sweeps_e2e, 0, world,
                                                 device=dev)
        e2e = {"value": sharding.throughput(ue_total, te_max), "unit": UNIT, "h2d_bytes_per_step": 9 * N,
               "d2h_bytes_per_step": 8 * N, "ms_per_step": te_max / args.steps}
        del ws

    cpu = None
    if rank == 0 and not args.skip_cpu_baseline:
        cpu, cpu_one = cpu_legs(values, mask, CPU_T[args.config], seed)
        cpu["single_thread"] = cpu_one

    state_gib = 2.0 * N * (16 if mode == "DP" else 8) / 2 ** 30
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": {"DP": "f64", "SP": "f64"}.get(mode, "f32"), "data": "synthetic",
            "config": {"workload": c.name, "L": L, "masked_fraction": c.f, "mode": mode, "n_eq": n_eq,
                       "n_meas": n_meas, "T_trials": state["trials"], "sweeps_per_step": state["sweeps"] // args.steps,
                       "path": path_used, "schedule": args.schedule, "fused_sweeps": k_eff,
                       "parallelism": "replicas x%d" % world,
                       "l2": ("state (%.2f GiB) larger than the 126 MB L2; no flush" % (state_gib)) if state_gib * 2 ** 30 > 126e6
                             else "state (%.1f MiB) is L2-resident by design of this config (BASELINE.json); no flush" % (state_gib * 1024)},
            "clocks": clk, "e2e": e2e, "gpu_launches": launches_total, "roofline": roofline,
            "cpu_baseline": cpu, "modes": modes, "site_fused": fused_leg, "two_sweeps_per_launch": k2_leg, "T_hat": T_hat, "e_sample": state.get("e_sample"),
            "e_mean": state["e"], "e_stderr": state["se"], "mae": mae, "rmse": rmse,
            "mae_of_sample_mean_predictor": base_mae, "input_generation_s": t_gen,
        }))
    if world > 1:
        dist.destroy_process_group()


def run_matrix(args):
    """PAPER.md:35 (eight precision settings), :39 / :47 (Fig. 1: R_X = t_DDD / t_X against L = 2^k, k = 5 .. 12, Gaussian
    N(50, 10) data with exponential covariance, kappa = 0.2, 90 % removed), :55-57 (Fig. 2: Delta MAAE_X in % over M mask
    realisations of one data set).  Synthetic stand-ins from inputs.make_problem (xi = 1 / kappa = 5)."""
    import torch
    from paper_1910_08448_b200 import inputs, mpr
    dev = torch.device("cuda", 0)
    n_eq, n_meas = 200, 50
    out = {"triples": list(mpr.TRIPLES), "n_eq": n_eq, "n_meas": n_meas, "f": 0.9, "kappa": 0.2, "R_X": {}, "ms": {}}
    for k in range(5, 13):
        L = 2 ** k
        values, mask, _ = inputs.make_problem(L, 5.0, 100 + k, 0.9, False)
        dv, dm = torch.from_numpy(values).to(dev), torch.from_numpy(mask).to(dev)
        g0 = mpr.Mpr(dv, dm, mode="DP", seed=7, device=dev)
        T_hat, _, _ = g0.estimate_temperature()
        g0.close()
        ms = {}
        for X in mpr.TRIPLES:
            g = mpr.Mpr(dv, dm, seed=7, device=dev)
            g.set_precision_triple(X)
            g.set_temperature(T_hat)
            g.run(20, 5, want_pred=False)
            best = None
            for _ in range(3):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize(dev)
                a.record()
                g.run(n_eq, n_meas, want_pred=True)
                b.record()
                torch.cuda.synchronize(dev)
                t = a.elapsed_time(b)
                best = t if best is None or t < best else best
            ms[X] = best
            g.close()
        out["ms"][str(L)] = ms
        out["R_X"][str(L)] = {X: ms["DDD"] / ms[X] for X in mpr.TRIPLES}
    # Delta MAAE_X: one data set, M masks; paired over the masks
    L, M = args.matrix_L, args.matrix_masks
    field_rng = np.random.default_rng(4242)
    z = 50.0 + 10.0 * inputs.matern_field(L, 5.0, field_rng)
    maes = {X: [] for X in mpr.TRIPLES}
    for m in range(M):
        rng = np.random.default_rng(9000 + m)
        mask = np.zeros(L * L, dtype=np.uint8)
        mask[rng.choice(L * L, size=round(0.9 * L * L), replace=False, shuffle=False)] = 1
        mask = mask.reshape(L, L)
        vals = np.where(mask == 1, np.nan, z)
        dv, dm, dt = torch.from_numpy(vals).to(dev), torch.from_numpy(mask).to(dev), torch.from_numpy(z).to(dev)
        g0 = mpr.Mpr(dv, dm, mode="DP", seed=11 + m, device=dev)
        T_hat, _, _ = g0.estimate_temperature()
        g0.close()
        free = dm.bool()
        for X in mpr.TRIPLES:
            g = mpr.Mpr(dv, dm, seed=11 + m, device=dev)
            g.set_precision_triple(X)
            g.set_temperature(T_hat)
            pred, _, _ = g.run(300, 100)
            maes[X].append(float((pred - dt)[free].abs().mean()))
            g.close()
    ref = np.array(maes["DDD"])
    out["delta_maae_pct"] = {}
    for X in mpr.TRIPLES:
        a = np.array(maes[X])
        d = 100.0 * (a.mean() / ref.mean() - 1.0)
        # error bar: standard error of the paired relative differences over the masks
        se = 100.0 * float(np.std(a / ref - 1.0, ddof=1) / np.sqrt(M)) if M > 1 else None
        out["delta_maae_pct"][X] = {"value": d, "stderr": se, "maae": float(a.mean())}
    out["delta_maae_config"] = {"L": L, "M": M, "n_eq": 300, "n_meas": 100}
    print(json.dumps({"matrix": out, "data": "synthetic"}))


def run_microbench():
    """Measured per-SM pipe throughputs and copy bandwidths (JSON lines on stdout): the denominators of the
    "alu" ceilings, taken on the box the bench runs on."""
    src = os.path.join(ROOT, "tests", "helpers", "pipe_microbench.cu")
    with tempfile.TemporaryDirectory() as td:
        exe = os.path.join(td, "pipe_microbench")
        subprocess.run([os.environ.get("NVCC", "nvcc"), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-o", exe, src],
                       check=True)
        subprocess.run([exe], check=True)


def run_slabs(args, rank, world, local_rank):
    """One problem (rank 0's seeds) on slabs: temperature matching + run(n_eq, n_meas) over all slabs."""
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1910_08448_b200 import inputs, mpr, slabs
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    c = inputs.CONFIGS[args.config]
    n_eq = c.n_eq if args.n_eq is None else args.n_eq
    n_meas = c.n_meas if args.n_meas is None else args.n_meas
    values, mask, truth = inputs.make_problem(c.L, c.xi, c.field_seed, c.f, c.lognormal)
    count = world if world > 1 else max(1, args.slabs)
    transport = slabs.DistTransport() if world > 1 else None
    peer = args.peer and world == 1
    ss = slabs.make_slab_set(values, mask, count, halo=4 if peer else args.halo, mode=args.mode, seed=c.mpr_seed, device=str(dev),
                             path="STRIP" if peer else args.path, schedule=args.schedule, transport=transport, peer=peer)

    def sync():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()

    def step():
        if args.temperature is not None:
            ss.set_temperature(args.temperature)
            ss.reset_chain(0)
            nt = 0
        else:
            ss.estimate_temperature()
            nt = ss.n_trials
        # the equilibration sweeps timed by themselves (all slabs, exchanges included), then the measuring sweeps
        q0, q1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        q0.record()
        ss.sweep(n_eq)
        q1.record()
        _, e, se = ss.run(0, n_meas)
        torch.cuda.synchronize(dev)
        eq["ms"] += q0.elapsed_time(q1)
        eq["sweeps"] += n_eq
        return nt * sum(ss.trial_lengths) + n_eq + n_meas, e, se

    eq = {"ms": 0.0, "sweeps": 0}

    for _ in range(args.warmup):
        step()
    sync()
    eq.update(ms=0.0, sweeps=0)
    clocks = ClockSampler(local_rank)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    sweeps = 0
    for _ in range(args.steps):
        n, e, se = step()
        sweeps += n
    ev1.record()
    sync()
    clk = clocks.stop()
    ms = ev0.elapsed_time(ev1)
    if world > 1:
        t = torch.tensor([ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    # prediction error over the own rows of this process's slabs, summed over the ranks
    err = np.zeros(2)
    for i, sl in ss.slabs.items():
        p = sl.plan
        pr, tr, mk = sl.own_prediction(), truth[p.own_begin_g:p.own_end_g], mask[p.own_begin_g:p.own_end_g] == 1
        err += [np.abs(pr - tr)[mk].sum(), mk.sum()]
    err = ss.transport.reduce_sum([err])
    check = None
    if world == 1 and count > 1 and args.temperature is not None:
        g = mpr.Mpr(values, mask, mode=args.mode, seed=c.mpr_seed, device=dev)
        g.set_path("STRIP" if peer else args.path); g.set_schedule(args.schedule); g.set_temperature(args.temperature)
        g.run(n_eq, n_meas)
        check = bool(np.array_equal(g.get_state().cpu().numpy(), ss.state()))
        g.close()
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": 2.0 * ss.n_free * sweeps / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f64" if args.mode == "DP" else "f32", "data": "synthetic",
            "config": {"workload": "config%d_L%d" % (args.config, c.L), "L": c.L, "masked_fraction": c.f, "mode": args.mode,
                       "n_eq": n_eq, "n_meas": n_meas, "parallelism": "slabs x%d%s" % (count, "" if world > 1 else " on one GPU, in turn"),
                       "halo_rows": ss.halo, "sweeps_per_exchange": ss.sweeps_per_exchange,
                       "exchange": "in-kernel peer stores" if peer else "export / import copies between launches",
                       "l2": "state larger than the 126 MB L2; no flush" if c.L >= 4096 else "L2-resident state"},
            "clocks": clk, "T_hat": ss.T, "e_mean": e, "e_stderr": se, "mae": float(err[0] / max(err[1], 1.0)),
            "exchanges": ss.exchanges, "identical_to_single_context": check,
            "ms_per_equilibration_sweep": eq["ms"] / max(eq["sweeps"], 1),
        }))
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.microbench:
        run_microbench()
        return
    if args.matrix:
        run_matrix(args)
        return
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    elif args.slabs:
        run_slabs(args, rank, world, local_rank)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
