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
CPU_CROP = 4096          # cpu_baseline / reference arm: top-left CPU_CROP^2 window of the workload
CPU_EQ, CPU_MEAS = 110, 4  # ~3.4e9 site-updates: ~15 s on the 16 host threads of the B200 box (measured 2.3e8 /s)
ALG_WARP_INST_PER_32_UNITS = 125.0   # Metropolis 91 + over-relaxation 34 per unit and sweep
# dram__bytes_read.sum + dram__bytes_write.sum of one launch of the dominant kernel at L = 16384, from the
# committed `ncu --set full` capture (profiles/r01g_ncu_full_tiled_v4.md); None for configurations not captured.
NCU_TRAFFIC_BYTES = {("SP_INTRINSIC", 1): 2.182e9 + 2.099e9}


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
    ap.add_argument("--fused", type=int, default=1)
    ap.add_argument("--temperature", type=float, default=None,
                    help="profiling only: fix T and skip the temperature estimate (not the benchmark step)")
    ap.add_argument("--skip-cpu-baseline", action="store_true")
    ap.add_argument("--skip-modes", action="store_true")
    ap.add_argument("--skip-e2e", action="store_true")
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


def cpu_sample(values, mask, T, seed):
    """The oracle, as it stands, on the top-left CPU_CROP^2 window: run(CPU_EQ, CPU_MEAS), all host threads."""
    from oracle import mpr_oracle
    n = min(CPU_CROP, values.shape[0])
    v = np.ascontiguousarray(values[:n, :n])
    m = np.ascontiguousarray(mask[:n, :n])
    cores = mpr_oracle.threads_available()
    o = mpr_oracle.Oracle(values=v, mask=m, seed=seed, threads=cores)
    o.set_temperature(T)
    return o, int(m.sum()), cores, n


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle on the box's host cores, bounded sample per step."""
    if rank != 0:
        return
    from paper_1910_08448_b200 import inputs
    c = inputs.CONFIGS[args.config]
    values, mask, _ = inputs.make_problem(c.L, c.xi, c.field_seed, c.f, c.lognormal)
    o, n_free, cores, n = cpu_sample(values, mask, 0.05, c.mpr_seed)
    upd = 2.0 * n_free * (CPU_EQ + CPU_MEAS)
    for _ in range(args.warmup):
        o.run(CPU_EQ, CPU_MEAS)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.run(CPU_EQ, CPU_MEAS)
    dt = time.perf_counter() - t0
    val = upd * args.steps / dt
    sample = "top-left %dx%d window of the L=%d workload, run(%d,%d) per step, T=0.05" % (n, n, c.L, CPU_EQ, CPU_MEAS)
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

    # prediction error of the last step (metric of PAPER.md Eq. 4; post-processing, not the path)
    m1 = d_mask.bool()
    diff = (state["pred"] - d_truth)[m1]
    mae, rmse = float(diff.abs().mean().item()), float(diff.pow(2).mean().sqrt().item())
    base_mae = float((d_truth[m1] - d_values[~m1].mean()).abs().mean().item())
    T_hat = state["T"]

    # ---- roofline of the dominant kernel: tiled_sweep_kernel<mode, false>, timed live ----------
    g = mpr.Mpr(d_values, d_mask, mode=mode, seed=seed, device=dev)
    g.set_fused_sweeps(args.fused)
    g.set_temperature(T_hat)
    g.sweep(8 * args.fused)
    n_l = 50
    torch.cuda.synchronize(dev)
    k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    k0.record()
    g.sweep(n_l * args.fused)
    k1.record()
    torch.cuda.synchronize(dev)
    kern_ms_burst = k0.elapsed_time(k1) / n_l      # the kernel timed alone, 50 launches after the steps
    g.close()
    # roofline uses the average launch duration INSIDE the timed steps (sustained clocks); the burst leg
    # is reported beside it and stands in only when the steps had no equilibration sweeps
    in_step = state["eq_launches"] > 0
    kern_ms = state["eq_ms"] / state["eq_launches"] if in_step else kern_ms_burst
    w = 16 if mode == "DP" else 8
    Wp = (((L + 1) // 2 + 15) // 16) * 16
    stored = 2 * L * Wp
    alg_bytes = stored * 2 * w + 2 * stored / 8.0          # read + write of every stored spin, mask bits
    peak, peak_src = peaks()
    achieved = alg_bytes / (kern_ms * 1e-3) / 1e9
    # second ceiling: warp-instruction issue.  Algorithmic count = 125 warp instructions per
    # 32 units (unit = 2 sites of one colour and row) per hybrid sweep; peak = 148 SMs x 4 schedulers x 1 / clk.
    alg_inst = (stored / 2.0) / 32.0 * ALG_WARP_INST_PER_32_UNITS * args.fused
    sm_hz = (clk.get("sm_max_mhz") or 1965.0) * 1e6
    issue_peak = 148 * 4 * sm_hz
    alu = {"bound": "alu", "achieved": alg_inst / (kern_ms * 1e-3), "peak": issue_peak, "unit": "warp-inst/s",
           "frac": alg_inst / (kern_ms * 1e-3) / issue_peak, "algorithmic_warp_inst_per_launch": alg_inst}
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": NCU_TRAFFIC_BYTES.get((mode, args.fused)) if L == 16384 else None, "kernel": "tiled_sweep_kernel<%s,0>" % mode,
                "kernel_ms": kern_ms,
                "kernel_ms_source": ("CUDA events around the %d equilibration launches inside the timed steps "
                                     "(mpr_get_run_timing)" % state["eq_launches"]) if in_step else "burst leg",
                "kernel_ms_burst": kern_ms_burst, "frac_burst": alg_bytes / (kern_ms_burst * 1e-3) / 1e9 / peak,
                "algorithmic_bytes_per_launch": alg_bytes, "sweeps_per_launch": args.fused, "peak_source": peak_src,
                "kernel_site_updates_per_s": 2.0 * state["n_free"] * args.fused / (kern_ms * 1e-3),
                "second_ceiling": alu}

    # ---- per-mode sweep rates (BASELINE.json: "per precision mode") ----------------------------
    modes = {}
    if not args.skip_modes:
        for md, n_sw in (("DP", 10), ("SP", 10), ("SP_PRECISE", 30), ("SP_INTRINSIC", 30)):
            if md not in c.modes:
                continue
            gm = mpr.Mpr(d_values, d_mask, mode=md, seed=seed, device=dev)
            gm.set_temperature(T_hat)
            gm.sweep(3)
            torch.cuda.synchronize(dev)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            gm.sweep(n_sw)
            b.record()
            torch.cuda.synchronize(dev)
            t = a.elapsed_time(b) / n_sw
            a.record()
            _, e_m, se_m = gm.run(0, 5, want_pred=False)
            b.record()
            torch.cuda.synchronize(dev)
            # same definitions as `roofline` above: every stored spin read and written once + the mask bits
            md_bytes = stored * 2 * (16 if md == "DP" else 8) + 2 * stored / 8.0
            modes[md] = {"ms_per_sweep": t, "site_updates_per_s": 2.0 * state["n_free"] / (t * 1e-3),
                         "hbm_roofline_frac": md_bytes / (t * 1e-3) / 1e9 / peak,
                         "ms_per_measurement_sweep": a.elapsed_time(b) / 5,
                         # mean of 5 samples taken 3 + n_sw sweeps after the chain reset: NOT an equilibrium
                         # value and not comparable between modes (n_sw differs); a plausibility figure only
                         "e_unequilibrated_after_%d_sweeps" % (3 + n_sw): e_m}
            gm.close()

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
        o, nf, cores, n = cpu_sample(values, mask, T_hat, seed)
        o.run(1, 0)
        t0 = time.perf_counter()
        o.run(CPU_EQ, CPU_MEAS)
        dt = time.perf_counter() - t0
        cpu = {"value": 2.0 * nf * (CPU_EQ + CPU_MEAS) / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": "top-left %dx%d window of the L=%d workload, run(%d,%d), T=T_hat, %.1f s" %
                         (n, n, L, CPU_EQ, CPU_MEAS, dt)}

    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": {"DP": "f64", "SP": "f64"}.get(mode, "f32"), "data": "synthetic",
            "config": {"workload": c.name, "L": L, "masked_fraction": c.f, "mode": mode, "n_eq": n_eq,
                       "n_meas": n_meas, "T_trials": state["trials"], "sweeps_per_step": state["sweeps"] // args.steps,
                       "fused_sweeps": args.fused, "parallelism": "replicas x%d" % world,
                       "l2": "state (%.1f GiB) larger than L2; no flush" % (stored * w / 2 ** 30)},
            "clocks": clk, "e2e": e2e, "gpu_launches": launches_total, "roofline": roofline,
            "cpu_baseline": cpu, "modes": modes, "T_hat": T_hat, "e_sample": state.get("e_sample"),
            "e_mean": state["e"], "e_stderr": state["se"], "mae": mae, "rmse": rmse,
            "mae_of_sample_mean_predictor": base_mae, "input_generation_s": t_gen,
        }))
    if world > 1:
        dist.destroy_process_group()


def run_microbench():
    """Measured per-SM pipe throughputs and copy bandwidths (JSON lines on stdout): the denominators of the
    "alu" ceilings, taken on the box the bench runs on."""
    src = os.path.join(ROOT, "tests", "helpers", "pipe_microbench.cu")
    with tempfile.TemporaryDirectory() as td:
        exe = os.path.join(td, "pipe_microbench")
        subprocess.run([os.environ.get("NVCC", "nvcc"), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-o", exe, src],
                       check=True)
        subprocess.run([exe], check=True)


def main():
    args = parse()
    if args.microbench:
        run_microbench()
        return
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
