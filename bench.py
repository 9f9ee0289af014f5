#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200 hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 4] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is one leap-frog time step of the whole hot path (whole-grid update, fractional-grid update,
reductions, bookkeeping -- SURVEY.md 8(a) rows S1-S9) over the workload's lattice.  Default workload:
BASELINE.json configs[4] ("bandwidth stress", 512 harmonics x 32001 phi_y points, 525 MB of state), the
configuration the HBM-roofline target is quoted on.  Prints ONE JSON line (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1401_6047_b200 import workloads as W  # noqa: E402

METRIC = "fp64 grid-point updates/s per time step; achieved HBM GB/s vs B200 peak"   # BASELINE.json "metric"
UNIT = "updates/s"
BYTES_PER_UPDATE = 64.0   # a_h, b_h, a_f, b_f each read once and written once


def measured_peak_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def recorded_traffic(workload_name, steps_per_launch):
    """dram bytes per launch of the dominant kernel from the committed ncu --set full capture."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        with open(p) as f:
            d = json.load(f)
        return d.get(workload_name, {}).get(f"S{int(round(steps_per_launch))}", {}).get("dram_bytes_per_launch")
    except Exception:
        return None


class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc = index, None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "50",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return None
        time.sleep(0.06)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            return None
        sm, smax, power, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in out.strip().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); smax.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for nm, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return None
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(smax), "power_w_max": max(power),
                "samples": len(sm), "reasons": sorted(reasons)}


from paper_1401_6047_b200.multi import dist_env, replica_workload, max_over_ranks as _max_over_ranks  # noqa: E402


# ---------------------------------------------------------------------------------------------------
# reference arm: the oracle, as it stands, on the host cores
# ---------------------------------------------------------------------------------------------------
def oracle_sample(w, steps, warmup, budget_updates=2.5e9):
    """A bounded sample of the workload: the same lattice rows, dt, dphi and parameters on a phi_y window
    of fewer columns (system 0), sized so that (steps + warmup) steps stay within budget_updates."""
    rows = w.grid.n_harm + 1
    cols = int(budget_updates / max(1, steps + warmup) / rows)
    cols = max(65, min(w.grid.n_phiy, cols | 1))
    p = W.Params(**vars(w.params[0]))
    dphi = (p.phiy_max - p.phiy_min) / (w.grid.n_phiy - 1)
    half = dphi * (cols - 1) / 2.0
    p.phiy_min, p.phiy_max, p.n_steps_total = -half, half, 0
    return cols, p


def run_reference(args):
    rank, world, _ = dist_env()
    if rank != 0:
        return 0
    from oracle import OracleSim, max_threads
    w = W.get(args.workload)
    threads = max_threads()
    cols, p = oracle_sample(w, args.steps, args.warmup, args.ref_budget)
    sim = OracleSim(w.grid.n_harm, cols, w.grid.dt, p, threads=threads)
    sim.init_equilibrium()
    sim.step(args.warmup)
    t0 = time.perf_counter()
    sim.step(args.steps)
    el = time.perf_counter() - t0
    pts = (w.grid.n_harm + 1) * cols
    val = pts * args.steps / el
    sample = (f"oracle/bte_oracle.cpp, {args.steps} steps on a {w.grid.n_harm + 1} x {cols} phi_y window of "
              f"{w.name} (same dt, dphi, parameters), {threads} OpenMP threads")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": el / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": w.name, **w.describe()},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def cpu_baseline(w, target_seconds=12.0):
    """Oracle timed beside the GPU number (rank 0, N=1): first steps of the same workload, system 0."""
    from oracle import OracleSim, max_threads
    threads = max_threads()
    sim = OracleSim(w.grid.n_harm, w.grid.n_phiy, w.grid.dt, w.params[0], threads=threads)
    sim.init_equilibrium()
    pts = w.points_per_system
    t0 = time.perf_counter()
    sim.step(1)
    one = max(time.perf_counter() - t0, 1e-6)
    n = int(max(2, min(2000, target_seconds / one)))
    t0 = time.perf_counter()
    sim.step(n)
    el = time.perf_counter() - t0
    # the same oracle on ONE thread (the paper's own CPU figure is single-threaded)
    sim1 = OracleSim(w.grid.n_harm, w.grid.n_phiy, w.grid.dt, w.params[0], threads=1)
    sim1.init_equilibrium()
    n1 = int(max(1, min(n, (target_seconds / 3.0) / (one * threads))))
    t0 = time.perf_counter()
    sim1.step(n1)
    el1 = time.perf_counter() - t0
    return {"value": pts * n / el, "unit": UNIT, "cores": threads, "kind": "oracle",
            "value_1_thread": pts * n1 / el1,
            "sample": f"oracle/bte_oracle.cpp, steps 2..{n + 1} of {w.name} system 0 "
                      f"({pts} points/step), {threads} OpenMP threads, {el:.1f} s; then {n1} step(s) on 1 thread, "
                      f"{el1:.1f} s"}


# ---------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1401_6047_b200 import Solver

    rank, world, local = dist_env()
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    w = replica_workload(args.workload, rank)
    pts_all = w.points_per_system * w.grid.n_batch

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x):
        return _max_over_ranks(x, dev)

    # ---- device-resident measurement: inputs (state) already in HBM ---------------------------------
    s = Solver(w.grid, w.params, device=dev, precision=args.precision)
    if args.variant:
        s.set_option("variant", args.variant)
    if args.tile_rows:
        s.set_option("tile_rows", args.tile_rows)
    if args.sweep_steps:
        s.set_option("sweep_steps", args.sweep_steps)
    if args.ctas:
        s.set_option("sweep_ctas", args.ctas)
    if args.res_ctas:
        s.set_option("resident_ctas", args.res_ctas)
    if args.sweep_threads:
        s.set_option("sweep_threads", args.sweep_threads)
    s.init_equilibrium()
    s.step(max(3, args.warmup))
    barrier()
    launches0 = s.launch_count()
    sampler = ClockSampler(local)
    sampler.start()
    e0 = torch.cuda.Event(enable_timing=True)
    e1 = torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(s.stream)
    s.step(args.steps)
    e1.record(s.stream)
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    launches = s.launch_count() - launches0
    ms = max_over_ranks(ms)
    warm = max(3, args.warmup)
    updates = w.updates_between(warm, warm + args.steps)
    value = updates * world / (ms * 1e-3)
    obs = s.observables()[0]
    # The same workload with ONE time step per pass (sweep_steps = 1): the plain HBM-bound form of the step
    # kernel, whose 64 B per update is what SURVEY 8(d) counts -- reported beside the headline so that the
    # HBM-roofline fraction of the memory-bound variant is measured in the same run (not the headline value).
    one_pass = None
    if 1 < launches < args.steps and not args.sweep_steps and args.variant in (0, 3):
        s.set_option("variant", 3)
        s.set_option("sweep_steps", 1)
        k1 = max(50, min(400, args.steps // 5))
        s.step(3)
        barrier()
        l0 = s.launch_count()
        e0.record(s.stream)
        s.step(k1)
        e1.record(s.stream)
        barrier()
        ms1 = max_over_ranks(e0.elapsed_time(e1))
        done = warm + args.steps + 3
        upd1 = w.updates_between(done, done + k1)
        one_pass = {"steps": k1, "launches": s.launch_count() - l0, "ms_per_step": ms1 / k1,
                    "updates_per_s": upd1 * world / (ms1 * 1e-3),
                    "achieved_gbs": BYTES_PER_UPDATE * upd1 / (ms1 * 1e-3) / 1e9}
    s.destroy()
    del s
    torch.cuda.empty_cache()

    # ---- end to end through the public API with HOST buffers ------------------------------------------
    # The state (a, b on both grids of every system) starts in pinned HOST memory and ends there.  Timed:
    # bte_create (table upload H2D) -> bte_set_state x 2 per system (H2D of the inputs) -> bte_step(K) ->
    # bte_observables -> bte_get_state x 2 per system (D2H of the result).  Wall clock, max over ranks.
    def configure(sol):
        if args.variant:
            sol.set_option("variant", args.variant)
        if args.tile_rows:
            sol.set_option("tile_rows", args.tile_rows)
        if args.sweep_steps:
            sol.set_option("sweep_steps", args.sweep_steps)
        if args.ctas:
            sol.set_option("sweep_ctas", args.ctas)
        if args.res_ctas:
            sol.set_option("resident_ctas", args.res_ctas)
        if args.sweep_threads:
            sol.set_option("sweep_threads", args.sweep_threads)

    nb, shape = w.grid.n_batch, (w.grid.n_harm + 1, w.grid.n_phiy)
    host_in = torch.empty((nb, 2, 2) + shape, dtype=torch.float64).pin_memory()
    host_out = torch.empty((nb, 2, 2) + shape, dtype=torch.float64).pin_memory()
    hin, hout = host_in.numpy(), host_out.numpy()
    s1 = Solver(w.grid, w.params, device=dev, precision=args.precision)   # untimed: the t = 0 state on the host
    s1.init_equilibrium()
    for i in range(nb):
        for g in (0, 1):
            s1.get_state(i, g, hin[i, g, 0], hin[i, g, 1])
    s1.destroy()
    del s1
    barrier()
    t0 = time.perf_counter()
    s2 = Solver(w.grid, w.params, device=dev, precision=args.precision)
    configure(s2)
    for i in range(nb):
        for g in (0, 1):
            s2.set_state(i, g, hin[i, g, 0], hin[i, g, 1])
    s2.step(args.steps)
    obs2 = s2.observables()
    for i in range(nb):
        for g in (0, 1):
            s2.get_state(i, g, hout[i, g, 0], hout[i, g, 1])
    torch.cuda.synchronize()
    e2e_s = max_over_ranks(time.perf_counter() - t0)
    rows, pitch = shape[0], (shape[1] + 7) // 8 * 8
    state_bytes = nb * 2 * 2 * 8 * shape[0] * shape[1]
    h2d = nb * (8 * rows + 16 * pitch + 80) + state_bytes      # c_n, g_m, phi_m tables + constants + state
    d2h = nb * 96 + state_bytes                                 # observables + state
    e2e_val = w.updates_between(0, args.steps) * world / e2e_s
    s2.destroy()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    peak, peak_src = measured_peak_gbs()
    # One launch of the sweep kernel advances every active system by S = steps / launches time steps in one
    # pass over the state (temporal blocking): what that launch must move is the state read once and written
    # once = 64 B per lattice point PER LAUNCH.
    per_launch_s = ms * 1e-3 / max(1, launches)
    steps_per_launch = args.steps / max(1, launches)
    alg_bytes = BYTES_PER_UPDATE * updates / args.steps          # per launch: 64 B x active points
    achieved = alg_bytes / per_launch_s / 1e9
    effective = BYTES_PER_UPDATE * updates / (ms * 1e-3) / 1e9   # at 64 B per update (one-step-per-pass model)
    fp64_peak = 148 * 64 * 1.965e9                               # DFMA-class thread-instructions/s
    fp64_rate = 2 * 26 * updates / (ms * 1e-3)                   # 26 fp64 instructions per half-update
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(3, args.warmup), "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None,
        "dtype": ("f64", "f32 storage / f64 arithmetic", "f32")[args.precision], "data": "synthetic",
        "config": {"workload": w.name, **w.describe(), "state_bytes": 32 * pts_all,
                   "l2_policy": (f"inputs larger than L2 ({32 * pts_all / 1e6:.0f} MB state vs 126 MB L2)"
                                 if 32 * pts_all > 2.6e8 else
                                 "state fits on chip / in L2: resident regime, reported as such"),
                   "multi_gpu": "independent replicas, one system per rank, no collective",
                   "paper_convention_updates_per_s": value * w.grid.n_harm / (w.grid.n_harm + 1)},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "frac_of_nominal_8TBs": achieved / 8000.0,
                     "traffic": recorded_traffic(w.name, steps_per_launch),
                     "kernel": "sweep_kernel" if launches > 1 else "resident_kernel", "steps_per_launch": steps_per_launch,
                     "algorithmic_bytes_per_launch": alg_bytes,
                     "peak_source": peak_src,
                     "effective_gbs_at_64B_per_update": effective,
                     "effective_note": ("temporal blocking: one pass over the state advances steps_per_launch "
                                        "time steps, so the one-step-per-pass figure (64 B per update) can exceed "
                                        "the HBM peak; 'achieved' counts what a launch really has to move"),
                     "fp64_pipe_frac": fp64_rate / fp64_peak,
                     "one_step_per_pass": (dict(one_pass, frac=one_pass["achieved_gbs"] / peak,
                                                frac_of_nominal_8TBs=one_pass["achieved_gbs"] / 8000.0,
                                                note="same workload, sweep_steps = 1: the HBM-bound form "
                                                     "(64 B of HBM traffic per update), measured in this run")
                                           if one_pass else None)},
        "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d / args.steps,
                "d2h_bytes_per_step": d2h / args.steps, "seconds": e2e_s,
                "what": "state in pinned host memory -> bte_create + bte_set_state (H2D) + bte_step(K) + bte_observables + bte_get_state (D2H) -> pinned host memory"},
        "gpu_launches": launches,
        "clocks": clocks,
        "check": {"norm": obs.norm, "v_dr": obs.v_dr, "step": obs.step, "e2e_step": obs2[0].step},
    }
    if w.name == "paper_table1":
        # the paper's own workload and MLUPS convention (n-harmonics x g-grid x steps / time, L328); its number is
        # fp32 on a GTX680 -- ours is fp64 unless --precision says otherwise: context, not the target
        mlups = value * w.grid.n_harm / (w.grid.n_harm + 1) / 1e6
        line["vs_baseline"] = mlups / W.PAPER_TABLE1_MLUPS_K6
        line["config"]["paper_mlups"] = {"ours": mlups, "paper_K6_GTX680_fp32": W.PAPER_TABLE1_MLUPS_K6,
                                         "paper_cpu_1_thread_fp32": 9.0, "source": "PAPER.md:L315-328 (Table 1)"}
    if launches == 1 and args.steps > 1:
        # resident kernel: the state never leaves the chip, HBM is not the roof.  Report against the fp64 pipe
        # (148 SMs x 64 FMA lanes x 2 flop x 1.965 GHz; 26 FMA-class instructions per half-update).
        line["roofline"] = {"bound": "alu", "achieved": 2 * fp64_rate / 1e12, "peak": 2 * fp64_peak / 1e12,
                            "unit": "TFLOP/s", "frac": fp64_rate / fp64_peak, "traffic": None,
                            "kernel": "resident_kernel", "steps_per_launch": steps_per_launch,
                            "note": "whole time loop in one launch, state in shared memory; bounded by the serial "
                                    "latency of a half-update plus one barrier (small lattices) or by the "
                                    "shared-memory and fp64 pipes of the SM (DESIGN.md 5.2)",
                            "peak_source": "derived: 148 SMs x 64 fp64 FMA/clk x 1.965 GHz (B200_PROFILING.md unit counts)"}
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(W.get(args.workload))
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--workload", type=int, default=4,
                    help="BASELINE.json config index (default 4); 5 = the paper's own Table 1 run (context)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--variant", type=int, default=0, help="0 auto, 1 split, 2 fused tiles, 3 sweep, 4 resident")
    ap.add_argument("--tile-rows", type=int, default=0)
    ap.add_argument("--sweep-steps", type=int, default=0, help="steps fused per launch (0 auto)")
    ap.add_argument("--ctas", type=int, default=0, help="persistent CTAs of the sweep kernel (0 auto)")
    ap.add_argument("--precision", type=int, default=0, choices=[0, 1, 2],
                    help="0 fp64 (the metric); 1 fp32 storage / fp64 arithmetic, 2 fp32 throughout (NEXT-4 variants, "
                         "two launches per step; reported with dtype f32 -- not the BASELINE metric)")
    ap.add_argument("--sweep-threads", type=int, default=0, help="threads per CTA of the sweep kernel (0 auto)")
    ap.add_argument("--res-ctas", type=int, default=0, help="slabs of the resident kernel (0 auto)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--ref-budget", type=float, default=2.5e9,
                    help="--impl reference: grid-point updates of the bounded oracle sample (steps + warmup together)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
