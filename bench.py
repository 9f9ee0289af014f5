#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200 hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 4] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is one leap-frog time step of the whole hot path (whole-grid update, fractional-grid update,
reductions, bookkeeping -- SURVEY.md 8(a) rows S1-S9) over the workload's lattice.  Headline workload:
BASELINE.json configs[4] ("bandwidth stress", 512 harmonics x 32001 phi_y points, 525 MB of state), the
configuration the HBM-roofline target is quoted on.  The other four BASELINE configs are timed in the same
process for a bounded number of steps and reported under "configs".  Prints ONE JSON line (rank 0).

Timing: W untimed warm-up steps, then blocks of EXACTLY K steps, each bracketed by a barrier and a device
synchronise and timed with CUDA events on the solver's stream; at least 5 blocks, and more until the
in-process NVML sampler holds at least 5 clock samples taken under load; the reported time is the MEDIAN
block (max over ranks).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1401_6047_b200 import workloads as W  # noqa: E402
from paper_1401_6047_b200.multi import dist_env, replica_workload, max_over_ranks as _max_over_ranks  # noqa: E402

METRIC = "fp64 grid-point updates/s per time step; achieved HBM GB/s vs B200 peak"   # BASELINE.json "metric"
UNIT = "updates/s"
BYTES_PER_UPDATE = 64.0       # a_h, b_h, a_f, b_f each read once and written once
FP64_PER_HALF_UPDATE = 23     # cn_partial + cn_complete + differences, src, mu (bte_device.cuh)
FP64_PEAK_INSTR = 148 * 64 * 1.965e9   # DFMA-class thread-instructions/s: 148 SMs x 64 lanes x max SM clock
VARIANT_KERNEL = {1: "half_update_kernel (two launches per step)", 2: "fused_step_kernel", 3: "sweep_kernel",
                  5: "warpsweep_kernel"}
VARIANT_BYTES = {1: 96.0, 2: 64.0, 3: 64.0, 5: 64.0}   # HBM bytes per lattice point and launch group


def measured_peak_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def recorded_traffic(workload_name, kernel, steps_per_launch):
    """dram bytes per launch of the dominant kernel from the committed ncu --set full capture."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        with open(p) as f:
            d = json.load(f)
        e = d.get(workload_name, {})
        key = f"S{int(round(steps_per_launch))}"
        if kernel.startswith("warpsweep"):
            key = "warp" + key
        return e.get(key, {}).get("dram_bytes_per_launch")
    except Exception:
        return None


# ---------------------------------------------------------------------------------------------------
# clocks and throttle reasons DURING the timed region
# ---------------------------------------------------------------------------------------------------
class ClockSampler:
    """NVML in-process: SM clock, power and clock-event reasons every ~2 ms while `active`.  Falls back to one
    `nvidia-smi` process polling every 20 ms; if both fail the error text is kept in the record."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown"}

    def __init__(self, cuda_index):
        self.idx = cuda_index
        self.samples = []          # (sm_mhz, power_w, reasons bitmask)
        self.sm_max = None
        self.active = False
        self.err = None
        self._stop = False
        self._thread = None
        self._smi = None
        self._h = None
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            h = None
            try:
                pr = torch.cuda.get_device_properties(cuda_index)
                bus = "%08x:%02x:%02x.0" % (getattr(pr, "pci_domain_id", 0), pr.pci_bus_id, pr.pci_device_id)
                h = pynvml.nvmlDeviceGetHandleByPciBusId(bus.encode())
            except Exception:
                vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
                ids = [x for x in vis.split(",") if x.strip().isdigit()]
                h = pynvml.nvmlDeviceGetHandleByIndex(int(ids[cuda_index]) if cuda_index < len(ids) else cuda_index)
            self._nv, self._h = pynvml, h
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            self._reason_fn = getattr(pynvml, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
                getattr(pynvml, "nvmlDeviceGetCurrentClocksThrottleReasons")
            self._thread = threading.Thread(target=self._loop, daemon=True)
            self._thread.start()
        except Exception as e:   # no NVML: nvidia-smi in the background
            self.err = f"nvml: {type(e).__name__}: {e}"
            self._h = None
            self._start_smi()

    def _loop(self):
        nv, h = self._nv, self._h
        while not self._stop:
            if self.active:
                try:
                    sm = float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                    pw = nv.nvmlDeviceGetPowerUsage(h) / 1000.0
                    rs = int(self._reason_fn(h))
                    if self.active:
                        self.samples.append((sm, pw, rs))
                except Exception as e:
                    self.err = f"nvml: {type(e).__name__}: {e}"
                time.sleep(0.002)
            else:
                time.sleep(0.0005)

    def _start_smi(self):
        q = "clocks.sm,clocks.max.sm,power.draw"
        try:
            self._smi = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-lms", "20",
                                          "-i", str(self.idx)], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
        except Exception as e:
            self.err = (self.err or "") + f"; nvidia-smi: {e}"

    def n(self):
        return len(self.samples)

    def finish(self):
        self._stop = True
        reasons_smi = None
        if self._smi is not None:   # everything the background poller saw (the whole run, not only the timed blocks)
            time.sleep(0.05)
            self._smi.terminate()
            try:
                out, err = self._smi.communicate(timeout=5)
            except Exception:
                self._smi.kill()
                out, err = "", "killed"
            for line in out.strip().splitlines():
                parts = [x.strip() for x in line.split(",")]
                try:
                    self.samples.append((float(parts[0]), float(parts[2]), 0))
                    self.sm_max = float(parts[1])
                except (ValueError, IndexError):
                    pass
            if err.strip():
                self.err = (self.err or "") + "; nvidia-smi: " + err.strip()[:200]
            try:   # throttle reasons in a second query (field names differ between driver generations)
                for names in ("clocks_event_reasons", "clocks_throttle_reasons"):
                    q = ",".join(f"{names}.{k}" for k in ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"))
                    r = subprocess.run(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader", "-i", str(self.idx)],
                                       capture_output=True, text=True, timeout=10)
                    if r.returncode == 0 and r.stdout.strip():
                        vals = [x.strip().lower() for x in r.stdout.strip().split(",")]
                        reasons_smi = [k for k, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown",
                                                          "sw_power_cap"), vals) if v.startswith("active")]
                        break
            except Exception as e:
                self.err = (self.err or "") + f"; nvidia-smi reasons: {e}"
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": None, "samples": 0,
                    "error": self.err or "no samples"}
        mask = 0
        for _, _, r in self.samples:
            mask |= r
        reasons = sorted(v for k, v in self.REASONS.items() if mask & k) if reasons_smi is None else reasons_smi
        out = {"sm_mhz": statistics.median(x[0] for x in self.samples), "sm_mhz_min": min(x[0] for x in self.samples),
               "sm_max_mhz": self.sm_max,
               "power_w_max": max(x[1] for x in self.samples), "samples": len(self.samples), "reasons": reasons,
               "how": "NVML in-process, ~2 ms period, inside the timed blocks only" if self._h is not None else
                      "nvidia-smi -lms 20 for the whole run"}
        if self.err:
            out["error"] = self.err
        return out


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


def config_of(w):
    """The `config` object of the JSON line: identical in both arms."""
    return {"workload": w.name, **w.describe()}


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
            "data": "synthetic", "config": config_of(w),
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
class Ctx:
    """Device, rank plumbing and the clock sampler shared by all timed legs."""

    def __init__(self, args):
        import torch
        import torch.distributed as dist
        self.torch, self.dist = torch, dist
        self.rank, self.world, self.local = dist_env()
        # under torchrun (RANK set) the NCCL process group is brought up even for a single rank, so that the barrier and
        # the max-over-ranks reduction of the timing run through NCCL exactly as they do for N > 1
        if self.world > 1 or os.environ.get("RANK") is not None:
            dist.init_process_group("nccl", device_id=torch.device(f"cuda:{self.local}"))
        torch.cuda.set_device(self.local)
        self.dev = f"cuda:{self.local}"
        self.args = args
        self.sampler = ClockSampler(self.local) if self.rank == 0 else None

    def barrier(self):
        if self.dist.is_initialized():
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def max_over_ranks(self, x):
        return _max_over_ranks(x, self.dev)


def apply_options(s, args, sweep_steps=None, variant=None):
    v = args.variant if variant is None else variant
    if v:
        s.set_option("variant", v)
    if args.tile_rows:
        s.set_option("tile_rows", args.tile_rows)
    ss = args.sweep_steps if sweep_steps is None else sweep_steps
    if ss:
        s.set_option("sweep_steps", ss)
    if args.ctas:
        s.set_option("sweep_ctas", args.ctas)
    if args.res_ctas:
        s.set_option("resident_ctas", args.res_ctas)
    if args.res_halo:
        s.set_option("resident_halo", args.res_halo)
    if args.sweep_threads:
        s.set_option("sweep_threads", args.sweep_threads)


def timed_blocks(cx, s, w, steps, k_done, min_blocks, sample_clocks, max_blocks=400, max_seconds=4.0):
    """Blocks of exactly `steps` steps; returns (median ms, list of ms, launches per block, steps done)."""
    torch = cx.torch
    e0 = torch.cuda.Event(enable_timing=True)
    e1 = torch.cuda.Event(enable_timing=True)
    times, launches = [], None
    t_start = time.perf_counter()
    n0 = cx.sampler.n() if (cx.sampler and sample_clocks) else 0
    while True:
        cx.barrier()
        l0 = s.launch_count()
        if cx.sampler and sample_clocks:
            cx.sampler.active = True
        e0.record(s.stream)
        s.step(steps)
        e1.record(s.stream)
        cx.barrier()
        if cx.sampler and sample_clocks:
            cx.sampler.active = False
        times.append(cx.max_over_ranks(e0.elapsed_time(e1)))
        launches = s.launch_count() - l0
        k_done += steps
        enough = len(times) >= min_blocks
        if enough and sample_clocks and cx.sampler and cx.world == 1:
            enough = cx.sampler.n() - n0 >= 5 or cx.sampler._h is None
        if enough or len(times) >= max_blocks or time.perf_counter() - t_start > max_seconds:
            break
    return statistics.median(times), times, launches, k_done


def hbm_roofline(w, updates_per_block, ms, launches, steps, variant, S, peak, peak_src, precision=0):
    """One launch of a sweep kernel advances every active system by S time steps in one pass over the state
    (temporal blocking): what that launch must move is the state read once and written once = 64 B per lattice
    point PER LAUNCH; the other variants move 96 / 64 B per point per step."""
    per_launch_s = ms * 1e-3 / max(1, launches)
    alg_bytes = VARIANT_BYTES[variant] * updates_per_block / steps       # per launch (sweep) / per step (others)
    if precision != 0:
        alg_bytes *= 0.5                                                  # fp32 pairs in HBM
    if variant in (3, 5):
        achieved = alg_bytes / per_launch_s / 1e9
    else:
        achieved = alg_bytes * steps / (ms * 1e-3) / 1e9
    effective = BYTES_PER_UPDATE * updates_per_block / (ms * 1e-3) / 1e9
    fp64_rate = 2 * FP64_PER_HALF_UPDATE * updates_per_block / (ms * 1e-3)
    kernel = VARIANT_KERNEL[variant]
    return {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
            "frac_of_nominal_8TBs": achieved / 8000.0,
            "traffic": recorded_traffic(w.name, kernel, S) if variant in (3, 5) else None,
            "kernel": kernel, "steps_per_launch": steps / max(1, launches),
            "algorithmic_bytes_per_launch": alg_bytes, "peak_source": peak_src,
            "effective_gbs_at_64B_per_update": effective,
            "effective_note": ("temporal blocking: one pass over the state advances steps_per_launch time steps, so "
                               "the one-step-per-pass figure (64 B per update) can exceed the HBM peak; 'achieved' "
                               "counts what a launch really has to move"),
            "fp64_pipe_frac": fp64_rate / FP64_PEAK_INSTR,
            "bound_note": ("SURVEY 8(d) counts HBM bytes, so 'bound' stays hbm; a pass of S >= 2 steps moves 64 / S B per "
                           "update by design and is limited by the fp64 pipe and the issue slots (fp64_pipe_frac; ncu: "
                           "profiles/r02f, r02c), the HBM-bound form of the same workload is one_step_per_pass")
            if S >= 2 else None}


def alu_roofline(updates_per_block, ms, steps, launches):
    fp64_rate = 2 * FP64_PER_HALF_UPDATE * updates_per_block / (ms * 1e-3)
    return {"bound": "alu", "achieved": 2 * fp64_rate / 1e12, "peak": 2 * FP64_PEAK_INSTR / 1e12, "unit": "TFLOP/s",
            "frac": fp64_rate / FP64_PEAK_INSTR, "traffic": None, "kernel": "resident_kernel",
            "steps_per_launch": steps / max(1, launches),
            "note": "whole time loop in one launch, state in shared memory; bounded by the serial latency of a "
                    "half-update plus one barrier (small lattices) or by the shared-memory and fp64 pipes of the SM "
                    "(DESIGN.md 5.2)",
            "peak_source": "derived: 148 SMs x 64 fp64 FMA/clk x 1.965 GHz (B200_PROFILING.md unit counts), "
                           f"{FP64_PER_HALF_UPDATE} fp64 instructions per half-update"}


def time_workload(cx, w, steps, warmup, min_blocks, sample_clocks, one_pass=False, precision=None):
    """Device-resident measurement of one workload: state already in HBM when the timed region starts."""
    from paper_1401_6047_b200 import Solver
    import copy
    args = cx.args
    if precision is not None and precision != args.precision:
        args = copy.copy(args)
        args.precision = precision
    peak, peak_src = measured_peak_gbs()
    s = Solver(w.grid, w.params, device=cx.dev, precision=args.precision)
    apply_options(s, args)
    s.init_equilibrium()
    warm = max(3, warmup)
    s.step(warm)
    ms, times, launches, k_done = timed_blocks(cx, s, w, steps, warm, min_blocks, sample_clocks)
    # the work of the median block (systems freeze at their budgets): take the first block's span -- all blocks
    # of a bounded run lie before the first budget, which bench.py checks below
    updates = w.updates_between(warm, warm + steps)
    last_updates = w.updates_between(k_done - steps, k_done)
    obs = s.observables()[0]
    variant = s.get_option("effective_variant") if args.precision != 2 else 1
    S = s.get_option("effective_sweep_steps") if variant in (3, 5) else 1
    resident = launches == 1 and steps > 1 and args.precision == 0
    out = {"value": updates * cx.world / (ms * 1e-3), "ms_per_step": ms / steps, "steps": steps,
           "blocks": len(times), "ms_min_max": [min(times) / steps, max(times) / steps],
           "gpu_launches": launches, "same_work_every_block": updates == last_updates,
           "roofline": (alu_roofline(updates, ms, steps, launches) if resident else
                        hbm_roofline(w, updates, ms, launches, steps, variant, S, peak, peak_src, args.precision)),
           "check": {"norm": obs.norm, "v_dr": obs.v_dr, "step": obs.step}}
    out["kernel"] = out["roofline"]["kernel"]
    # The same workload with ONE time step per pass (sweep_steps = 1): the plain HBM-bound form of the step
    # kernel, whose 64 B per update is what SURVEY 8(d) counts -- reported beside the headline so that the
    # HBM-roofline fraction of the memory-bound variant is measured in the same run (not the headline value).
    if one_pass and not resident and not args.sweep_steps and args.variant in (0, 3, 5) and args.precision == 0:
        s.set_option("variant", 3)
        s.set_option("sweep_steps", 1)
        k1 = max(20, min(200, steps))
        s.step(3)
        ms1, t1, l1, k_end = timed_blocks(cx, s, w, k1, k_done + 3, 3, False)
        upd1 = w.updates_between(k_done + 3, k_done + 3 + k1)
        gbs = BYTES_PER_UPDATE * upd1 / (ms1 * 1e-3) / 1e9
        out["roofline"]["one_step_per_pass"] = {
            "steps": k1, "blocks": len(t1), "launches": l1, "ms_per_step": ms1 / k1,
            "updates_per_s": upd1 * cx.world / (ms1 * 1e-3), "achieved_gbs": gbs, "frac": gbs / peak,
            "frac_of_nominal_8TBs": gbs / 8000.0,
            "note": "same workload, sweep_steps = 1: the HBM-bound form (64 B of HBM traffic per update), "
                    "measured in this run"}
    s.destroy()
    del s
    cx.torch.cuda.empty_cache()
    return out, updates


def run_e2e(cx, w, steps):
    """End to end through the public API with HOST buffers.  The state (a, b on both grids of every system)
    starts in pinned HOST memory and ends there.  Timed: bte_create (table upload H2D) -> bte_set_state_batch x 2
    (H2D of the inputs) -> bte_step(K) -> bte_observables -> bte_get_state_batch x 2 (D2H of the result)."""
    from paper_1401_6047_b200 import Solver
    torch, args = cx.torch, cx.args
    nb, shape = w.grid.n_batch, (w.grid.n_harm + 1, w.grid.n_phiy)
    host_in = torch.empty((2, 2, nb) + shape, dtype=torch.float64).pin_memory()    # [grid][a|b][system][n][m]
    host_out = torch.empty((2, 2, nb) + shape, dtype=torch.float64).pin_memory()
    hin, hout = host_in.numpy(), host_out.numpy()
    s1 = Solver(w.grid, w.params, device=cx.dev, precision=args.precision)   # untimed: the t = 0 state on the host
    s1.init_equilibrium()
    for g in (0, 1):
        s1.get_state_batch(g, hin[g, 0], hin[g, 1])
    s1.destroy()
    del s1
    cx.barrier()
    t0 = time.perf_counter()
    s2 = Solver(w.grid, w.params, device=cx.dev, precision=args.precision)
    apply_options(s2, args)
    for g in (0, 1):
        s2.set_state_batch(g, hin[g, 0], hin[g, 1])
    s2.step(steps)
    obs2 = s2.observables()
    for g in (0, 1):
        s2.get_state_batch(g, hout[g, 0], hout[g, 1])
    torch.cuda.synchronize()
    e2e_s = cx.max_over_ranks(time.perf_counter() - t0)
    rows, pitch = shape[0], (shape[1] + 7) // 8 * 8
    state_bytes = nb * 2 * 2 * 8 * shape[0] * shape[1]
    h2d = nb * (8 * rows + 16 * pitch + 80) + state_bytes      # c_n, g_m, phi_m tables + constants + state
    d2h = nb * 96 + state_bytes                                 # observables + state
    val = w.updates_between(0, steps) * cx.world / e2e_s
    s2.destroy()
    return {"value": val, "unit": UNIT, "h2d_bytes_per_step": h2d / steps, "d2h_bytes_per_step": d2h / steps,
            "seconds": e2e_s, "steps": steps,
            "what": "state in pinned host memory -> bte_create + bte_set_state_batch (H2D) + bte_step(K) + "
                    "bte_observables + bte_get_state_batch (D2H) -> pinned host memory"}, obs2[0].step


# bounded runs of the other BASELINE configs: (index, steps per block, warm-up steps)
SECONDARY = [(3, 240, 12), (2, 2000, 8), (1, 4000, 8), (0, 4000, 8)]


def run_ours(args):
    cx = Ctx(args)
    w = replica_workload(args.workload, cx.rank)
    pts_all = w.points_per_system * w.grid.n_batch

    main, updates = time_workload(cx, w, args.steps, args.warmup, 5, True, one_pass=True)
    clocks = cx.sampler.finish() if cx.sampler else None
    e2e, e2e_step = run_e2e(cx, w, args.steps)

    configs = {}
    if not args.no_other_configs and cx.world == 1 and args.precision == 0:
        for idx, k, warm in SECONDARY:
            if idx == args.workload:
                continue
            wi = W.get(idx)
            r, _ = time_workload(cx, wi, min(k, wi.n_steps), warm, 3, False, one_pass=(idx == 3))
            r["config"] = config_of(wi)
            configs[wi.name] = r

    # NEXT-4 beside the headline, never as the headline: the same workload with the state stored as fp32 pairs (the
    # paper's storage precision) and fp64 arithmetic, through the same production kernel
    other_precisions = {}
    if not args.no_other_configs and cx.world == 1 and args.precision == 0 and not args.sweep_steps and args.variant == 0:
        r, _ = time_workload(cx, w, min(240, args.steps), 6, 3, False, precision=1)
        r["dtype"] = "f32 storage / f64 arithmetic"
        other_precisions["f32_storage"] = r

    if cx.rank != 0:
        if cx.dist.is_initialized():
            cx.dist.destroy_process_group()
        return 0

    line = {
        "metric": METRIC, "value": main["value"], "unit": UNIT, "n_gpus": cx.world, "steps": args.steps,
        "warmup": max(3, args.warmup), "ms_per_step": main["ms_per_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None,
        "dtype": ("f64", "f32 storage / f64 arithmetic", "f32")[args.precision], "data": "synthetic",
        "config": config_of(w),
        "config_detail": {"state_bytes": 32 * pts_all,
                          "l2_policy": (f"inputs larger than L2 ({32 * pts_all / 1e6:.0f} MB state vs 126 MB L2)"
                                        if 32 * pts_all > 2.6e8 else
                                        "state fits on chip / in L2: resident regime, reported as such"),
                          "multi_gpu": "independent replicas, one system per rank, no collective",
                          "paper_convention_updates_per_s": main["value"] * w.grid.n_harm / (w.grid.n_harm + 1),
                          "timing": f"median of {main['blocks']} blocks of exactly {args.steps} steps, CUDA events on the "
                                    "solver's stream, barrier + synchronise around every block, max over ranks",
                          "ms_per_step_min_max": main["ms_min_max"]},
        "roofline": main["roofline"],
        "e2e": e2e,
        "gpu_launches": main["gpu_launches"],
        "clocks": clocks,
        "check": dict(main["check"], e2e_step=e2e_step),
        "configs": configs, "other_precisions": other_precisions,
    }
    if w.name == "paper_table1":
        # the paper's own workload and MLUPS convention (n-harmonics x g-grid x steps / time, L328); its number is
        # fp32 on a GTX680 -- ours is fp64 unless --precision says otherwise: context, not the target
        mlups = main["value"] * w.grid.n_harm / (w.grid.n_harm + 1) / 1e6
        line["vs_baseline"] = mlups / W.PAPER_TABLE1_MLUPS_K6
        line["config_detail"]["paper_mlups"] = {"ours": mlups, "paper_K6_GTX680_fp32": W.PAPER_TABLE1_MLUPS_K6,
                                                "paper_cpu_1_thread_fp32": 9.0, "source": "PAPER.md:L315-328 (Table 1)"}
    if cx.world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(W.get(args.workload))
    print(json.dumps(line), flush=True)
    if cx.dist.is_initialized():
        cx.dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=600)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--workload", type=int, default=4,
                    help="BASELINE.json config index (default 4); 5 = the paper's own Table 1 run (context)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--variant", type=int, default=0,
                    help="0 auto, 1 split, 2 fused tiles, 3 sweep (shared-memory rings), 4 resident, 5 register-pipelined sweep")
    ap.add_argument("--tile-rows", type=int, default=0)
    ap.add_argument("--sweep-steps", type=int, default=0, help="steps fused per launch (0 auto)")
    ap.add_argument("--ctas", type=int, default=0, help="persistent CTAs of the sweep kernel (0 auto)")
    ap.add_argument("--precision", type=int, default=0, choices=[0, 1, 2],
                    help="0 fp64 (the metric); 1 fp32 storage / fp64 arithmetic, 2 fp32 throughout (NEXT-4 variants, "
                         "reported with dtype f32 -- not the BASELINE metric)")
    ap.add_argument("--sweep-threads", type=int, default=0, help="threads per CTA of the sweep kernel (0 auto)")
    ap.add_argument("--res-ctas", type=int, default=0, help="slabs of the resident kernel (0 auto)")
    ap.add_argument("--res-halo", type=int, default=0, help="halo columns of the resident kernel's grid mode (0 auto)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="time the headline workload only")
    ap.add_argument("--ref-budget", type=float, default=2.5e9,
                    help="--impl reference: grid-point updates of the bounded oracle sample (steps + warmup together)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
