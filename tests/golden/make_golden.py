#!/usr/bin/env python
"""Writes tests/golden/config<i>_full.json: expected values of the BASELINE.json configs at FULL length.

    python tests/golden/make_golden.py [0 1 2 3 4]

Every number comes from the CPU oracle (oracle/bte_oracle.cpp) run on the workload generator's inputs --
this script imports nothing of the CUDA path.  The paper prints no numerical value of f, v_dr or A for any
run (PAPER.md: Fig. 3-5 are plots, Table 1 L315-321 holds timings only), so there is no paper-printed
fixture to store; what pins the oracle itself is tests/test_oracle_pins.py (closed forms, invariants).
These files only spare the GPU test-suite the minutes of CPU time a full-length oracle run takes:
tests/test_gpu_full_size.py runs the same configs at full length through the C ABI in the launch
configuration bench.py times and compares

  * the observables of bte_obs (step, norm eq. 12, v_dr eq. 20, the running sums of eq. 17, window, edge leak),
  * the state at SAMPLES seeded lattice points per grid (whole / fractional), a and b,

against the values stored here (tolerances of DESIGN.md C15).  Config 3 stores 8 of its 512 systems
(indices 0, 73, 146, ...), each run to its own step budget.
"""
from __future__ import annotations

import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import OracleSim, max_threads  # noqa: E402
from paper_1401_6047_b200 import workloads as W  # noqa: E402  (input generator only: no method arithmetic)

SAMPLES = 96
SYSTEMS_CONFIG3 = list(range(0, 512, 73))


def sample_points(n_rows: int, n_cols: int, seed: int):
    """Seeded lattice points, biased towards where f lives (low harmonics, centre columns) but also
    covering edges and corners."""
    rng = np.random.default_rng(seed)
    pts = {(0, 0), (0, n_cols - 1), (n_rows - 1, 0), (n_rows - 1, n_cols - 1), (1, n_cols // 2), (0, n_cols // 2)}
    while len(pts) < SAMPLES:
        n = int(min(n_rows - 1, abs(rng.normal(0.0, max(2.0, n_rows / 6.0)))))
        m = int(np.clip(rng.normal(n_cols / 2.0, n_cols / 6.0), 0, n_cols - 1))
        if rng.random() < 0.25:
            n, m = int(rng.integers(0, n_rows)), int(rng.integers(0, n_cols))
        pts.add((n, m))
    return sorted(pts)


def run_system(w, i, n_steps, threads):
    p = w.params[i]
    sim = OracleSim(w.grid.n_harm, w.grid.n_phiy, w.grid.dt, p, threads=threads)
    sim.init_equilibrium()
    sim.step(n_steps)
    o = sim.observables()
    rec = {"system": i, "n_steps": int(n_steps), "params": vars(p).copy(),
           "obs": {k: getattr(o, k) for k in ("step", "t", "norm", "v_dr", "sum_v_dt", "sum_vcos_dt",
                                               "sum_vsin_dt", "window", "edge_leak")}}
    pts = sample_points(w.grid.n_harm + 1, w.grid.n_phiy, seed=1401 + 6047 * i)
    scale = 0.0
    grids = []
    for g in (0, 1):
        a, b = sim.get_state(g)
        scale = max(scale, float(np.abs(a).max()), float(np.abs(b).max()))
        grids.append({"a": [float(a[n, m]).hex() for n, m in pts], "b": [float(b[n, m]).hex() for n, m in pts]})
    rec["points"] = [[int(n), int(m)] for n, m in pts]
    rec["state"] = grids
    rec["max_abs_f"] = scale
    sim.close()
    return rec


def main():
    which = [int(x) for x in sys.argv[1:]] or [0, 1, 2, 3, 4]
    threads = max_threads()
    for idx in which:
        w = W.get(idx)
        t0 = time.time()
        systems = SYSTEMS_CONFIG3 if w.grid.n_batch > 1 else [0]
        recs = []
        for i in systems:
            tot = w.params[i].n_steps_total
            n = w.n_steps if tot == 0 else max(w.n_steps, tot)   # run past the budget: the system must freeze
            recs.append(run_system(w, i, n, threads))
        out = {"_written_by": "tests/golden/make_golden.py (CPU oracle only)", "workload": w.name,
               "n_harm": w.grid.n_harm, "n_phiy": w.grid.n_phiy, "n_batch": w.grid.n_batch, "dt": w.grid.dt,
               "n_steps": int(w.n_steps), "systems": recs}
        path = os.path.join(HERE, f"config{idx}_full.json")
        with open(path, "w") as f:
            json.dump(out, f, indent=1)
        print(f"config {idx}: {len(recs)} system(s), {time.time() - t0:.0f} s -> {path}", flush=True)


if __name__ == "__main__":
    main()
