"""Worker of tests/test_multirank_cpu.py: one rank of a world_size-2 gloo job on CPU.

Runs the N > 1 plumbing of bench.py (paper_1401_6047_b200.multi) with the CPU oracle standing in for the
GPU step: shard the work, barrier, time, max over ranks, whole-job rate; rank 0 prints one JSON line."""
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import torch.distributed as dist  # noqa: E402

from oracle import OracleSim  # noqa: E402
from paper_1401_6047_b200 import multi, workloads as W  # noqa: E402


def main():
    dist.init_process_group("gloo")
    rank, world, _ = multi.dist_env()
    assert world == dist.get_world_size() and rank == dist.get_rank()
    # (a) weak scaling: one replica per rank, distinct parameter points
    w = multi.replica_workload(0, rank)
    e_dc = w.params[0].E_dc
    # (b) a batch sharded over ranks: every system exactly once
    batch = W.random_batch(n_batch=5, N=6, M1=40, dt=0.004, seed=9, periods=0.05)
    mine = multi.shard_workload(batch, rank, world)
    steps = 20
    multi.barrier()
    t0 = time.perf_counter()
    v = []
    for p in mine.params:
        sim = OracleSim(mine.grid.n_harm, mine.grid.n_phiy, mine.grid.dt, p)
        sim.init_equilibrium()
        sim.step(steps)
        v.append(sim.observables().v_dr)
    el = time.perf_counter() - t0 + 0.01 * (rank + 1)          # rank 1 is "slower": the max must pick it
    multi.barrier()
    units = len(mine.params) * (mine.grid.n_harm + 1) * mine.grid.n_phiy * steps
    rate, t_max = multi.whole_job_rate(units, el)
    owned = [0.0] * batch.grid.n_batch
    for i, x in zip(multi.shard_systems(batch.grid.n_batch, rank, world), v):
        owned[i] = x
    import torch
    t = torch.tensor(owned, dtype=torch.float64)
    dist.all_reduce(t)                                          # test-only gather of the per-system results
    if rank == 0:
        print(json.dumps({"world": world, "e_dc_rank0": e_dc, "rate": rate, "t_max": t_max, "el_rank0": el,
                          "units_total": multi.sum_over_ranks(units), "v": t.tolist()}), flush=True)
    else:
        multi.sum_over_ranks(units)
        assert abs(e_dc - (1.0 + 0.01 * rank)) < 1e-15
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
