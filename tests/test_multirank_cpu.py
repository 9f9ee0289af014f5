"""N > 1 host logic on CPU: world_size 2, gloo backend, rendezvous on 127.0.0.1 (no GPU needed).

The path shards with no data-path collective; what has to be right is the plumbing
bench.py uses: sharding, barrier, max-over-ranks timing and the whole-job rate."""
import json
import os
import socket
import subprocess
import sys

from paper_1401_6047_b200 import multi, workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shard_systems_partitions_every_batch():
    for n in (1, 2, 5, 8, 512):
        for world in (1, 2, 3, 8):
            seen = []
            for r in range(world):
                seen += list(multi.shard_systems(n, r, world))
            assert seen == list(range(n))
            sizes = [len(multi.shard_systems(n, r, world)) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1


def test_shard_workload_keeps_lattice_and_parameters():
    w = W.config3()
    a, b = multi.shard_workload(w, 0, 2), multi.shard_workload(w, 1, 2)
    assert a.grid.n_batch == b.grid.n_batch == 256 and a.grid.dt == w.grid.dt
    assert a.params[0] is w.params[0] and b.params[0] is w.params[256]
    assert max(a.n_steps, b.n_steps) == w.n_steps


def test_replicas_are_distinct_parameter_points():
    assert multi.replica_workload(4, 0).params[0].E_dc == W.config4().params[0].E_dc
    assert multi.replica_workload(4, 3).params[0].E_dc == W.config4().params[0].E_dc + 0.03


def test_world_size_2_gloo():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "tests", "_rank_worker.py")]
    env = dict(os.environ, OMP_NUM_THREADS="1")
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    line = [ln for ln in res.stdout.splitlines() if ln.startswith("{")][-1]
    d = json.loads(line)
    assert d["world"] == 2 and d["e_dc_rank0"] == 1.0
    assert d["t_max"] >= d["el_rank0"] + 0.005              # the max picked the slower rank
    assert d["units_total"] == 5 * 7 * 40 * 20
    assert abs(d["rate"] - d["units_total"] / d["t_max"]) <= 1e-9 * d["rate"]
    # every system was advanced by exactly one rank: compare with a single-process oracle run
    from oracle import OracleSim
    batch = W.random_batch(n_batch=5, N=6, M1=40, dt=0.004, seed=9, periods=0.05)
    for i, p in enumerate(batch.params):
        sim = OracleSim(6, 40, 0.004, p)
        sim.init_equilibrium()
        sim.step(20)
        assert sim.observables().v_dr == d["v"][i]
