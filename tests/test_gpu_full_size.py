"""Full-size parity: every BASELINE.json config at FULL length through the C ABI, in the launch configuration
bench.py times (automatic variant selection), against oracle values stored by tests/golden/make_golden.py
(a script that calls only oracle/).  Compared: all observables of the stored systems and the state at 96
seeded lattice points per grid -- tolerances of DESIGN.md C15 (1e-12 max|f| for the state, 1e-10 for the
observables).  Run on the B200 box: pytest -m gpu."""
import json
import os
from types import SimpleNamespace

import numpy as np
import pytest

from paper_1401_6047_b200 import workloads as W

from parity_util import TOL_STATE, assert_obs_close

pytestmark = pytest.mark.gpu
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def load(idx):
    path = os.path.join(GOLDEN, f"config{idx}_full.json")
    if not os.path.exists(path):
        pytest.skip(f"{path} not generated (python tests/golden/make_golden.py {idx})")
    with open(path) as f:
        return json.load(f)


def run_and_compare(idx, variant=0, sweep_steps=0):
    from paper_1401_6047_b200 import Solver
    gold = load(idx)
    w = W.get(idx)
    assert (gold["n_harm"], gold["n_phiy"], gold["n_batch"], gold["dt"]) == \
        (w.grid.n_harm, w.grid.n_phiy, w.grid.n_batch, w.grid.dt)
    s = Solver(w.grid, w.params)
    s.set_option("variant", variant)
    s.set_option("sweep_steps", sweep_steps)
    s.init_equilibrium()
    n = gold["systems"][0]["n_steps"]
    assert all(r["n_steps"] == n for r in gold["systems"])
    s.step(n)
    obs = s.observables()
    worst = 0.0
    for rec in gold["systems"]:
        i = rec["system"]
        p = w.params[i]
        for k, v in rec["params"].items():                      # same generated inputs on both sides
            assert getattr(p, k) == v, (i, k)
        what = f"{w.name}[{i}] full length ({n} steps)"
        assert_obs_close(obs[i], SimpleNamespace(**rec["obs"]), p, w.grid.dt, what=what)
        pts = np.array(rec["points"])
        for g in (0, 1):
            a, b = s.get_state(i, g)
            for name, arr in (("a", a), ("b", b)):
                ref = np.array([float.fromhex(x) for x in rec["state"][g][name]])
                got = arr[pts[:, 0], pts[:, 1]]
                assert np.isfinite(got).all(), what
                err = np.abs(got - ref).max()
                worst = max(worst, err / rec["max_abs_f"])
                assert err <= TOL_STATE * rec["max_abs_f"], f"{what}: grid {g} {name}: {err:.3e} vs max|f| {rec['max_abs_f']:.3e}"
            assert np.all(b[0] == 0.0), f"{what}: b_0 must stay exactly 0 (eq. 23)"
    s.destroy()
    return worst


def test_config0_full_length():
    run_and_compare(0)


def test_config1_full_length():
    run_and_compare(1)


def test_config2_full_length():
    run_and_compare(2)


def test_config3_full_length_all_512_systems_advance():
    run_and_compare(3)


def test_config4_full_length():
    run_and_compare(4)


@pytest.mark.parametrize("idx", [3, 4])
@pytest.mark.parametrize("sweep_steps", [1, 2, 3])
def test_streaming_configs_full_length_every_sweep_depth(idx, sweep_steps):
    """Configs 3 (512 systems, step budgets: launches are cut at every budget boundary) and 4 at full length with
    1, 2 and 3 time steps per pass."""
    run_and_compare(idx, variant=3, sweep_steps=sweep_steps)


@pytest.mark.parametrize("idx", [3, 4])
@pytest.mark.parametrize("sweep_steps", [2, 3, 4])
def test_streaming_configs_full_length_warp_kernel(idx, sweep_steps):
    """The same through the warp kernel (variant 5: registers + tensor memory, bte_warpsweep.cuh); config 4 is what
    the automatic choice runs."""
    run_and_compare(idx, variant=5, sweep_steps=sweep_steps)


def test_config2_full_length_warp_kernel():
    """Config 2 (78 540 steps, 151 rows) through the warp kernel with graph replay."""
    run_and_compare(2, variant=5)


def test_config2_full_length_streaming_kernel():
    """Config 2 (78 540 steps) through the sweep kernel with graph replay instead of the resident kernel."""
    run_and_compare(2, variant=3)


@pytest.mark.parametrize("sweep_steps", [1, 2, 3])
def test_config1_full_length_streaming_kernel(sweep_steps):
    """The same 62 832 steps through the HBM-streaming sweep kernel (graph replay) instead of the resident one."""
    run_and_compare(1, variant=3, sweep_steps=sweep_steps)
