"""fp32 variants of the step (the paper ran in float throughout) against the oracle's
fp32 modes, and the paper's time-step floor in float (L328).  Run on the B200 box: pytest -m gpu."""
import numpy as np
import pytest

from paper_1401_6047_b200 import workloads as W

pytestmark = pytest.mark.gpu
EPS32 = float(np.finfo(np.float32).eps)


def run_pair(w, n_steps, precision, system=0, graph_steps=None):
    from paper_1401_6047_b200 import Solver
    from oracle import OracleSim
    s = Solver(w.grid, w.params, precision=precision)
    if graph_steps is not None:
        s.set_option("graph_steps", graph_steps)
    s.init_equilibrium()
    s.step(n_steps)
    sim = OracleSim(w.grid.n_harm, w.grid.n_phiy, w.grid.dt, w.params[system], threads=4, precision=precision)
    sim.init_equilibrium()
    sim.step(n_steps)
    return s, sim


@pytest.mark.parametrize("N,M1", [(2, 5), (9, 128), (21, 300)])
def test_fp32_arithmetic_is_bit_identical_to_the_float_oracle(N, M1):
    """precision 2: the same IEEE float operations in the same order on both sides.  What may differ: E(t) (cos of
    the two math libraries, rounded to float) and c_n (two Bessel routines, rounded to float) -- a last-bit difference
    of an fp64 value only rarely survives the rounding to fp32.  B = 0 and a dc field remove E(t) from the list."""
    w = W.small_case(N=N, M1=M1, dt=0.004, n_steps=40, E_omega=0.0, omega=0.0, avg_start=5)
    s, sim = run_pair(w, 40, 2)
    for g in (0, 1):
        a, b = s.get_state(0, g)
        ra, rb = sim.get_state(g)
        assert a.dtype == np.float64 and np.array_equal(a, a.astype(np.float32).astype(np.float64))
        same = np.mean(a == ra) * 0.5 + np.mean(b == rb) * 0.5
        scale = max(np.abs(ra).max(), np.abs(rb).max())
        worst = max(np.abs(a - ra).max(), np.abs(b - rb).max()) / scale
        assert same > 0.999 and worst <= 4 * EPS32, (g, same, worst)
    o, r = s.observables()[0], sim.observables()
    assert o.step == r.step and abs(o.v_dr - r.v_dr) <= 1e-6 * max(abs(r.v_dr), 0.05) and abs(o.norm - r.norm) <= 1e-6
    s.destroy()


@pytest.mark.parametrize("precision", [1, 2])
def test_fp32_modes_match_the_oracle_with_ac_field_and_budget(precision):
    """Crossed ac + dc fields, graph replay and plain launches, a step budget; tolerance: a few fp32 ulps of max|f|
    (fp32 storage + fp64 arithmetic differs from the oracle only where the two fp64 results straddle an fp32 rounding
    boundary; such one-ulp differences are damped by the contractive map)."""
    w = W.small_case(N=12, M1=190, dt=0.004, n_steps=150, avg_start=20)
    w.params[0].n_steps_total = 140
    for graph_steps in (0, 8):
        s, sim = run_pair(w, 150, precision, graph_steps=graph_steps)
        scale = max(np.abs(x).max() for g in (0, 1) for x in sim.get_state(g))
        for g in (0, 1):
            a, b = s.get_state(0, g)
            ra, rb = sim.get_state(g)
            assert max(np.abs(a - ra).max(), np.abs(b - rb).max()) <= 8 * EPS32 * scale, (precision, g)
            assert np.all(b[0] == 0.0)
        o, r = s.observables()[0], sim.observables()
        assert o.step == r.step == 140
        assert abs(o.v_dr - r.v_dr) <= 1e-5 * max(abs(r.v_dr), 0.05)
        assert abs(o.sum_vcos_dt - r.sum_vcos_dt) <= 1e-5 * max(abs(r.sum_vcos_dt), 0.05 * r.window)
        s.destroy()


@pytest.mark.parametrize("sweep_steps", [2, 3, 4])
@pytest.mark.parametrize("N,M1", [(40, 801), (97, 300), (33, 90)])
def test_fp32_storage_through_the_warp_kernel(N, M1, sweep_steps):
    """precision 1 on lattices of at least 32 rows runs the multi-step warp kernel with fp32 rows in HBM (half the bytes)
    and fp64 arithmetic; single steps (remainders) run the two-launch form.  Inside a pass the intermediate time levels stay
    fp64 in registers, so the result differs from the oracle (which rounds every half-update to fp32) by a few fp32 ulps of
    max|f| -- the same bound as the two-launch form."""
    from paper_1401_6047_b200 import Solver
    from oracle import OracleSim
    w = W.small_case(N=N, M1=M1, dt=0.004, n_steps=50, avg_start=7)
    s = Solver(w.grid, w.params, precision=1)
    s.set_option("sweep_steps", sweep_steps)
    s.set_option("graph_steps", 0)
    assert s.get_option("effective_variant") == 5
    s.init_equilibrium()
    n0 = s.launch_count()
    s.step(17); s.step(1); s.step(32)
    sim = OracleSim(w.grid.n_harm, w.grid.n_phiy, w.grid.dt, w.params[0], threads=4, precision=1)
    sim.init_equilibrium()
    sim.step(50)
    scale = max(np.abs(x).max() for g in (0, 1) for x in sim.get_state(g))
    for g in (0, 1):
        a, b = s.get_state(0, g)
        ra, rb = sim.get_state(g)
        assert np.array_equal(a, a.astype(np.float32).astype(np.float64))          # what is stored is fp32
        assert max(np.abs(a - ra).max(), np.abs(b - rb).max()) <= 8 * EPS32 * scale, (g,)
        assert np.all(b[0] == 0.0)
    o, r = s.observables()[0], sim.observables()
    assert o.step == r.step == 50
    assert abs(o.v_dr - r.v_dr) <= 1e-5 * max(abs(r.v_dr), 0.05) and abs(o.norm - r.norm) <= 1e-5
    assert abs(o.sum_vcos_dt - r.sum_vcos_dt) <= 1e-5 * max(abs(r.sum_vcos_dt), 0.05 * r.window)
    s.destroy()


def test_fp32_storage_batch_with_budgets_through_the_warp_kernel():
    from paper_1401_6047_b200 import Solver
    from oracle import OracleSim
    w = W.random_batch(n_batch=5, N=40, M1=200, dt=0.004, seed=77, periods=0.2)
    n = w.n_steps + 4
    s = Solver(w.grid, w.params, precision=1)
    assert s.get_option("effective_variant") == 5
    s.init_equilibrium()
    s.step(n)
    obs = s.observables()
    for i in range(5):
        sim = OracleSim(w.grid.n_harm, w.grid.n_phiy, w.grid.dt, w.params[i], threads=4, precision=1)
        sim.init_equilibrium()
        sim.step(n)
        scale = max(np.abs(x).max() for g in (0, 1) for x in sim.get_state(g))
        for g in (0, 1):
            a, b = s.get_state(i, g)
            ra, rb = sim.get_state(g)
            assert max(np.abs(a - ra).max(), np.abs(b - rb).max()) <= 8 * EPS32 * scale, (i, g)
        assert obs[i].step == w.params[i].n_steps_total
    s.destroy()


def test_fp32_state_roundtrip_and_batch():
    from paper_1401_6047_b200 import Solver
    rng = np.random.default_rng(3)
    w = W.random_batch(n_batch=3, N=6, M1=70, dt=0.004, seed=21, periods=0.0, n_steps=10)
    s = Solver(w.grid, w.params, precision=2)
    s.init_equilibrium()
    a = rng.standard_normal((7, 70)).astype(np.float32).astype(np.float64)
    b = rng.standard_normal((7, 70)).astype(np.float32).astype(np.float64)
    b[0] = 0
    s.set_state(1, 0, a, b)
    ga, gb = s.get_state(1, 0)
    assert np.array_equal(ga, a) and np.array_equal(gb, b)
    o0 = s.observables()[0].v_dr
    s.step(10)
    assert s.observables()[2].step == 10 and np.isfinite(s.get_state(2, 1)[0]).all() and s.observables()[0].v_dr != o0
    s.destroy()


def test_norm_drift_in_float_grows_as_the_time_step_shrinks():
    """in float the norm drifts for small dt ('diverges' for dt <= 1e-5 on the paper's runs to t = 10);
    drift at fixed t ~ eps32 / dt.  fp64 on the same lattice keeps the norm to 1e-12."""
    from paper_1401_6047_b200 import Solver
    drift = {}
    for prec, dts in ((2, (1e-2, 1e-3, 1e-4, 2e-5)), (0, (1e-4,))):
        for dt in dts:
            w = W.small_case(N=8, M1=81, dt=dt, E_dc=2.0, E_omega=0.0, omega=0.0, B=1.0, mu=2.0, phiy_max=6.0)
            s = Solver(w.grid, w.params, precision=prec)
            s.init_equilibrium()
            s.step(int(round(0.5 / dt)))
            drift[(prec, dt)] = abs(s.observables()[0].norm - 1.0)
            s.destroy()
    print(drift)
    assert drift[(2, 1e-3)] > 3 * drift[(2, 1e-2)] and drift[(2, 1e-4)] > 3 * drift[(2, 1e-3)]
    assert drift[(2, 2e-5)] > 2 * drift[(2, 1e-4)] and drift[(2, 2e-5)] > 2e-4
    assert drift[(0, 1e-4)] < 1e-12
