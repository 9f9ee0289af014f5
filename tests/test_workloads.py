"""The seeded input generator (paper_1401_6047_b200/workloads.py): shapes, step counts and the phi_y-extent
rule of DESIGN.md section 3 / SURVEY.md 8(d).  Host logic only."""
import math

from paper_1401_6047_b200 import workloads as W


def test_config_shapes_and_step_counts():
    want = {0: (20, 201, 1, 0.005, 4000), 1: (50, 1001, 1, 0.002, 62832), 2: (150, 4001, 1, 0.001, 78540),
            4: (512, 32001, 1, 0.001, 2000)}
    for i, (N, M1, nb, dt, steps) in want.items():
        w = W.get(i)
        assert (w.grid.n_harm, w.grid.n_phiy, w.grid.n_batch, w.grid.dt, w.n_steps) == (N, M1, nb, dt, steps), i
    w = W.get(3)
    assert (w.grid.n_harm, w.grid.n_phiy, w.grid.n_batch, w.grid.dt) == (40, 801, 512, 0.002)
    budgets = [p.n_steps_total for p in w.params]
    assert min(budgets) >= 7854 and max(budgets) <= 125664 and w.n_steps == max(budgets)
    for p in w.params:
        assert p.n_steps_total == round(20 * 2 * math.pi / (p.omega * 0.002))
        assert p.avg_start_step == p.n_steps_total // 2 and p.E_omega == 0.1
        assert 0 <= p.E_dc <= 8 and 0.5 <= p.omega <= 8 and 0 <= p.B <= 5 and 0.5 <= p.mu <= 5


def test_phiy_extents_of_the_table():
    assert W.get(0).params[0].phiy_max == 7.5
    assert W.get(1).params[0].phiy_max == 11.0
    assert W.get(2).params[0].phiy_max == 8.0        # CFL term binds
    assert W.get(4).params[0].phiy_max == 32.0       # CFL term binds


def test_every_system_is_stable_and_symmetric():
    for i in range(5):
        w = W.get(i)
        M = w.grid.n_phiy - 1
        for p in w.params:
            dphi = (p.phiy_max - p.phiy_min) / M
            assert abs(p.B) * w.grid.dt / dphi <= 1.0 + 1e-12          # C11, generator keeps <= 1
            assert p.phiy_min == -p.phiy_max and p.mu > 0 and p.alpha == 1.0


def test_config3_is_seeded():
    a, b = W.config3(), W.config3()
    assert [vars(p) for p in a.params] == [vars(p) for p in b.params]
    c = W.config3(seed=W.SEED_CONFIG3 + 1)
    assert vars(c.params[0]) != vars(a.params[0])
    r = W.SplitMix64(1)
    u = [r.uniform() for _ in range(1000)]
    assert all(0.0 <= x < 1.0 for x in u) and 0.45 < sum(u) / 1000 < 0.55


def test_updates_between_counts_frozen_systems_out():
    w = W.random_batch(n_batch=3, N=4, M1=30, dt=0.004, seed=5, periods=0.1)
    pts = 5 * 30
    total = sum(p.n_steps_total for p in w.params) * pts
    assert w.updates_between(0, w.n_steps + 10) == total
    assert w.updates_between(0, 1) == 3 * pts


def test_absorption_sweep_windows_are_whole_periods():
    w = W.absorption_sweep([1.0, 2.5, 7.0], E_dc=5.0, E_omega=1.0, B=0.0, mu=50.0, N=6, M1=41, dt=0.002,
                           periods=6)
    assert w.grid.n_batch == 3 and w.n_steps == max(p.n_steps_total for p in w.params)
    for p in w.params:
        assert p.avg_start_step == 5000                                   # t = 10
        n_avg = p.n_steps_total - p.avg_start_step
        assert abs(n_avg * 0.002 - 6 * 2 * math.pi / p.omega) <= 0.002    # an integer number of periods


def test_tucker_helper_against_the_oracle_on_cpu():
    """The closed form used by the GPU spectrum test, checked here against the oracle at one frequency."""
    from oracle import OracleSim
    from parity_util import absorption, tucker_averages
    w = W.absorption_sweep([3.0], E_dc=5.0, E_omega=1.0, B=0.0, mu=50.0, N=3, M1=21, dt=0.002, periods=6)
    sim = OracleSim(3, 21, 0.002, w.params[0])
    sim.init_equilibrium()
    sim.step(w.n_steps)
    A = absorption(sim.observables(), 50.0)
    ref = tucker_averages(50.0, 5.0, 1.0, 3.0)[2]
    assert abs(A - ref) < 2e-3 * max(abs(ref), 0.05)


def test_paper_table1_workload_is_the_papers_command_line():
    w = W.get(5)
    p = w.params[0]
    assert (w.grid.n_harm, w.grid.n_phiy, w.grid.dt, w.n_steps) == (120, 4000, 1e-4, 100000)       # L325-326
    assert (p.E_dc, p.E_omega, p.omega, p.B, p.mu, p.alpha, p.phiy_min, p.phiy_max) == \
        (7.0, 0.1, 10.0, 4.0, 116.0, 0.9496, -6.0, 6.0)
    assert abs(p.B) * w.grid.dt / ((p.phiy_max - p.phiy_min) / (w.grid.n_phiy - 1)) < 1.0           # C11
    assert abs(120 * 4000 * 1e5 / 43.85 / 1e6 - W.PAPER_TABLE1_MLUPS_K6) < 1.0                       # Table 1, K6 column
