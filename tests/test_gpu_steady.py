"""steady-state detection and averaging policy on the device (C23) against
the oracle's implementation of the same policy.  Run on the B200 box: pytest -m gpu."""
import math

import numpy as np
import pytest

from paper_1401_6047_b200 import workloads as W

from parity_util import assert_obs_close, assert_state_close

pytestmark = pytest.mark.gpu


def run_both(w, n_steps, tol, n_avg, min_relax, variant, sweep_steps, chunks):
    from paper_1401_6047_b200 import Solver
    from oracle import OracleSim
    s = Solver(w.grid, w.params)
    s.set_option("variant", variant)
    s.set_option("sweep_steps", sweep_steps)
    s.set_steady_policy(tol, n_avg, min_relax)
    s.init_equilibrium()
    for c in chunks:
        s.step(c)
    assert sum(chunks) == n_steps
    obs = s.observables()
    steps, phases = s.steady_info()
    sims = []
    for i in range(w.grid.n_batch):
        sim = OracleSim(w.grid.n_harm, w.grid.n_phiy, w.grid.dt, w.params[i], threads=4)
        sim.set_steady_policy(tol, n_avg, min_relax)
        sim.init_equilibrium()
        sim.step(int(obs[i].step))          # a finished system stops within one launch group after its window
        sims.append(sim)
    return s, obs, steps, phases, sims


@pytest.mark.parametrize("variant,sweep_steps", [(5, 4), (5, 3), (5, 2), (3, 2), (3, 1), (0, 0)])
def test_steady_policy_batch_matches_the_oracle(variant, sweep_steps):
    """Six systems with different frequencies (different comparison intervals and windows) in one batch: the step at
    which each is found relaxed, its phase, window and sums, and its state at the step where it stopped."""
    w = W.random_batch(n_batch=6, N=33, M1=120, dt=0.004, seed=9, periods=0.0, n_steps=9000)
    for i, p in enumerate(w.params):
        p.E_omega = 0.3
        p.omega = 2.0 + 0.9 * i
        p.n_steps_total = 0
        p.avg_start_step = 0
    n = 9000
    s, obs, steps, phases, sims = run_both(w, n, 1e-4, 2, 0, variant, sweep_steps, [1000, 1, 4999, 3000])
    assert s.get_option("effective_variant") in (3, 5)
    finished = 0
    for i, sim in enumerate(sims):
        st, ph = sim.steady_info()
        assert (steps[i], phases[i]) == (st, ph), (i, steps[i], phases[i], st, ph)
        p = w.params[i]
        if ph == 2:
            finished += 1
            win = round(2 * 2 * math.pi / (p.omega * w.grid.dt))
            assert st > 0 and st + win <= obs[i].step <= st + win + 3
            assert abs(obs[i].window - win * w.grid.dt) < 1e-9
        assert_state_close(s, sim, i, what=f"steady batch[{i}] v{variant} S{sweep_steps}")
        assert_obs_close(obs[i], sim.observables(), p, w.grid.dt, what=f"steady batch[{i}] v{variant} S{sweep_steps}")
    assert finished >= 4
    s.destroy()


def test_steady_policy_absorption_spectrum_matches_tucker_at_B0():
    """The paper's use of the solver (Fig. 3: A(omega) at B = 0) without a hand-set relaxation time: every frequency
    point relaxes, averages 3 periods and stops by itself; closed form of eq. (42)-(43), normalisation C9."""
    from scipy import special
    from paper_1401_6047_b200 import Solver
    omegas = np.linspace(1.0, 6.0, 11)
    mu, E_dc, E_w = 5.0, 5.0, 1.0
    w = W.absorption_sweep(omegas, E_dc=E_dc, E_omega=E_w, B=0.0, mu=mu, N=40, M1=33, dt=0.002, periods=3)
    for p in w.params:
        p.n_steps_total = 0
        p.avg_start_step = 0
    s = Solver(w.grid, w.params)
    s.set_steady_policy(1e-6, 3, 0)
    s.init_equilibrium()
    s.step(22000)
    obs = s.observables()
    steps, phases = s.steady_info()
    r = special.iv(1, mu) / special.iv(0, mu)
    nn = np.arange(-60, 61)
    for i, om in enumerate(omegas):
        assert phases[i] == 2, (i, om, steps[i], phases[i])
        beta = E_w / om
        xi = (E_dc + nn * om) / (1.0 + (E_dc + nn * om) ** 2)
        J = special.jv(nn, beta)
        vc = 0.5 * r * np.sum(J * (special.jv(nn + 1, beta) + special.jv(nn - 1, beta)) * xi)
        got = obs[i].sum_vcos_dt / obs[i].window
        assert abs(got - vc) < 3e-3 * abs(vc) + 2e-6, (om, got, vc)
    s.destroy()


def test_steady_policy_is_refused_where_it_cannot_run():
    from paper_1401_6047_b200 import Solver
    from paper_1401_6047_b200.binding import BteError
    w = W.small_case(N=12, M1=100, dt=0.004, n_steps=10)
    s = Solver(w.grid, w.params, precision=2)
    with pytest.raises(BteError):
        s.set_steady_policy(1e-4, 1, 0)
    s.destroy()
    s = Solver(w.grid, w.params)
    s.set_option("variant", 1)
    with pytest.raises(BteError):
        s.set_steady_policy(1e-4, 1, 0)
    with pytest.raises(BteError):
        s.set_steady_policy(-1.0, 1, 0)
    s.set_steady_policy(0.0, 0, 0)          # off: always allowed
    s.destroy()
