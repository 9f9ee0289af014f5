"""the zero-temperature pendulum model, eq. (44)-(46), on the GPU against the oracle, and
against the Boltzmann solver itself at low temperature (the paper's Fig. 4 comparison, L225: "match very close, but
not quite, due to the finite temperature").  Run on the B200 box: pytest -m gpu."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

SETS = [(1.0, 0.0, 0.0, 0.0),        # dc only, B = 0: Esaki-Tsu at T = 0
        (2.0, 0.5, 1.5, 0.0),        # Tucker regime
        (0.0, 0.1, 3.0, 4.0),        # Fig. 4(a): E_dc = 0
        (6.0, 0.1, 4.0, 4.0),        # Fig. 4(b): E_dc = 6
        (6.0, 0.1, 7.5, 4.0),
        (3.0, 1.0, 2.0, 2.0),        # config-4-like fields
        (5.0, 0.0, 0.0, 1.0)]        # dc, crossed fields


def test_pendulum_matches_oracle():
    """Same RK4 / Simpson / phase rule on both sides; they differ in the sin / cos / exp implementations (<= 2 ulp)
    and in the order of the phase sum.  Along a trajectory such differences grow at most like the local stretching
    rate (<= B) while the memory weight decays like e^{-s}; 1e-9 covers every set used here (measured: 1e-16)."""
    from paper_1401_6047_b200 import pendulum_averages
    from oracle import pendulum_averages as ref_averages
    n_phase, h, n_rk = 48, 0.004, 7500
    got = pendulum_averages(SETS, n_phase, h, n_rk)
    worst = 0.0
    for ps, g in zip(SETS, got):
        r = ref_averages(*ps, n_phase, h, n_rk)
        for x, y in zip(g, r):
            worst = max(worst, abs(x - y))
            assert abs(x - y) <= 1e-9 * max(abs(y), 0.05), (ps, g, r)
    print("pendulum worst abs diff", worst)


def test_pendulum_rejects_bad_arguments():
    from paper_1401_6047_b200 import BteError, pendulum_averages
    with pytest.raises(BteError):
        pendulum_averages(SETS[:1], 16, 0.004, 7501)          # odd number of RK4 steps
    with pytest.raises(BteError):
        pendulum_averages([(float("nan"), 0, 0, 0)], 16, 0.004, 100)


def test_low_temperature_boltzmann_solution_approaches_the_pendulum_model():
    """P11 of SURVEY 8(c): at mu = 116 the absorption from the Boltzmann solver is close to the T = 0 pendulum
    value (paper, Fig. 4b parameters: B = 4, E_dc = 6, E_omega = 0.1, alpha = 0.9496).  Loose by nature."""
    from paper_1401_6047_b200 import Solver, pendulum_averages, workloads as W
    from parity_util import absorption
    omegas = [3.0, 5.0]
    w = W.absorption_sweep(omegas, E_dc=6.0, E_omega=0.1, B=4.0, mu=116.0, N=100, M1=2001, dt=0.002, t_relax=10.0,
                           periods=4, alpha=0.9496)
    s = Solver(w.grid, w.params)
    s.init_equilibrium()
    s.step(w.n_steps)
    obs = s.observables()
    pend = pendulum_averages([(6.0, 0.1, om, 4.0) for om in omegas], 64, 0.004, 10000)
    for i, om in enumerate(omegas):
        assert abs(obs[i].norm - 1.0) < 1e-6, obs[i].norm
        A_bte = absorption(obs[i], 116.0)
        A_pend = 2.0 * pend[i][1]
        print("omega", om, "A_bte", A_bte, "A_pendulum", A_pend, "v_mean", obs[i].sum_v_dt / obs[i].window, pend[i][0])
        assert abs(A_bte - A_pend) <= 0.15 * max(abs(A_pend), 0.02), (om, A_bte, A_pend)
        assert abs(obs[i].sum_v_dt / obs[i].window - pend[i][0]) <= 5e-3 * abs(pend[i][0])     # measured: 1.1e-3
    s.destroy()
