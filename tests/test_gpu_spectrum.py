"""the absorption spectrum A(omega) as a first-class batched workload (the paper's use of
the solver, Fig. 3: mu = 50, alpha = 0.9496, B = 0, E_omega = 1, E_dc = 5).  One system per frequency, relaxed
to t = 10 (L103), then an integer number of ac periods; checked against the Tucker closed form (eq. 42-43) and,
system by system, against the oracle.  Run on the B200 box: pytest -m gpu."""
import numpy as np
import pytest

from paper_1401_6047_b200 import workloads as W

from parity_util import absorption, assert_obs_close, assert_state_close, oracle_run, tucker_averages

pytestmark = pytest.mark.gpu


def test_absorption_spectrum_B0_matches_tucker_and_oracle():
    from paper_1401_6047_b200 import Solver
    omegas = np.linspace(1.0, 12.0, 23)
    w = W.absorption_sweep(omegas, E_dc=5.0, E_omega=1.0, B=0.0, mu=50.0, N=6, M1=41, dt=0.002, periods=6,
                           alpha=0.9496)
    s = Solver(w.grid, w.params)
    s.init_equilibrium()
    s.step(w.n_steps)
    obs = s.observables()
    A = np.array([absorption(o, 50.0) for o in obs])
    ref = np.array([tucker_averages(50.0, 5.0, 1.0, om)[2] for om in omegas])
    for i, p in enumerate(w.params):
        assert obs[i].step == p.n_steps_total
        assert abs(obs[i].window - (p.n_steps_total - p.avg_start_step) * w.grid.dt) < 1e-9
    # time discretisation (dt^2) and the e^{-10} transient bound the agreement with the continuous closed form
    assert np.max(np.abs(A - ref)) < 2e-3 * np.max(np.abs(ref)), (A, ref)
    assert (ref.max() > 0) and (ref.min() < 0)                     # the sweep crosses gain and loss
    for i, sim in oracle_run(w, w.n_steps, systems=[0, 7, 22]).items():
        assert_state_close(s, sim, i, what=f"A(omega)[{i}]")
        assert_obs_close(obs[i], sim.observables(), w.params[i], w.grid.dt, what=f"A(omega)[{i}]")
    s.destroy()


def test_absorption_spectrum_crossed_fields_against_oracle():
    """Fig. 4-like parameters (B = 4, E_omega = 0.1, low temperature) on a small lattice: no closed form, parity
    with the oracle on every system."""
    from paper_1401_6047_b200 import Solver
    w = W.absorption_sweep([2.0, 3.5, 5.0], E_dc=6.0, E_omega=0.1, B=4.0, mu=20.0, N=24, M1=161, dt=0.004,
                           t_relax=2.0, periods=2, alpha=0.9496)
    s = Solver(w.grid, w.params)
    s.init_equilibrium()
    s.step(w.n_steps)
    obs = s.observables()
    for i, sim in oracle_run(w, w.n_steps).items():
        assert_state_close(s, sim, i, what=f"A(omega) crossed[{i}]")
        assert_obs_close(obs[i], sim.observables(), w.params[i], w.grid.dt, what=f"A(omega) crossed[{i}]")
    s.destroy()


@pytest.mark.parametrize("N,M1,K", [(6, 41, 16), (20, 300, 64), (33, 129, 37), (150, 500, 128)])
def test_pdf_reconstruction_matches_oracle(N, M1, K):
    """f(phi_x, phi_y) of eq. (8) from the evolved state, both grids, against the oracle's
    plain Fourier sum; odd K and K not a multiple of the per-thread chunk included."""
    from paper_1401_6047_b200 import Solver
    from oracle import OracleSim
    w = W.small_case(N=N, M1=M1, dt=0.004, n_steps=9, avg_start=2)
    s = Solver(w.grid, w.params)
    s.init_equilibrium()
    s.step(9)
    sim = OracleSim(N, M1, w.grid.dt, w.params[0])
    sim.init_equilibrium()
    sim.step(9)
    for g in (0, 1):
        f = s.reconstruct_pdf(0, g, K).cpu().numpy()
        ref = sim.reconstruct_pdf(g, K)
        assert f.shape == ref.shape == (K, M1)
        assert np.abs(f - ref).max() <= 1e-12 * np.abs(ref).max()
    s.destroy()
