"""the real-space-phi_x variant (one cyclic tridiagonal Crank-Nicolson solve per phi_y row) through
the C ABI against its oracle (oracle/bte_rs_oracle.py), and against the harmonic-form solver.  pytest -m gpu."""
import numpy as np
import pytest

from paper_1401_6047_b200 import workloads as W

pytestmark = pytest.mark.gpu


def run_pair(K, M1, n_steps, **kw):
    from paper_1401_6047_b200 import RealSpaceSolver
    from oracle.bte_rs_oracle import RealSpaceSim
    w = W.small_case(N=2, M1=M1, **kw)
    p = w.params[0]
    s = RealSpaceSolver(K, M1, w.grid.dt, p)
    s.init_equilibrium()
    s.step(n_steps)
    sim = RealSpaceSim(K, M1, w.grid.dt, p)
    sim.init_equilibrium()
    sim.step(n_steps)
    return s, sim, p, w.grid.dt


@pytest.mark.parametrize("K,M1", [(4, 3), (8, 9), (16, 5), (37, 41), (64, 130), (96, 33), (128, 257), (512, 43), (1024, 19), (2048, 11)])
def test_realspace_matches_oracle(K, M1):
    n_steps = 12 if K * M1 > 5000 else 30
    s, sim, p, dt = run_pair(K, M1, n_steps, dt=0.004, avg_start=3)
    scale = max(np.abs(sim.fh).max(), np.abs(sim.ff).max())
    for g, ref in ((0, sim.fh), (1, sim.ff)):
        f = s.get_state(g)
        assert f.shape == ref.shape and np.isfinite(f).all()
        assert np.abs(f - ref).max() <= 1e-12 * scale, (K, M1, g, np.abs(f - ref).max() / scale)
    o = s.observables()
    assert o.step == n_steps
    assert abs(o.norm - sim.norm()) <= 1e-10 and abs(o.v_dr - sim.v_dr()) <= 1e-10 * max(abs(sim.v_dr()), 0.05)
    assert abs(o.sum_vcos_dt - sim.sum_c) <= 1e-10 * max(abs(sim.sum_c), 0.05 * sim.window)
    assert abs(o.window - sim.window) <= 1e-12
    s.destroy()


def test_realspace_budget_and_rejections():
    from paper_1401_6047_b200 import BteError, RealSpaceSolver
    w = W.small_case(N=2, M1=21, dt=0.004)
    w.params[0].n_steps_total = 7
    s = RealSpaceSolver(16, 21, 0.004, w.params[0])
    s.init_equilibrium()
    s.step(20)
    assert s.observables().step == 7
    s.destroy()
    with pytest.raises(BteError):
        RealSpaceSolver(2, 21, 0.004, w.params[0])                     # too few phi_x points
    bad = W.small_case(N=2, M1=41, dt=0.5, B=4.0, phiy_max=4.0)
    with pytest.raises(BteError) as e:
        RealSpaceSolver(16, 41, 0.5, bad.params[0])
    assert e.value.code == -2


def test_realspace_config0_approaches_the_harmonic_form():
    """BASELINE config 0 both ways: 20 harmonics vs 64 periodic phi_x points, 201 phi_y points, to t = 2.  The two
    discretisations of phi_x differ by O(dx^2) (modified wavenumber sin(dx)/dx); both conserve the norm."""
    from paper_1401_6047_b200 import RealSpaceSolver, Solver
    w = W.config0()
    h = Solver(w.grid, w.params)
    h.init_equilibrium()
    h.step(400)
    vh = h.observables()[0].v_dr
    err = []
    for K in (32, 64):
        r = RealSpaceSolver(K, w.grid.n_phiy, w.grid.dt, w.params[0])
        r.init_equilibrium()
        r.step(400)
        o = r.observables()
        assert abs(o.norm - 1.0) < 1e-10
        err.append(abs(o.v_dr - vh))
        r.destroy()
    assert 3.0 < err[0] / err[1] < 5.0 and err[1] < 1e-3 * abs(vh), (err, vh)
    h.destroy()
