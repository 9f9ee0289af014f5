"""Helpers for the GPU-vs-oracle parity tests (tests only)."""
from __future__ import annotations

import numpy as np
from scipy import special

from oracle import OracleSim

# north_star tolerances (fp64): max |df| <= 1e-12 max|f| over both grids of a system; observables 1e-10
# relative, with the floors of DESIGN.md C15 for quantities that can pass through zero.
TOL_STATE = 1e-12
TOL_OBS = 1e-10


def oracle_run(w, n_steps, systems=None, threads=4):
    """Run the oracle for the listed systems of workload w; returns {sys: (sim, obs)}."""
    out = {}
    for s in (range(w.grid.n_batch) if systems is None else systems):
        sim = OracleSim(w.grid.n_harm, w.grid.n_phiy, w.grid.dt, w.params[s], threads=threads)
        sim.init_equilibrium()
        sim.step(n_steps)
        out[s] = sim
    return out


def v_floor(p):
    return float(special.ive(1, p.mu) / special.ive(0, p.mu) / 2.0)


def assert_state_close(solver, sim, sys_index, tol=TOL_STATE, what=""):
    ha, hb = sim.get_state(0)
    fa, fb = sim.get_state(1)
    scale = max(np.abs(ha).max(), np.abs(hb).max(), np.abs(fa).max(), np.abs(fb).max())
    worst = 0.0
    for g, (ra, rb) in ((0, (ha, hb)), (1, (fa, fb))):
        ga, gb = solver.get_state(sys_index, g)
        assert np.isfinite(ga).all() and np.isfinite(gb).all(), f"{what}: non-finite GPU state"
        worst = max(worst, np.abs(ga - ra).max(), np.abs(gb - rb).max())
        assert np.all(gb[0] == 0.0), f"{what}: b_0 must stay exactly 0 (eq. 23)"
    assert worst <= tol * scale, f"{what}: max|df| = {worst:.3e} > {tol:g} * max|f| = {tol * scale:.3e}"
    return worst / scale


def assert_obs_close(got, ref, p, dt, tol=TOL_OBS, what=""):
    vf = v_floor(p)
    assert got.step == ref.step, f"{what}: step {got.step} != {ref.step}"
    assert abs(got.t - ref.t) <= 1e-12 * max(1.0, abs(ref.t))
    assert abs(got.norm - ref.norm) <= tol * max(abs(ref.norm), 1.0), f"{what}: norm {got.norm} vs {ref.norm}"
    assert abs(got.v_dr - ref.v_dr) <= tol * max(abs(ref.v_dr), vf), f"{what}: v_dr {got.v_dr} vs {ref.v_dr}"
    win = max(ref.window, dt)
    for k in ("sum_v_dt", "sum_vcos_dt", "sum_vsin_dt"):
        g, r = getattr(got, k), getattr(ref, k)
        assert abs(g - r) <= tol * max(abs(r), vf * win), f"{what}: {k} {g} vs {r}"
    assert abs(got.window - ref.window) <= 1e-12 * max(ref.window, dt), f"{what}: window"
    assert abs(got.edge_leak - ref.edge_leak) <= tol * max(abs(ref.edge_leak), vf), f"{what}: edge_leak"


def tucker_averages(mu, E_dc, E_w, w, nmax=60):
    """B = 0 closed forms, eq. (42)-(43) of the paper (L208-213) in eq. (17)'s normalisation (C9):
    <v> = (I1/I0) sum_n J_n(b)^2 xi(E_dc + n w),  <v cos wt> = (I1/2I0) sum_n J_n(b)[J_{n+1}(b) + J_{n-1}(b)]
    xi(E_dc + n w), b = E_w / w, xi(E) = E / (1 + E^2).  Returns (<v>, <v cos wt>, A = (2 I0/I1) <v cos wt>)."""
    nn = np.arange(-nmax, nmax + 1)
    beta = E_w / w
    J, Jp, Jm = special.jv(nn, beta), special.jv(nn + 1, beta), special.jv(nn - 1, beta)
    xi = (E_dc + nn * w) / (1 + (E_dc + nn * w) ** 2)
    r = float(special.ive(1, mu) / special.ive(0, mu))
    v_mean = r * float(np.sum(J * J * xi))
    v_cos = 0.5 * r * float(np.sum(J * (Jp + Jm) * xi))
    return v_mean, v_cos, 2.0 / r * v_cos


def tucker_sin_average(mu, E_dc, E_w, w, nmax=60):
    """The quadrature partner of eq. (43) at B = 0 (same derivation: v(t) = (I1/I0) Im sum_{n,m} J_n J_m
    e^{i (n-m) w t} / (1 - i (E_dc + m w)); <e^{i(n-m)wt} sin wt> = -+ 1/(2i) for n - m = +-1):
    <v sin wt> = (I1/2I0) sum_n J_n(b) [J_{n+1}(b) - J_{n-1}(b)] / (1 + (E_dc + n w)^2),  b = E_w / w."""
    nn = np.arange(-nmax, nmax + 1)
    beta = E_w / w
    J, Jp, Jm = special.jv(nn, beta), special.jv(nn + 1, beta), special.jv(nn - 1, beta)
    r = float(special.ive(1, mu) / special.ive(0, mu))
    return 0.5 * r * float(np.sum(J * (Jp - Jm) / (1 + (E_dc + nn * w) ** 2)))


def absorption(obs, mu):
    """Eq. (17): A = (2 I0(mu)/I1(mu)) <v_dr cos wt>, from the raw sums the library returns (C9)."""
    return 2.0 * float(special.ive(0, mu) / special.ive(1, mu)) * obs.sum_vcos_dt / obs.window
