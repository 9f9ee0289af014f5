"""Pins of the real-space-phi_x oracle (oracle/bte_rs_oracle.py) -- the variant is not in the
paper, so everything here is mathematics: a fixed point, an exact invariant, a closed form of the discrete scheme, and
second-order convergence to the (independently pinned) harmonic-form oracle."""
import math

import numpy as np
import pytest

from oracle import OracleSim
from oracle.bte_rs_oracle import RealSpaceSim
from paper_1401_6047_b200 import workloads as W


def params(**kw):
    w = W.small_case(**kw)
    return w.params[0]


def test_f0_is_a_fixed_point_without_fields_and_relaxes_at_rate_xi_over_nu():
    p = params(N=2, M1=9, E_dc=0.0, E_omega=0.0, omega=0.0, B=0.0, mu=2.0, phiy_max=3.0)
    s = RealSpaceSim(16, 9, 0.01, p)
    s.init_equilibrium()
    s.step(5)
    assert np.abs(s.fh - s.f0).max() <= 1e-15 * s.f0.max() and np.abs(s.ff - s.f0).max() <= 1e-15 * s.f0.max()
    rng = np.random.default_rng(0)
    d0 = 1e-3 * rng.standard_normal(s.fh.shape)
    s.fh = s.f0 + d0
    s.step(1)
    assert np.abs((s.fh - s.f0) - d0 * (1 - 0.005) / (1 + 0.005)).max() <= 1e-15     # no fields: pure relaxation (rounding only)


def test_norm_is_conserved_in_crossed_fields():
    p = params(N=2, M1=41, E_dc=2.0, E_omega=0.5, omega=1.5, B=1.0, mu=2.0, phiy_max=6.0)
    s = RealSpaceSim(32, 41, 0.01, p)
    s.init_equilibrium()
    n0 = s.norm()
    s.step(100)
    assert abs(n0 - 1.0) < 1e-6                       # eq. (6): phi_y cut at +-6, rectangle rules spectrally accurate
    assert abs(s.norm() - n0) < 1e-12                  # centred differences telescope: exact up to rounding / edge leak


def test_B0_steady_drift_velocity_is_esaki_tsu_with_the_modified_wavenumber():
    """B = 0, dc field: the first discrete Fourier mode obeys (1 + i E sin(dx)/dx) c_1 = c_1^(0) at the fixed point
    (the centred difference of e^{ix} is i sin(dx)/dx e^{ix}), hence
    v* = sqrt(alpha) dx dphi sum_m [sum_i f0 cos x_i] E_eff / (1 + E_eff^2), E_eff = E sin(dx)/dx -- exactly."""
    K, M1, dt, E = 16, 5, 0.01, 1.3
    p = params(N=2, M1=M1, E_dc=E, E_omega=0.0, omega=0.0, B=0.0, mu=1.5, alpha=0.9496, phiy_max=1.0)
    s = RealSpaceSim(K, M1, dt, p)
    s.init_equilibrium()
    s.step(int(round(24.0 / dt)))
    Eeff = E * math.sin(s.dx) / s.dx
    want = math.sqrt(p.alpha) * s.dx * s.dphi * float((np.cos(s.x)[:, None] * s.f0).sum()) * Eeff / (1 + Eeff ** 2)
    assert abs(s.v_dr() - want) < 1e-9 * abs(want) + 1e-12


def test_second_order_convergence_to_the_harmonic_form():
    """Same physical problem in both representations (crossed fields, t = 0.5): the real-space result approaches the
    harmonic-form oracle like dx^2 (the harmonic form treats phi_x exactly)."""
    kw = dict(N=24, M1=41, dt=0.005, E_dc=2.0, E_omega=0.0, omega=0.0, B=1.0, mu=2.0, phiy_max=6.0)
    p = params(**kw)
    ref = OracleSim(24, 41, 0.005, p)
    ref.init_equilibrium()
    ref.step(100)
    v_ref = ref.observables().v_dr
    err = []
    for K in (16, 32, 64):
        s = RealSpaceSim(K, 41, 0.005, p)
        s.init_equilibrium()
        s.step(100)
        err.append(abs(s.v_dr() - v_ref))
    assert 3.3 < err[0] / err[1] < 4.7 and 3.3 < err[1] / err[2] < 4.7, err
    assert err[2] < 2e-3 * abs(v_ref)


def test_running_sums_match_the_harmonic_form():
    """sum v dt, sum v cos(wt) dt, sum v sin(wt) dt of the real-space oracle against the harmonic-form oracle (whose
    three sums are pinned by the Tucker closed forms, P9): same problem, ac field, K = 64 phi_x points (dx^2 error)."""
    kw = dict(N=24, M1=41, dt=0.005, E_dc=2.0, E_omega=0.5, omega=1.5, B=1.0, mu=2.0, phiy_max=6.0, avg_start=40)
    p = params(**kw)
    ref = OracleSim(24, 41, 0.005, p)
    ref.init_equilibrium()
    ref.step(240)
    o = ref.observables()
    s = RealSpaceSim(64, 41, 0.005, p)
    s.init_equilibrium()
    s.step(240)
    assert abs(s.window - o.window) < 1e-12 and o.window > 0.9
    assert min(abs(o.sum_vcos_dt), abs(o.sum_vsin_dt)) > 0.02 * abs(o.sum_v_dt)   # all three sums are significant here
    assert abs(o.sum_vcos_dt - o.sum_vsin_dt) > 0.02 * abs(o.sum_v_dt)            # ... and distinguishable
    for got, want in ((s.sum_v, o.sum_v_dt), (s.sum_c, o.sum_vcos_dt), (s.sum_s, o.sum_vsin_dt)):
        assert abs(got - want) < 3e-3 * abs(o.sum_v_dt), (got, want)
