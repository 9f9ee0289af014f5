"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU needed).

Each test names the pin (P1..P14 of DESIGN.md) and the PAPER.md passage it rests on.  None of them
re-types the oracle's own update formula: they use closed forms, invariants, library routines
(scipy Bessel functions, a dense linear solve of eqs. (24)-(27), an FFT of eq. (13)) or
convergence behaviour.
"""
import math

import numpy as np
import pytest
from scipy import special

from oracle import OracleSim
from paper_1401_6047_b200 import workloads as W


def make(N, M1, dt, **kw):
    d = dict(E_dc=0.0, E_omega=0.0, omega=0.0, B=0.0, mu=1.0, alpha=1.0, phiy_min=-6.0, phiy_max=6.0,
             kappa_scale=1.0, n_steps_total=0, avg_start_step=0)
    d.update(kw)
    p = W.Params(**d)
    return OracleSim(N, M1, dt, p), p


# ---------------------------------------------------------------------------------------------------
# Equilibrium: eq. (13), (15), (16); readings C1, C8, C13
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mu,alpha", [(1.0, 1.0), (2.0, 0.9496), (10.0, 1.0), (116.0, 0.9496)])
def test_equilibrium_is_fourier_series_of_eq13(mu, alpha):
    """a_n^(0) must be the cosine-Fourier coefficients (eq. 7) of f0 as printed in eq. (13).
    f0 is sampled on a phi_x grid straight from eq. (13) and transformed with numpy's FFT; I0 comes from
    scipy.  Pins sigma(n) (C1), the prefactor of eq. (15) and the Bessel ratios (C13)."""
    N, M1 = 24, 41
    s, p = make(N, M1, 0.01, mu=mu, alpha=alpha, phiy_min=-1.5, phiy_max=1.5)
    phi, a0 = s.equilibrium()
    K = 512
    x = 2 * np.pi * np.arange(K) / K
    # eq. (13) with exp(mu cos x)/I0(mu) written through the scaled Bessel function to avoid overflow
    f0 = (1.0 / (2 * np.pi * special.ive(0, mu))) * math.sqrt(mu / (2 * np.pi * alpha)) * \
        np.exp(mu * (np.cos(x)[None, :] - 1.0) - 0.5 * mu * phi[:, None] ** 2)
    c = np.fft.rfft(f0, axis=1).real / K          # c_0 = a_0, c_n = a_n / 2
    want = np.empty_like(a0)
    want[0] = c[:, 0]
    want[1:] = 2.0 * c[:, 1:N + 1].T
    scale = np.abs(want).max()
    assert np.abs(a0 - want).max() <= 2e-15 * scale * 50


def test_phi_lattice_is_exactly_symmetric():
    """C8: phi_m = centre + (m - M/2) dphi includes both ends and is bit-symmetric."""
    s, _ = make(3, 101, 0.01, phiy_min=-7.5, phiy_max=7.5)
    phi, _ = s.equilibrium()
    assert phi[0] == -7.5 and phi[-1] == 7.5
    assert np.array_equal(phi, -phi[::-1])


def test_initial_norm_is_one():
    """eq. (12) on the initial state: 2 pi sqrt(alpha) dphi sum a_0 = 1 (Gaussian quadrature error only)."""
    s, _ = make(5, 201, 0.01, mu=1.0, alpha=0.9496, phiy_min=-7.5, phiy_max=7.5)
    s.init_equilibrium()
    assert abs(s.observables().norm - 1.0) < 1e-12


# ---------------------------------------------------------------------------------------------------
# P1: B = 0, constant E -- closed form for every (n, m, k) on both grids
# ---------------------------------------------------------------------------------------------------
def test_P1_closed_form_B0_every_point():
    """With B=0 and constant E the scheme (32)-(37) decouples per point.  In w = a + i b it is the
    scalar affine map w' = rho w + a0 dt/(nu - i mu) whose k-th iterate is
    w* + (w0 - w*) rho^k, w* = a0 / (1 - i n E), rho = (xi + i mu)/(nu - i mu).  The fractional grid
    starts from one map with dt/2 (L202)."""
    N, M1, dt, E = 9, 33, 0.01, 1.7
    s, p = make(N, M1, dt, E_dc=E, mu=1.5, phiy_min=-5.0, phiy_max=5.0)
    s.init_equilibrium()
    _, a0 = s.equilibrium()
    n = np.arange(N + 1)[:, None].astype(float)
    wstar = a0 / (1.0 - 1j * n * E)

    def rho(delta):
        mu = n * E * delta / 2
        return ((1 - delta / 2) + 1j * mu) / ((1 + delta / 2) - 1j * mu)

    wf0 = wstar + (a0 - wstar) * rho(dt / 2)
    scale = a0.max()
    for k_total, nstep in [(0, 0), (1, 1), (7, 6), (250, 243)]:
        s.step(nstep)
        ah, bh = s.get_state(0)
        af, bf = s.get_state(1)
        wh = wstar + (a0 - wstar) * rho(dt) ** k_total
        wf = wstar + (wf0 - wstar) * rho(dt) ** k_total
        for got_a, got_b, want in ((ah, bh, wh), (af, bf, wf)):
            assert np.abs(got_a - want.real).max() <= 1e-13 * scale
            assert np.abs(got_b[1:] - want.imag[1:]).max() <= 1e-13 * scale
            assert np.all(got_b[0] == 0.0)


# ---------------------------------------------------------------------------------------------------
# P2: steady drift velocity at B = 0 (config 0) -- PAPER.md:L208 "exact analytical solution"
# ---------------------------------------------------------------------------------------------------
def test_P2_esaki_tsu_steady_drift_config0():
    w = W.config0()
    p = w.params[0]
    s = OracleSim(w.grid.n_harm, w.grid.n_phiy, w.grid.dt, p)
    s.init_equilibrium()
    s.step(w.n_steps)
    o = s.observables()
    want = special.ive(1, p.mu) / special.ive(0, p.mu) * p.E_dc / (1 + p.E_dc ** 2)
    assert abs(want - 0.2231949829) < 1e-9          # value quoted in DESIGN.md for mu=1, E=1
    assert abs(o.v_dr - want) / want < 1e-3          # north_star bar
    assert abs(o.v_dr - want) / want < 5e-9          # what the scheme actually reaches (e^-20 transient)
    assert abs(o.norm - 1.0) < 1e-12
    assert o.step == 4000 and abs(o.t - 20.0) < 1e-12


# ---------------------------------------------------------------------------------------------------
# P3: norm conservation, eq. (12)
# ---------------------------------------------------------------------------------------------------
def test_P3_norm_conserved_crossed_fields():
    """Summing eq. (32) at n=0 over m telescopes the stencil (31): the norm can only change through the
    edge values of b_1, which are ~0 for a wide enough phi_y range.  Config 1 parameters, 3000 steps."""
    w = W.config1()
    s = OracleSim(w.grid.n_harm, w.grid.n_phiy, w.grid.dt, w.params[0], threads=4)
    s.init_equilibrium()
    _, norms = s.step(3000, trace=True)
    assert np.abs(norms - 1.0).max() < 1e-12
    assert s.observables().edge_leak < 1e-30


# ---------------------------------------------------------------------------------------------------
# P4: E = B = 0 -- relaxation to f0
# ---------------------------------------------------------------------------------------------------
def test_P4_equilibrium_is_fixed_point_and_relaxation_rate():
    N, M1, dt = 6, 21, 0.02
    s, p = make(N, M1, dt, mu=2.0, phiy_min=-4.0, phiy_max=4.0)
    s.init_equilibrium()
    _, a0 = s.equilibrium()
    s.step(50)
    for g in (0, 1):
        a, b = s.get_state(g)
        assert np.abs(a - a0).max() <= 1e-14 * a0.max()
        assert np.all(b == 0.0)
    # from a perturbed start the deviation shrinks by xi/nu per step on each grid
    rng = np.random.default_rng(1)
    da = 1e-3 * rng.standard_normal(a0.shape)
    db = 1e-3 * rng.standard_normal(a0.shape)
    db[0] = 0.0
    s.set_state(0, a0 + da, db)
    s.set_state(1, a0 + 0.5 * da, 0.25 * db)
    k = 17
    s.step(k)
    q = ((1 - dt / 2) / (1 + dt / 2)) ** k
    a, b = s.get_state(0)
    assert np.abs((a - a0) - q * da).max() <= 1e-14 * a0.max()
    assert np.abs(b - q * db).max() <= 1e-14 * a0.max()
    a, b = s.get_state(1)
    assert np.abs((a - a0) - q * 0.5 * da).max() <= 1e-14 * a0.max()
    assert np.abs(b - q * 0.25 * db).max() <= 1e-14 * a0.max()


# ---------------------------------------------------------------------------------------------------
# P5 / P6: mirror symmetries
# ---------------------------------------------------------------------------------------------------
def test_P5_B0_mirror_phiy_bit_exact():
    """north_star: phi_y -> -phi_y symmetry at B=0 (no phi_y coupling and phi_m = -phi_{M-m}, C8)."""
    s, _ = make(8, 51, 0.01, E_dc=1.2, E_omega=0.7, omega=2.0, mu=2.0, phiy_min=-5.0, phiy_max=5.0)
    s.init_equilibrium()
    s.step(100)
    for g in (0, 1):
        a, b = s.get_state(g)
        assert np.array_equal(a, a[:, ::-1])
        assert np.array_equal(b, b[:, ::-1])


def test_P6_field_reversal_mirror_any_B():
    """Eq. (5) is invariant under (phi_x, phi_y, E) -> (-phi_x, -phi_y, -E): a_n(m; E) = a_n(M-m; -E),
    b_n(m; E) = -b_n(M-m; -E); hence v_dr is odd in E.  Sensitive to every sign in eq. (30)-(31)."""
    kw = dict(omega=1.5, B=1.5, mu=2.0, phiy_min=-8.0, phiy_max=8.0)
    sp, _ = make(10, 81, 0.01, E_dc=2.0, E_omega=0.5, **kw)
    sm, _ = make(10, 81, 0.01, E_dc=-2.0, E_omega=-0.5, **kw)
    for s in (sp, sm):
        s.init_equilibrium()
        s.step(150)
    for g in (0, 1):
        ap, bp = sp.get_state(g)
        am, bm = sm.get_state(g)
        scale = np.abs(ap).max()
        assert np.abs(ap - am[:, ::-1]).max() <= 1e-15 * scale
        assert np.abs(bp + bm[:, ::-1]).max() <= 1e-15 * scale
    assert abs(sp.observables().v_dr + sm.observables().v_dr) < 1e-15
    assert abs(sp.observables().v_dr) > 0.05


# ---------------------------------------------------------------------------------------------------
# P7: E = 0, B != 0 leaves f0 stationary up to the discretisation error, which is second order
# ---------------------------------------------------------------------------------------------------
def _dev_E0(M1, dt, kappa_scale=1.0, alpha=1.0):
    N = 16
    s, _ = make(N, M1, dt, B=2.0, mu=2.0, alpha=alpha, phiy_min=-8.0, phiy_max=8.0,
                kappa_scale=kappa_scale)
    s.init_equilibrium()
    _, a0 = s.equilibrium()
    s.step(int(round(1.0 / dt)))
    a, b = s.get_state(0)
    return max(np.abs(a - a0).max(), np.abs(b).max()) / a0.max()


def test_P7_magnetic_field_alone_keeps_f0_second_order():
    """f0 depends on (phi_x, phi_y) only through the energy, which the magnetic rotation conserves
    (eq. 3, 5), so with E=0 the exact solution is f = f0.  Halving dphi and dt must divide the numerical
    deviation by 4.  Pins the signs and the prefactor of eq. (30)-(31), chi(1)=2, and reading C4."""
    d1 = _dev_E0(161, 0.008)
    d2 = _dev_E0(321, 0.004)
    assert d1 < 5e-3
    assert 3.6 < d1 / d2 < 4.4


def test_P7b_printed_alpha_factor_is_not_consistent():
    """Reading C4: with kappa_scale = alpha (the factor printed in eq. 30-31) and alpha != 1, f0 as
    printed in eq. (13) is NOT stationary under B alone -- the deviation does not converge away."""
    alpha = 0.9496
    good = _dev_E0(321, 0.004, kappa_scale=1.0, alpha=alpha)
    bad = _dev_E0(321, 0.004, kappa_scale=alpha, alpha=alpha)
    assert bad > 10 * good


# ---------------------------------------------------------------------------------------------------
# P8: second-order convergence in dt (north_star: "first- or second-order grid convergence")
# ---------------------------------------------------------------------------------------------------
def _v_at_t1(dt, M1=161):
    s, _ = make(16, M1, dt, E_dc=2.0, E_omega=0.5, omega=1.5, B=1.0, mu=2.0, phiy_min=-10.0,
                phiy_max=10.0)
    s.init_equilibrium()
    s.step(int(round(1.0 / dt)))
    return s.observables().v_dr


def test_P8_second_order_in_dt_and_dphi():
    """CN + staggered leap-frog + start-up with dt/2 (C5, C6): successive differences shrink x4."""
    v1, v2, v4 = _v_at_t1(0.02), _v_at_t1(0.01), _v_at_t1(0.005)
    r = (v1 - v2) / (v2 - v4)
    assert 3.7 < r < 4.3
    u1, u2, u4 = _v_at_t1(0.005, 81), _v_at_t1(0.005, 161), _v_at_t1(0.005, 321)
    r = (u1 - u2) / (u2 - u4)
    assert 3.5 < r < 4.5


# ---------------------------------------------------------------------------------------------------
# P9: B = 0 with ac field -- Tucker formula, eq. (42)-(43), normalisation per reading C9
# ---------------------------------------------------------------------------------------------------
def test_P9_tucker_time_averages():
    """<v> = (I1/I0) sum_n J_n(b)^2 xi(E_dc + n w) and
    <v cos wt> = (I1/2I0) sum_n J_n(b)[J_{n+1}(b) + J_{n-1}(b)] xi(E_dc + n w), b = E_w/w (eq. 42-43 with
    eq. 17's normalisation).  Bessel functions from scipy.  Averages over 6 periods after t > 10 (L103)."""
    mu, E_dc, E_w, w, dt = 2.0, 2.0, 0.5, 1.5, 0.002
    per = 2 * math.pi / w
    n_avg = int(round(6 * per / dt))
    n_relax = int(round(12.0 / dt))
    s, _ = make(2, 41, dt, E_dc=E_dc, E_omega=E_w, omega=w, mu=mu, phiy_min=-6.0, phiy_max=6.0,
                avg_start_step=n_relax)
    s.init_equilibrium()
    s.step(n_relax + n_avg)
    o = s.observables()
    nn = np.arange(-40, 41)
    beta = E_w / w
    J = special.jv(nn, beta)
    Jp = special.jv(nn + 1, beta)
    Jm = special.jv(nn - 1, beta)
    xi = (E_dc + nn * w) / (1 + (E_dc + nn * w) ** 2)
    r = special.ive(1, mu) / special.ive(0, mu)
    v_mean = r * np.sum(J * J * xi)
    v_cos = 0.5 * r * np.sum(J * (Jp + Jm) * xi)
    assert abs(o.window - n_avg * dt) < 1e-9
    assert abs(o.sum_v_dt / o.window - v_mean) < 2e-4 * abs(v_mean)
    assert abs(o.sum_vcos_dt / o.window - v_cos) < 2e-3 * abs(v_cos) + 1e-6
    # the third accumulator, sum v sin(wt) dt: the quadrature partner of eq. (43) -- in the derivation of (42)-(43),
    # v(t) = (I1/I0) Im sum_{n,m} J_n J_m e^{i(n-m)wt} / (1 - i(E_dc + m w)), the sin wt average picks n - m = +-1 with
    # weights -+1/(2i), which leaves (I1/2I0) sum_n J_n [J_{n+1} - J_{n-1}] / (1 + (E_dc + n w)^2)
    v_sin = 0.5 * r * np.sum(J * (Jp - Jm) / (1 + (E_dc + nn * w) ** 2))
    assert abs(v_sin) > 3 * abs(v_cos) > 0                      # cos / sin swapped or a wrong sign cannot pass
    assert abs(o.sum_vsin_dt / o.window - v_sin) < 2e-3 * abs(v_sin) + 1e-6


# ---------------------------------------------------------------------------------------------------
# P10: brute force on tiny grids -- eqs. (24)-(27) assembled as one dense linear system
# ---------------------------------------------------------------------------------------------------
def _dense_T(N, M1, delta, B, dphi, phi, a0, Ea, Eb, Xa, Xb, Sa, Sb):
    """Independent statement: write (24)+(26) and (25)+(27) for all unknowns (a', b') as A z' = r and
    solve with LAPACK; the stencil terms (30)-(31) are built as dense matrices acting on S."""
    P = (N + 1) * M1

    def k(n, m):
        return n * M1 + m

    Da = np.zeros((P, P))   # A_{n,m} = sum Da[(n,m),(n',m')] Sa[n',m']
    Db = np.zeros((P, P))
    kap = B * delta / (4 * dphi)
    for n in range(N + 1):
        for m in range(M1):
            for dn, dm, sgn_b, sgn_a in ((+1, +1, +1, -1), (+1, -1, -1, +1), (-1, +1, -1, +1),
                                         (-1, -1, +1, -1)):
                n2, m2 = n + dn, m + dm
                if 0 <= n2 <= N and 0 <= m2 < M1:
                    Db[k(n, m), k(n2, m2)] += kap * sgn_b
                    chi = 2.0 if (n == 1 and dn == -1) else 1.0
                    Da[k(n, m), k(n2, m2)] += kap * sgn_a * chi
    Sb = Sb.copy()
    Sb[0] = 0.0                       # eq. (23)
    At = (Da @ Sa.ravel()).reshape(N + 1, M1)
    Bt = (Db @ Sb.ravel()).reshape(N + 1, M1)
    nidx = np.arange(N + 1)[:, None]
    mu_a = nidx * (Ea + B * phi[None, :]) * delta / 2
    mu_b = nidx * (Eb + B * phi[None, :]) * delta / 2
    A = np.zeros((2 * P, 2 * P))
    r = np.zeros(2 * P)
    for n in range(N + 1):
        for m in range(M1):
            i = k(n, m)
            # (24)+(26): 2a' - 2a = 2 a0 d - (a + a') d - 2 b mu_a - 2 b' mu_b + 2 Bt
            A[i, i] = 2 + delta
            A[i, P + i] = 2 * mu_b[n, m]
            r[i] = (2 - delta) * Xa[n, m] + 2 * a0[n, m] * delta - 2 * Xb[n, m] * mu_a[n, m] + 2 * Bt[n, m]
            # (25)+(27): 2b' - 2b = -(b + b') d + 2 a mu_a + 2 a' mu_b + 2 At
            A[P + i, P + i] = 2 + delta
            A[P + i, i] = -2 * mu_b[n, m]
            r[P + i] = (2 - delta) * Xb[n, m] + 2 * Xa[n, m] * mu_a[n, m] + 2 * At[n, m]
    z = np.linalg.solve(A, r)
    a1 = z[:P].reshape(N + 1, M1)
    b1 = z[P:].reshape(N + 1, M1)
    b1[0] = 0.0                       # eq. (23): b_0 is not an unknown
    return a1, b1


@pytest.mark.parametrize("N,M1", [(2, 4), (3, 5), (4, 6)])
def test_P10_dense_bruteforce_matches_T(N, M1):
    rng = np.random.default_rng(100 * N + M1)
    dt, B, E_dc, E_w, w = 0.05, 1.3, 0.8, 0.4, 2.0
    s, p = make(N, M1, dt, E_dc=E_dc, E_omega=E_w, omega=w, B=B, mu=1.5, phiy_min=-2.0, phiy_max=2.0)
    phi, a0 = s.equilibrium()
    dphi = 4.0 / (M1 - 1)
    Xa = rng.standard_normal((N + 1, M1)); Xb = rng.standard_normal((N + 1, M1)); Xb[0] = 0
    Sa = rng.standard_normal((N + 1, M1)); Sb = rng.standard_normal((N + 1, M1)); Sb[0] = 0
    ta, tb = 0.35, 0.40
    Ea = E_dc + E_w * math.cos(w * ta)
    Eb = E_dc + E_w * math.cos(w * tb)
    for target in (0, 1):
        s.set_state(target, Xa, Xb)
        s.set_state(1 - target, Sa, Sb)
        s.apply_T(target, dt, ta, tb)
        got_a, got_b = s.get_state(target)
        want_a, want_b = _dense_T(N, M1, dt, B, dphi, phi, a0, Ea, Eb, Xa, Xb, Sa, Sb)
        assert np.abs(got_a - want_a).max() < 5e-15 * 5
        assert np.abs(got_b - want_b).max() < 5e-15 * 5
        oa, ob = s.get_state(1 - target)       # the stencil grid is untouched
        assert np.array_equal(oa, Sa) and np.array_equal(ob, Sb)


def test_P10b_hand_evaluated_point():
    """One point by hand from eq. (28)-(37): N=2, M+1=3, state = unit impulses."""
    dt, B = 0.1, 2.0
    s, p = make(2, 3, dt, E_dc=1.0, B=B, mu=1.0, phiy_min=-1.0, phiy_max=1.0)
    phi, a0 = s.equilibrium()            # phi = (-1, 0, 1), dphi = 1
    Xa = np.zeros((3, 3)); Xb = np.zeros((3, 3)); Sa = np.zeros((3, 3)); Sb = np.zeros((3, 3))
    Xa[1, 1] = 3.0; Xb[1, 1] = -2.0
    Sa[0, 2] = 5.0; Sa[2, 0] = 7.0; Sb[2, 2] = 11.0
    s.set_state(0, Xa, Xb); s.set_state(1, Sa, Sb)
    s.apply_T(0, dt, 0.0, 0.0)
    a, b = s.get_state(0)
    kap = B * dt / 4.0                    # 0.05
    mu = 1 * (1.0 + B * 0.0) * dt / 2     # 0.05 at (n=1, m=1)
    Bt = kap * (11.0 - 0 - 0 + 0)         # b_{2,2} - b_{2,0} - b_{0,2} + b_{0,0}
    At = kap * (2.0 * (5.0 - 0.0) - 0.0 + 7.0)   # chi(1)=2: 2(a_{0,2} - a_{0,0}) - a_{2,2} + a_{2,0}
    g = 3.0 * 0.95 + 2.0 * mu + Bt + a0[1, 1] * dt
    h = -2.0 * 0.95 + 3.0 * mu + At
    det = 1.05 ** 2 + mu ** 2
    assert abs(a[1, 1] - (g * 1.05 - h * mu) / det) < 1e-15
    assert abs(b[1, 1] - (g * mu + h * 1.05) / det) < 1e-15


# ---------------------------------------------------------------------------------------------------
# P13 / P14: structure of T
# ---------------------------------------------------------------------------------------------------
def test_P13_checkerboard_independence():
    """The stencil (30)-(31) couples (n,m) only to (n+-1, m+-1) (Fig. 7 cross): sub-lattices with
    (n+m) even and odd never interact.  Perturb one even point; odd points stay bit-identical."""
    kw = dict(E_dc=2.0, E_omega=0.5, omega=1.5, B=1.5, mu=2.0, phiy_min=-8.0, phiy_max=8.0)
    s1, _ = make(9, 40, 0.01, **kw)
    s2, _ = make(9, 40, 0.01, **kw)
    s1.init_equilibrium(); s2.init_equilibrium()
    a, b = s2.get_state(0)
    a[4, 20] *= 1.5                       # 4 + 20 even
    s2.set_state(0, a, b)
    a, b = s2.get_state(1)
    b[3, 11] += 1e-3                      # 3 + 11 even
    s2.set_state(1, a, b)
    s1.step(30); s2.step(30)
    n, m = np.meshgrid(np.arange(10), np.arange(40), indexing="ij")
    odd = ((n + m) % 2) == 1
    for g in (0, 1):
        a1, b1 = s1.get_state(g); a2, b2 = s2.get_state(g)
        assert np.array_equal(a1[odd], a2[odd]) and np.array_equal(b1[odd], b2[odd])
        assert not np.array_equal(a1[~odd], a2[~odd])


def test_P14_T_is_affine():
    rng = np.random.default_rng(7)
    N, M1, dt = 5, 12, 0.03
    kw = dict(E_dc=1.0, E_omega=0.3, omega=2.0, B=1.0, mu=1.0, phiy_min=-3.0, phiy_max=3.0)

    def run(xa, xb, sa, sb):
        s, _ = make(N, M1, dt, **kw)
        s.set_state(0, xa, xb); s.set_state(1, sa, sb)
        s.step(3)
        return np.stack(s.get_state(0) + s.get_state(1))

    def rnd():
        v = rng.standard_normal((4, N + 1, M1))
        v[1, 0] = 0; v[3, 0] = 0
        return v

    x, y, z = rnd(), rnd(), np.zeros((4, N + 1, M1))
    r = run(*(x + y)) - run(*x) - run(*y) + run(*z)
    assert np.abs(r).max() < 1e-14


# ---------------------------------------------------------------------------------------------------
# stability reading C11 and frozen systems
# ---------------------------------------------------------------------------------------------------
def test_C11_stability_threshold():
    """|B| dt / dphi < 2 is needed by the staggered scheme (the paper calls it unconditionally stable,
    L23): ratio 1.9 stays bounded, 2.1 blows up."""
    def run(ratio):
        M1, ext = 81, 4.0
        dphi = 2 * ext / (M1 - 1)
        B = 2.0
        dt = ratio * dphi / B
        s, _ = make(12, M1, dt, E_dc=0.5, B=B, mu=4.0, phiy_min=-ext, phiy_max=ext)
        s.init_equilibrium()
        s.step(600)
        a, _b = s.get_state(0)
        return np.abs(a).max()
    assert run(1.9) < 10.0
    big = run(2.1)
    assert (not np.isfinite(big)) or big > 1e6


def test_frozen_system_stops_at_budget():
    s, _ = make(4, 21, 0.01, E_dc=1.0, mu=1.0, n_steps_total=25, avg_start_step=10)
    s.init_equilibrium()
    s.step(25)
    a1 = s.get_state(0)[0].copy()
    o1 = s.observables()
    s.step(10)
    o2 = s.observables()
    assert o2.step == 25 and np.array_equal(a1, s.get_state(0)[0])
    assert o1.sum_v_dt == o2.sum_v_dt and abs(o2.window - 15 * 0.01) < 1e-12


# ---------------------------------------------------------------------------------------------------
# NEXT-3: reconstruction of f(phi_x, phi_y), eq. (8)
# ---------------------------------------------------------------------------------------------------
def test_pdf_reconstruction_at_t0_is_eq13():
    """At t = 0 the state is the equilibrium, so the reconstructed f must be the Boltzmann distribution as
    printed in eq. (13) (up to the truncation at N harmonics: I_N(mu)/I_0(mu) ~ 1e-17 for mu = 2, N = 24)."""
    mu, alpha, N, M1, K = 2.0, 0.9496, 24, 65, 48
    s, p = make(N, M1, 0.01, mu=mu, alpha=alpha, phiy_min=-4.0, phiy_max=4.0)
    s.init_equilibrium()
    f = s.reconstruct_pdf(0, K)
    phi, _ = s.equilibrium()
    x = -np.pi + 2 * np.pi * np.arange(K) / K
    want = (1.0 / (2 * np.pi * special.ive(0, mu))) * math.sqrt(mu / (2 * np.pi * alpha)) * \
        np.exp(mu * (np.cos(x)[:, None] - 1.0) - 0.5 * mu * phi[None, :] ** 2)
    assert f.shape == (K, M1)
    assert np.abs(f - want).max() <= 1e-14 * want.max()
    # and it integrates to 1: sqrt(alpha) int int f dphi_x dphi_y = 1, eq. (6)
    dphi = phi[1] - phi[0]
    assert abs(math.sqrt(alpha) * f.sum() * (2 * np.pi / K) * dphi - 1.0) < 1e-6   # phi_y cut at +-4


def test_pdf_reconstruction_is_the_fourier_sum_of_any_state():
    """Random state with sine terms: compare with a numpy contraction over n (b_n sin(n phi_x) included, sign
    and the phi_x origin at -pi)."""
    rng = np.random.default_rng(11)
    N, M1, K = 5, 7, 16
    s, _ = make(N, M1, 0.01, phiy_min=-1.0, phiy_max=1.0)
    a, b = rng.standard_normal((N + 1, M1)), rng.standard_normal((N + 1, M1))
    b[0] = 0.0
    s.set_state(1, a, b)
    f = s.reconstruct_pdf(1, K)
    x = -np.pi + 2 * np.pi * np.arange(K) / K
    n = np.arange(N + 1)
    want = np.einsum("in,nm->im", np.cos(np.outer(x, n)), a) + np.einsum("in,nm->im", np.sin(np.outer(x, n)), b)
    assert np.abs(f - want).max() <= 1e-13
    assert abs(f[K // 2, 3] - a[:, 3].sum()) <= 1e-13            # phi_x = 0: cos = 1, sin = 0


# ---------------------------------------------------------------------------------------------------
# NEXT-2: zero-temperature pendulum model, eq. (44)-(46)
# ---------------------------------------------------------------------------------------------------
def test_pendulum_dc_B0_is_esaki_tsu_at_T0():
    """B = 0, dc field: phi_x = E s, so <v_dr> = int_0^S e^{-s} sin(E s) ds in closed form (S -> inf: E/(1+E^2))."""
    from oracle import pendulum_averages
    for E in (0.3, 1.0, 2.5):
        S, h = 40.0, 0.005
        v, vc, vs = pendulum_averages(E, 0.0, 0.0, 0.0, 1, h, int(round(S / h)))
        want = (E - math.exp(-S) * (E * math.cos(E * S) + math.sin(E * S))) / (1 + E * E)
        assert abs(v - want) < 1e-10                  # Simpson: O(h^4)
        assert abs(want - E / (1 + E * E)) < 1e-15


def test_pendulum_ac_B0_is_tucker_at_T0():
    """B = 0 with an ac field: the Tucker sums (eq. 42-43) with I1/I0 -> 1 (mu -> infinity)."""
    from oracle import pendulum_averages
    from parity_util import tucker_averages
    E_dc, E_w, w = 2.0, 0.5, 1.5
    from parity_util import tucker_sin_average
    v, vc, vs = pendulum_averages(E_dc, E_w, w, 0.0, 64, 0.004, 10000)
    r = float(special.ive(1, 1e6) / special.ive(0, 1e6))       # -> 1
    v_ref, vc_ref, _ = tucker_averages(1e6, E_dc, E_w, w)
    vs_ref = tucker_sin_average(1e6, E_dc, E_w, w)
    assert abs(v - v_ref / r) < 1e-9 and abs(vc - vc_ref / r) < 1e-9
    assert abs(vs_ref) > 3 * abs(vc_ref) and abs(vs - vs_ref / r) < 1e-9        # third output: <v_dr sin wt>


def test_P11_low_temperature_oracle_approaches_the_pendulum_model():
    """P11 (Fig. 4b parameters B = 4, E_dc = 6, E_omega = 0.1, alpha = 0.9496, mu = 116): the
    oracle's time averages against the T = 0 pendulum model (itself pinned by the closed forms above), on a lattice
    small enough for the CPU suite.  "Very close, but not quite, due to the finite temperature" (L225): <v_dr> within
    2 %, the absorption within 15 % of the pendulum value."""
    from oracle import pendulum_averages
    from parity_util import absorption
    mu, E_dc, E_w, B, alpha, om, dt = 116.0, 6.0, 0.1, 4.0, 0.9496, 5.0, 0.004
    n_relax = int(round(10.0 / dt))
    n_avg = int(round(4 * 2 * math.pi / (om * dt)))
    s, _ = make(64, 501, dt, E_dc=E_dc, E_omega=E_w, omega=om, B=B, mu=mu, alpha=alpha, phiy_min=-5.0, phiy_max=5.0,
                avg_start_step=n_relax)
    s.init_equilibrium()
    s.step(n_relax + n_avg)
    o = s.observables()
    v_p, vc_p, vs_p = pendulum_averages(E_dc, E_w, om, B, 64, 0.004, 10000)
    assert abs(o.norm - 1.0) < 1e-6
    assert abs(o.sum_v_dt / o.window - v_p) < 0.02 * abs(v_p)
    assert abs(absorption(o, mu) - 2.0 * vc_p) < 0.15 * max(abs(2.0 * vc_p), 0.02)
    assert abs(o.sum_vsin_dt / o.window - vs_p) < 0.15 * max(abs(vs_p), 0.01)


def test_pendulum_energy_invariant_and_phase_count():
    """Constant E: (E + B phi_y)^2 / 2 - B^2 cos(phi_x) is conserved by (44)-(45) (RK4: to O(h^4)); and the phase
    average is converged (64 vs 128 start phases agree: periodic rectangle rule)."""
    from oracle import pendulum_averages, pendulum_trajectory
    E, B, h = 3.0, 2.0, 0.002
    px, py = pendulum_trajectory(E, 0.0, 0.0, B, 0.0, h, 10000)
    inv = 0.5 * (E + B * py) ** 2 - B * B * np.cos(px)
    assert np.abs(inv - inv[0]).max() < 1e-9 * abs(inv[0])
    a = pendulum_averages(6.0, 0.1, 4.0, 4.0, 64, 0.004, 7500)
    b = pendulum_averages(6.0, 0.1, 4.0, 4.0, 128, 0.004, 7500)
    assert max(abs(x - y) for x, y in zip(a, b)) < 1e-10


# ---------------------------------------------------------------------------------------------------
# NEXT-4: fp32 storage / fp32 arithmetic (the paper's precision, L311) and its time-step floor (L328)
# ---------------------------------------------------------------------------------------------------
def _run_prec(precision, dt, t_end, N=8, M1=81):
    from paper_1401_6047_b200 import workloads as W
    w = W.small_case(N=N, M1=M1, dt=dt, E_dc=2.0, E_omega=0.0, omega=0.0, B=1.0, mu=2.0, phiy_max=6.0)
    sim = OracleSim(N, M1, dt, w.params[0], threads=2, precision=precision)
    sim.init_equilibrium()
    sim.step(int(round(t_end / dt)))
    return sim


def test_fp32_modes_stay_close_to_fp64_and_hold_fp32_values():
    ref = _run_prec(0, 0.004, 0.4)
    ra, rb = ref.get_state(0)
    scale = max(np.abs(ra).max(), np.abs(rb).max())
    for prec in (1, 2):
        s = _run_prec(prec, 0.004, 0.4)
        a, b = s.get_state(0)
        assert np.array_equal(a, a.astype(np.float32).astype(np.float64))      # exactly representable in fp32
        assert np.array_equal(b, b.astype(np.float32).astype(np.float64))
        err = max(np.abs(a - ra).max(), np.abs(b - rb).max()) / scale
        assert 0 < err < 1e-5, (prec, err)                                      # O(eps32 / dt), not zero
        assert abs(s.observables().v_dr - ref.observables().v_dr) < 1e-5


def test_fp32_norm_drift_grows_as_dt_shrinks():
    """in float the norm of f drifts away from 1 when the time step gets small (the paper saw it
    'diverge' for dt <= 1e-5).  Every step adds a rounding error O(eps32) that the relaxation removes at rate dt, so
    the drift at fixed t scales like eps32 / dt; in fp64 it is invisible."""
    drift = {dt: abs(_run_prec(2, dt, 0.5).observables().norm - 1.0) for dt in (1e-2, 1e-3, 1e-4)}
    assert drift[1e-3] > 3 * drift[1e-2] and drift[1e-4] > 3 * drift[1e-3], drift
    assert drift[1e-4] > 3e-5
    assert abs(_run_prec(0, 1e-4, 0.5).observables().norm - 1.0) < 1e-12
    d1 = abs(_run_prec(1, 1e-4, 0.5).observables().norm - 1.0)
    assert 1e-8 < d1 < drift[1e-4] / 10      # storage rounding alone: unbiased, a random walk -- far smaller


# ---------------------------------------------------------------------------------------------------
# P12: finite-temperature characteristics (Chambers path integral) -- an absolute pin for B != 0
# ---------------------------------------------------------------------------------------------------
def _chambers_drift_velocity(E, B, mu, nx=96, ny=160, h=0.01, s_max=24.0):
    """Exact steady solution of eq. (5) for constant fields by the method of characteristics ("closely
    related to the method of characteristic curves"; eq. (46) generalised from the T = 0 delta function to the Boltzmann
    f0 of eq. (13)):  f(phi, t) = int_0^inf ds e^-s f0(phi(t - s)) along the characteristics (44)-(45), whose flow is
    area preserving (the divergence of (E + B phi_y, -B sin phi_x) vanishes), hence

        v_dr = int_0^inf ds e^-s < sin phi_x(s) >,   (phi_x, phi_y)(0) drawn from f0.

    f0 factorises (eq. 13): phi_x ~ exp(mu cos phi_x), phi_y ~ N(0, 1/mu).  Both averages by the rectangle rule on uniform
    nodes (periodic in phi_x, +-7 sigma in phi_y: spectrally accurate once the phase mixing exp(i B s phi_y) is resolved;
    Gauss-Hermite nodes converge much more slowly here).  Trajectories by classical RK4, the s-integral by the
    trapezoidal rule on the RK4 nodes (error ~ h^2 / 12).  Nothing of the finite-difference scheme enters.  Converged to
    ~1e-5 (E, B, mu = 2, 1, 2) and ~5e-5 (3, 2, 1) against nx, ny = 128, 256, h = 0.005."""
    px = -np.pi + 2 * np.pi * (np.arange(nx) + 0.5) / nx
    wx = np.exp(mu * (np.cos(px) - 1.0)); wx /= wx.sum()
    ymax = 7.0 / math.sqrt(mu)
    py = -ymax + 2 * ymax * (np.arange(ny) + 0.5) / ny
    wy = np.exp(-0.5 * mu * py * py); wy /= wy.sum()
    X, Y = np.meshgrid(px, py, indexing="ij")
    Wt = wx[:, None] * wy[None, :]

    def rhs(x, y):
        return E + B * y, -B * np.sin(x)

    n = int(round(s_max / h))
    acc = 0.5 * np.sum(Wt * np.sin(X))                     # trapezoid: half weight at s = 0
    for k in range(1, n + 1):
        k1x, k1y = rhs(X, Y)
        k2x, k2y = rhs(X + 0.5 * h * k1x, Y + 0.5 * h * k1y)
        k3x, k3y = rhs(X + 0.5 * h * k2x, Y + 0.5 * h * k2y)
        k4x, k4y = rhs(X + h * k3x, Y + h * k3y)
        X = X + h / 6.0 * (k1x + 2 * k2x + 2 * k3x + k4x)
        Y = Y + h / 6.0 * (k1y + 2 * k2y + 2 * k3y + k4y)
        acc += (0.5 if k == n else 1.0) * math.exp(-k * h) * np.sum(Wt * np.sin(X))
    return acc * h


def test_P12_chambers_integral_reduces_to_esaki_tsu_at_B0():
    """The validator itself, pinned: at B = 0 the path integral is (I1/I0) E / (1 + E^2) in closed form."""
    E, mu = 1.3, 2.0
    ref = special.iv(1, mu) / special.iv(0, mu) * E / (1.0 + E * E)
    assert abs(_chambers_drift_velocity(E, 0.0, mu, nx=64, ny=16, h=0.01) - ref) < 2e-5    # trapezoid in s: O(h^2)


@pytest.mark.parametrize("E,B,mu,N,M1,dt", [(2.0, 1.0, 2.0, 40, 401, 0.004),      # config 1's fields, dc part
                                            (3.0, 2.0, 1.0, 48, 481, 0.004)])     # config 4's fields, dc part
def test_P12_steady_drift_velocity_in_crossed_fields_matches_the_characteristics(E, B, mu, N, M1, dt):
    """Absolute pin at B != 0: the oracle's steady v_dr in crossed dc fields at finite temperature against
    the exact solution of eq. (5) by characteristics.  Every term of eq. (30)-(33) takes part (the phi_y stencil with
    its signs and chi(1) = 2, the rotation n (E + B phi_y), the relaxation), so a dropped term, a wrong sign or a
    transposed index moves v_dr by far more than the 5e-4 asked for (the discretisation error is O(dt^2 + dphi^2))."""
    ymax = W.phiy_extent(mu, E, 0.0, B, dt, M1)
    s, p = make(N, M1, dt, E_dc=E, B=B, mu=mu, phiy_min=-ymax, phiy_max=ymax)
    s.threads = 4
    s.init_equilibrium()
    s.step(int(round(24.0 / dt)))
    o = s.observables()
    ref = _chambers_drift_velocity(E, B, mu)
    assert abs(o.norm - 1.0) < 1e-10 and o.edge_leak < 1e-12
    assert abs(o.v_dr - ref) < 5e-4 * max(abs(ref), 0.05), (o.v_dr, ref)


# ---------------------------------------------------------------------------------------------------
# NEXT-1: steady-state detection and averaging policy (C23)
# ---------------------------------------------------------------------------------------------------
def _tucker_averages(E_dc, E_w, w, mu, nmax=40):
    """<v> and <v cos wt> of eq. (42)-(43) in the normalisation of C9."""
    beta = E_w / w
    r = special.iv(1, mu) / special.iv(0, mu)
    n = np.arange(-nmax, nmax + 1)
    xi = (E_dc + n * w) / (1.0 + (E_dc + n * w) ** 2)
    J = special.jv(n, beta)
    return r * np.sum(J * J * xi), 0.5 * r * np.sum(J * (special.jv(n + 1, beta) + special.jv(n - 1, beta)) * xi)


def test_steady_policy_gives_the_tucker_averages_without_a_hand_set_window():
    """B = 0, Fig. 3-like fields: the policy finds the relaxed state by itself and averages an integer number of
    periods; the result is the closed form of eq. (42)-(43) (P9 reaches the same with a hand-set window)."""
    E_dc, E_w, w, mu, dt = 2.0, 0.5, 1.5, 2.0, 0.002
    s, p = make(2, 41, dt, E_dc=E_dc, E_omega=E_w, omega=w, mu=mu, phiy_min=-6.0, phiy_max=6.0)
    s.set_steady_policy(1e-7, 3, 0)
    s.init_equilibrium()
    s.step(40000)
    step, phase = s.steady_info()
    o = s.observables()
    P = round(2 * math.pi / (w * dt))
    assert phase == 2 and step > 0 and step % P == 0
    assert abs(o.window - round(3 * 2 * math.pi / (w * dt)) * dt) < 1e-9
    v, vc = _tucker_averages(E_dc, E_w, w, mu)
    assert abs(o.sum_v_dt / o.window - v) < 2e-4 * abs(v)
    assert abs(o.sum_vcos_dt / o.window - vc) < 2e-3 * abs(vc) + 1e-6
    # finished: the sums are final however long the system is stepped
    before = (o.sum_v_dt, o.sum_vcos_dt, o.sum_vsin_dt, o.window)
    s.step(777)
    o2 = s.observables()
    assert (o2.sum_v_dt, o2.sum_vcos_dt, o2.sum_vsin_dt, o2.window) == before and o2.step == 40777


def test_steady_policy_detection_time_follows_the_relaxation_law():
    """Relaxation-time scattering: the transient decays like e^{-t} (tau = 1), so tightening the tolerance by a factor
    F delays the detection by ln F, up to the granularity of one comparison interval."""
    E_dc, E_w, w, mu, dt = 3.0, 0.3, 4.0, 1.0, 0.004
    P = round(2 * math.pi / (w * dt))
    t = {}
    for tol in (1e-3, 1e-6):
        s, p = make(16, 11, dt, E_dc=E_dc, E_omega=E_w, omega=w, mu=mu, phiy_min=-6.0, phiy_max=6.0)
        s.set_steady_policy(tol, 1, 0)
        s.init_equilibrium()
        s.step(12000)
        step, phase = s.steady_info()
        assert phase == 2 and step % P == 0
        t[tol] = step * dt
    assert abs((t[1e-6] - t[1e-3]) - math.log(1e3)) <= 1.5 * P * dt, t


def test_steady_policy_window_equals_a_hand_set_window_bit_for_bit():
    """The accumulation itself is the pinned one (P9): a second run with avg_start_step = detected step and a budget at
    the end of the window gives the same sums to the last bit.  Also: a dc system compares intervals of one relaxation
    time, min_relax_periods delays the detection, tol = 0 switches the policy off."""
    kw = dict(E_dc=1.5, E_omega=0.4, omega=2.5, B=1.0, mu=2.0, phiy_min=-8.0, phiy_max=8.0)
    dt = 0.005
    s, p = make(14, 81, dt, **kw)
    s.set_steady_policy(1e-5, 2, 0)
    s.init_equilibrium()
    s.step(9000)
    step, phase = s.steady_info()
    assert phase == 2
    o = s.observables()
    P = round(2 * math.pi / (2.5 * dt))
    s2, _ = make(14, 81, dt, n_steps_total=step + round(2 * 2 * math.pi / (2.5 * dt)), avg_start_step=step, **kw)
    s2.init_equilibrium()
    s2.step(9000)
    o2 = s2.observables()
    assert (o.sum_v_dt, o.sum_vcos_dt, o.sum_vsin_dt, o.window) == (o2.sum_v_dt, o2.sum_vcos_dt, o2.sum_vsin_dt, o2.window)
    s3, _ = make(14, 81, dt, **kw)
    s3.set_steady_policy(1e-5, 2, 12)
    s3.init_equilibrium()
    s3.step(9000)
    assert s3.steady_info() == (12 * P, 2) and 12 * P > step
    sd, _ = make(6, 11, dt, E_dc=1.0, mu=1.0)
    sd.set_steady_policy(1e-6, 1, 0)
    sd.init_equilibrium()
    sd.step(6000)
    st_dc, ph_dc = sd.steady_info()
    assert ph_dc == 2 and st_dc % round(1.0 / dt) == 0 and abs(sd.observables().window - 1.0) < 1e-9
    s4, _ = make(6, 11, dt, avg_start_step=10, **kw)
    s4.set_steady_policy(0.0, 1, 0)
    s4.init_equilibrium()
    s4.step(50)
    assert s4.steady_info() == (0, 0) and abs(s4.observables().window - 40 * dt) < 1e-12
