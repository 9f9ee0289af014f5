"""Real-space-phi_x variant of the step -- TEST INFRASTRUCTURE (oracle), SURVEY 8(f) NEXT-5.

BASELINE.json's config 0 names it as the alternative to the harmonic representation ("20 phi_x harmonics (or 64
periodic phi_x points)").  It is NOT in the paper: the paper diagonalises the phi_x direction with the Fourier
representation (7)-(8), which turns the implicit Crank-Nicolson solve into the 2x2 blocks of eq. (32)-(33).  Kept in
real space, the same splitting of eq. (5),

    df/dt = -(E + B phi_y) df/dphi_x + B sin(phi_x) df/dphi_y + f0 - f,

gives one CYCLIC TRIDIAGONAL system per phi_y lattice row (reading C22 of DESIGN.md):

  lattice   phi_x_i = -pi + 2 pi i / K (periodic, dx = 2 pi / K), phi_y_m as in the harmonic form (C8); f = 0 outside m in [0, M]
  T_delta(X; S; ta, tb), for every m:   beta_a,b = E(ta,b) + B phi_m,   gamma_a,b = beta_a,b delta / (4 dx),
                                        kappa' = kappa_scale B delta / (2 dphi),   nu, xi = 1 +- delta / 2
      rhs_i = xi X_i - gamma_a (X_{i+1} - X_{i-1}) + kappa' sin(phi_x_i) (S_{i,m+1} - S_{i,m-1}) + f0_{i,m} delta
      nu X'_i + gamma_b (X'_{i+1} - X'_{i-1}) = rhs_i          (indices i cyclic)
  i.e. Crank-Nicolson for relaxation and the phi_x advection (centred differences), the phi_y derivative explicit from
  the OTHER grid -- exactly the roles the terms have in eq. (24)-(27); leap-frog over the two staggered grids
  (eq. 40-41) and the dt/2 start-up (L202) as in the harmonic form.
  observables: norm = sqrt(alpha) dx dphi sum f_h (eq. 6), v_dr = sqrt(alpha) dx dphi sum sin(phi_x_i) f_h (eq. 18-19).

The linear systems are solved with numpy's dense LAPACK solve on the explicitly assembled cyclic matrix.
Pins (tests/test_rs_oracle_pins.py): f0 is a fixed point at E = B = 0; the norm is conserved to rounding; at B = 0 the
steady drift velocity is the Esaki-Tsu form with the modified wavenumber of the centred difference, in closed form;
second-order convergence to the harmonic-form oracle as K grows.
"""
from __future__ import annotations

import math

import numpy as np
from scipy import special


class RealSpaceSim:
    def __init__(self, K: int, n_phiy: int, dt: float, p):
        self.K, self.M1, self.dt, self.p = K, n_phiy, dt, p
        M = n_phiy - 1
        self.dx = 2.0 * math.pi / K
        self.dphi = (p.phiy_max - p.phiy_min) / M
        self.x = -math.pi + self.dx * np.arange(K)
        self.phi = 0.5 * (p.phiy_min + p.phiy_max) + (np.arange(n_phiy) - M / 2.0) * self.dphi      # C8
        g = np.exp(-p.mu * self.phi ** 2 / 2.0)
        g[g < 1e-300] = 0.0                                                                        # C19
        ex = np.exp(p.mu * (np.cos(self.x) - 1.0)) / special.ive(0, p.mu)                          # exp(mu cos x)/I0(mu)
        self.f0 = (1.0 / (2.0 * math.pi)) * math.sqrt(p.mu / (2.0 * math.pi * p.alpha)) * ex[:, None] * g[None, :]  # eq. (13)
        self.fh = np.zeros((K, n_phiy))
        self.ff = np.zeros((K, n_phiy))
        self.step_count = 0
        self.sum_v = self.sum_c = self.sum_s = self.window = 0.0

    def E(self, t):
        return self.p.E_dc + self.p.E_omega * math.cos(self.p.omega * t)

    def apply_T(self, delta, X, S, ta, tb):
        """Returns the new X (X and S are not modified)."""
        K, M1, p = self.K, self.M1, self.p
        nu, xi = 1.0 + delta / 2.0, 1.0 - delta / 2.0
        kap = p.kappa_scale * p.B * delta / (2.0 * self.dphi)
        Sp = np.zeros((K, M1 + 2))
        Sp[:, 1:-1] = S                                          # f = 0 outside m in [0, M]
        out = np.empty_like(X)
        sinx = np.sin(self.x)
        for m in range(M1):
            ga = (self.E(ta) + p.B * self.phi[m]) * delta / (4.0 * self.dx)
            gb = (self.E(tb) + p.B * self.phi[m]) * delta / (4.0 * self.dx)
            col = X[:, m]
            rhs = xi * col - ga * (np.roll(col, -1) - np.roll(col, 1)) + kap * sinx * (Sp[:, m + 2] - Sp[:, m]) \
                + self.f0[:, m] * delta
            A = nu * np.eye(K)
            for i in range(K):
                A[i, (i + 1) % K] += gb
                A[i, (i - 1) % K] -= gb
            out[:, m] = np.linalg.solve(A, rhs)
        return out

    def init_equilibrium(self):
        self.fh = self.f0.copy()
        self.ff = self.apply_T(self.dt / 2.0, self.fh, self.fh, 0.0, self.dt / 2.0)                # L202, C6
        self.step_count = 0
        self.sum_v = self.sum_c = self.sum_s = self.window = 0.0

    def step(self, n):
        dt = self.dt
        for _ in range(n):
            k = float(self.step_count)
            self.fh = self.apply_T(dt, self.fh, self.ff, k * dt, (k + 1.0) * dt)                   # eq. (40)
            self.ff = self.apply_T(dt, self.ff, self.fh, (k + 0.5) * dt, (k + 1.5) * dt)           # eq. (41), C5
            self.step_count += 1
            if self.step_count > self.p.avg_start_step:
                t = self.step_count * dt
                v = self.v_dr()
                self.sum_v += v * dt
                self.sum_c += v * math.cos(self.p.omega * t) * dt
                self.sum_s += v * math.sin(self.p.omega * t) * dt
                self.window += dt

    def norm(self):
        return math.sqrt(self.p.alpha) * self.dx * self.dphi * float(self.fh.sum())

    def v_dr(self):
        return math.sqrt(self.p.alpha) * self.dx * self.dphi * float((np.sin(self.x)[:, None] * self.fh).sum())
