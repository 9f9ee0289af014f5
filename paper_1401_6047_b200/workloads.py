"""Seeded, synthetic workload generator shared by the CUDA path, the oracle tests and bench.py.

This module holds NONE of the method's arithmetic (no stencil, no solve, no equilibrium): it only
turns the five BASELINE.json configs into concrete (grid, params[]) records -- plain Python numbers --
that both the C-ABI library and the CPU oracle are fed with.  The recipe is stated in DESIGN.md
("Input recipe") and follows SURVEY.md section 8(d):

* phi_y extent rule (the paper adjusts it "manually"; its own run uses +-6, L325):
      w_th  = sqrt(2 ln(1e12) / mu)                      thermal width where f0 drops to 1e-12
      E_max = |E_dc| + |E_omega|
      D     = 0 if B == 0 else min(B ln(1e12), (E_max + sqrt(E_max^2 + 4 B^2)) / B)
      phiy_max = max(ceil(2 (w_th + D)) / 2,  |B| dt M / 2),   phiy_min = -phiy_max
  The second term keeps |B| dt / dphi <= 1 (stability of the staggered scheme, reading C11).
* config 3 draws per-system parameters from SplitMix64(seed = 14016047), u = (x >> 11) * 2^-53, in the
  order E_dc = 8u, omega = 0.5 + 7.5u, B = 5u, mu = 0.5 + 4.5u; E_omega = 0.1.

The paper uses no dataset: its workloads are parameter sets, so these
configs *are* the stand-ins; the state itself is always produced by the equilibrium initialisation.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, asdict
from typing import List

SEED_CONFIG3 = 14016047
_MASK64 = (1 << 64) - 1


@dataclass
class Grid:
    n_harm: int      # N   : highest harmonic kept, rows n = 0..N           (eq. 22)
    n_phiy: int      # M+1 : number of phi_y lattice points, m = 0..M       (eq. 22)
    n_batch: int     # independent systems sharing shape and dt
    dt: float        # time step in units of tau                            (PAPER.md:L325 `dt`)


@dataclass
class Params:
    E_dc: float
    E_omega: float
    omega: float
    B: float
    mu: float
    alpha: float = 1.0
    phiy_min: float = 0.0
    phiy_max: float = 0.0
    kappa_scale: float = 1.0
    n_steps_total: int = 0     # 0 = never freezes
    avg_start_step: int = 0


@dataclass
class Workload:
    name: str
    grid: Grid
    params: List[Params]
    n_steps: int                       # steps of the longest system (= what bte_step is asked for)
    note: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def points_per_system(self) -> int:
        return (self.grid.n_harm + 1) * self.grid.n_phiy

    def total_updates(self, n_steps: int | None = None) -> int:
        """Grid-point updates (whole + fractional counted once) over all systems."""
        tot = 0
        for p in self.params:
            s = self.n_steps if n_steps is None else n_steps
            if p.n_steps_total > 0:
                s = min(s, p.n_steps_total)
            tot += self.points_per_system * s
        return tot

    def updates_between(self, k0: int, k1: int) -> int:
        """Grid-point updates done by steps k0 < k <= k1 of the job (systems past their budget do none)."""
        tot = 0
        for p in self.params:
            a, b = k0, k1
            if p.n_steps_total > 0:
                a, b = min(a, p.n_steps_total), min(b, p.n_steps_total)
            tot += self.points_per_system * (b - a)
        return tot

    def describe(self) -> dict:
        d = asdict(self.grid)
        d.update(name=self.name, n_steps=self.n_steps, note=self.note)
        return d


def phiy_extent(mu: float, E_dc: float, E_omega: float, B: float, dt: float, n_phiy: int) -> float:
    """phi_y half-extent by the rule in the module docstring (input recipe, not method arithmetic)."""
    L = math.log(1e12)
    w_th = math.sqrt(2.0 * L / mu)
    e_max = abs(E_dc) + abs(E_omega)
    if B == 0.0:
        D = 0.0
    else:
        b = abs(B)
        D = min(b * L, (e_max + math.sqrt(e_max * e_max + 4.0 * b * b)) / b)
    thermal = math.ceil(2.0 * (w_th + D)) / 2.0
    cfl = abs(B) * dt * (n_phiy - 1) / 2.0
    return max(thermal, cfl)


def steps_for_periods(periods: float, omega: float, dt: float) -> int:
    return int(round(periods * 2.0 * math.pi / (omega * dt)))


class SplitMix64:
    """Counter-based generator used for config 3 (public-domain algorithm, restated)."""

    def __init__(self, seed: int):
        self.state = seed & _MASK64

    def next_u64(self) -> int:
        self.state = (self.state + 0x9E3779B97F4A7C15) & _MASK64
        z = self.state
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK64
        return z ^ (z >> 31)

    def uniform(self) -> float:
        return (self.next_u64() >> 11) * (1.0 / 9007199254740992.0)


def _single(name, N, M1, dt, n_steps, E_dc, E_omega, omega, B, mu, avg_start, note, alpha=1.0):
    ext = phiy_extent(mu, E_dc, E_omega, B, dt, M1)
    p = Params(E_dc=E_dc, E_omega=E_omega, omega=omega, B=B, mu=mu, alpha=alpha,
               phiy_min=-ext, phiy_max=ext, kappa_scale=1.0, n_steps_total=0,
               avg_start_step=avg_start)
    return Workload(name=name, grid=Grid(N, M1, 1, dt), params=[p], n_steps=n_steps, note=note)


def config0() -> Workload:
    """B=0, dc only: 20 harmonics x 201 phi_y points, dt=0.005, 4000 steps (BASELINE.json configs[0])."""
    return _single("config0_dc_B0", 20, 201, 0.005, 4000, 1.0, 0.0, 0.0, 0.0, 1.0, 0,
                   "steady v_dr checked against (I1/I0) E/(1+E^2)")


def config1() -> Workload:
    """Crossed fields dc+ac: 50 x 1001, dt=0.002, 30 ac periods (BASELINE.json configs[1])."""
    n = steps_for_periods(30, 1.5, 0.002)
    return _single("config1_crossed_ac", 50, 1001, 0.002, n, 2.0, 0.5, 1.5, 1.0, 2.0,
                   n - steps_for_periods(20, 1.5, 0.002), "averages over the last 20 periods")


def config2() -> Workload:
    """Paper-scale single run: 150 x 4001, dt=0.001, 50 ac periods (BASELINE.json configs[2])."""
    n = steps_for_periods(50, 4.0, 0.001)
    return _single("config2_paper_scale", 150, 4001, 0.001, n, 6.0, 0.1, 4.0, 4.0, 10.0,
                   n - steps_for_periods(30, 4.0, 0.001), "averages over the last 30 periods")


def config3(n_batch: int = 512, seed: int = SEED_CONFIG3) -> Workload:
    """Batched sweep: n_batch systems of 40 x 801, dt=0.002, 20 ac periods each (configs[3])."""
    N, M1, dt = 40, 801, 0.002
    rng = SplitMix64(seed)
    ps = []
    longest = 0
    for _ in range(n_batch):
        E_dc = 8.0 * rng.uniform()
        omega = 0.5 + 7.5 * rng.uniform()
        B = 5.0 * rng.uniform()
        mu = 0.5 + 4.5 * rng.uniform()
        E_omega = 0.1
        ext = phiy_extent(mu, E_dc, E_omega, B, dt, M1)
        total = steps_for_periods(20, omega, dt)
        longest = max(longest, total)
        ps.append(Params(E_dc=E_dc, E_omega=E_omega, omega=omega, B=B, mu=mu, alpha=1.0,
                         phiy_min=-ext, phiy_max=ext, kappa_scale=1.0,
                         n_steps_total=total, avg_start_step=total // 2))
    return Workload(name="config3_batched_sweep", grid=Grid(N, M1, n_batch, dt), params=ps,
                    n_steps=longest, note="per-system step budget = 20 ac periods; averages over the last 10",
                    extra={"seed": seed})


def config4() -> Workload:
    """Bandwidth stress: 512 x 32001 (~263 MB per (a,b) grid), dt=0.001, 2000 steps (configs[4])."""
    return _single("config4_bandwidth_stress", 512, 32001, 0.001, 2000, 3.0, 1.0, 2.0, 2.0, 1.0, 0,
                   "transient to t=2; state 525 MB > L2 => HBM streaming")


def paper_table1() -> Workload:
    """The paper's own timing run (Table 1): n-harmonics=120, g-grid=4000, dt=0.0001, t-max=10
    (1e5 steps), E_dc=7, E_omega=0.1, omega=10, B=4, mu=116, alpha=0.9496, PhiYmin=-6, PhiYmax=6.  The paper ran it in
    fp32 and counts MLUPS as n-harmonics x g-grid x steps / time.  Context workload (index 5), not a BASELINE config."""
    p = Params(E_dc=7.0, E_omega=0.1, omega=10.0, B=4.0, mu=116.0, alpha=0.9496, phiy_min=-6.0, phiy_max=6.0,
               kappa_scale=1.0, n_steps_total=0, avg_start_step=0)
    return Workload(name="paper_table1", grid=Grid(120, 4000, 1, 1e-4), params=[p], n_steps=100000,
                    note="the paper's Table 1 run (fp32 there): 1094 MLUPS on a GTX680, 9 MLUPS on one i7-3770 core")


CONFIGS = {0: config0, 1: config1, 2: config2, 3: config3, 4: config4, 5: paper_table1}
PAPER_TABLE1_MLUPS_K6 = 1094.0     # fastest CUDA kernel of the paper, GTX680, fp32


def absorption_sweep(omegas, E_dc: float, E_omega: float, B: float, mu: float, N: int, M1: int, dt: float,
                     t_relax: float = 10.0, periods: int = 8, alpha: float = 1.0) -> Workload:
    """The paper's use of the solver (Fig. 3, Fig. 4): one system per frequency omega_i, all
    other parameters shared.  Each system relaxes until t_relax (the paper: t = 10), then the
    running sums of eq. (17) cover an integer number of ac periods; the step budget ends the system there."""
    ps = []
    k_relax = int(round(t_relax / dt))
    longest = 0
    for w in omegas:
        ext = phiy_extent(mu, E_dc, E_omega, B, dt, M1)
        total = k_relax + steps_for_periods(periods, w, dt)
        longest = max(longest, total)
        ps.append(Params(E_dc=E_dc, E_omega=E_omega, omega=float(w), B=B, mu=mu, alpha=alpha, phiy_min=-ext,
                         phiy_max=ext, kappa_scale=1.0, n_steps_total=total, avg_start_step=k_relax))
    return Workload(name="absorption_sweep", grid=Grid(N, M1, len(ps), dt), params=ps, n_steps=longest,
                    note=f"A(omega): relax to t = {t_relax}, then {periods} ac periods per system")


def get(index: int) -> Workload:
    return CONFIGS[index]()


def small_case(N=12, M1=75, dt=0.004, n_steps=40, E_dc=1.3, E_omega=0.4, omega=2.0, B=1.5, mu=3.0,
               alpha=1.0, avg_start=10, n_batch=1, kappa_scale=1.0, phiy_max=None) -> Workload:
    """Arbitrary small single/batched case for parity tests (ragged sizes, several tiles)."""
    ext = phiy_extent(mu, E_dc, E_omega, B, dt, M1) if phiy_max is None else phiy_max
    ps = [Params(E_dc=E_dc, E_omega=E_omega, omega=omega, B=B, mu=mu, alpha=alpha, phiy_min=-ext,
                 phiy_max=ext, kappa_scale=kappa_scale, n_steps_total=0, avg_start_step=avg_start)
          for _ in range(n_batch)]
    return Workload(name="small_case", grid=Grid(N, M1, n_batch, dt), params=ps, n_steps=n_steps)


def random_batch(n_batch: int, N: int, M1: int, dt: float, seed: int, periods: float = 0.0,
                 n_steps: int = 50) -> Workload:
    """Config-3-shaped batch at arbitrary (small) size: same distributions, own seed."""
    rng = SplitMix64(seed)
    ps = []
    longest = 0
    for _ in range(n_batch):
        E_dc = 8.0 * rng.uniform()
        omega = 0.5 + 7.5 * rng.uniform()
        B = 5.0 * rng.uniform()
        mu = 0.5 + 4.5 * rng.uniform()
        ext = phiy_extent(mu, E_dc, 0.1, B, dt, M1)
        total = steps_for_periods(periods, omega, dt) if periods > 0 else 0
        longest = max(longest, total)
        ps.append(Params(E_dc=E_dc, E_omega=0.1, omega=omega, B=B, mu=mu, alpha=1.0, phiy_min=-ext,
                         phiy_max=ext, kappa_scale=1.0, n_steps_total=total,
                         avg_start_step=(total // 2 if total else n_steps // 2)))
    return Workload(name="random_batch", grid=Grid(N, M1, n_batch, dt), params=ps,
                    n_steps=(longest if periods > 0 else n_steps), extra={"seed": seed})
