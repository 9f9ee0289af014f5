"""ctypes wrapper of oracle/bte_oracle.cpp (TEST INFRASTRUCTURE; argument marshalling only).

All of the method's arithmetic is in the C++ file, which cites PAPER.md passage by passage.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass

import numpy as np

from . import build as _build


class _Params(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("E_dc", "E_omega", "omega", "B", "mu", "alpha", "phiy_min",
                                          "phiy_max", "kappa_scale")] + \
               [("n_steps_total", C.c_int64), ("avg_start_step", C.c_int64)]


class _Obs(C.Structure):
    _fields_ = [("step", C.c_int64)] + [(k, C.c_double) for k in (
        "t", "norm", "v_dr", "sum_v_dt", "sum_vcos_dt", "sum_vsin_dt", "window", "edge_leak")]


@dataclass
class OracleObs:
    step: int
    t: float
    norm: float
    v_dr: float
    sum_v_dt: float
    sum_vcos_dt: float
    sum_vsin_dt: float
    window: float
    edge_leak: float


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(_build.build())
        lib.oracle_create.restype = C.c_void_p
        lib.oracle_create.argtypes = [C.c_int32, C.c_int32, C.c_double, C.POINTER(_Params), C.c_int32]
        lib.oracle_destroy.argtypes = [C.c_void_p]
        lib.oracle_set_precision.argtypes = [C.c_void_p, C.c_int32]
        lib.oracle_init_equilibrium.argtypes = [C.c_void_p]
        lib.oracle_startup_from_whole.argtypes = [C.c_void_p]
        lib.oracle_step.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
        lib.oracle_observables.argtypes = [C.c_void_p, C.POINTER(_Obs)]
        lib.oracle_get_state.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
        lib.oracle_set_state.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
        lib.oracle_get_equilibrium.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        lib.oracle_apply_T.argtypes = [C.c_void_p, C.c_int32, C.c_double, C.c_double, C.c_double]
        lib.oracle_reconstruct_pdf.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p]
        lib.oracle_pendulum_averages.argtypes = [C.c_double] * 4 + [C.c_int32, C.c_double, C.c_int32, C.c_void_p]
        lib.oracle_pendulum_trajectory.argtypes = [C.c_double] * 6 + [C.c_int32, C.c_void_p, C.c_void_p]
        lib.oracle_set_steady_policy.argtypes = [C.c_void_p, C.c_double, C.c_int32, C.c_int32]
        lib.oracle_steady_info.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int32)]
        lib.oracle_max_threads.restype = C.c_int32
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def pendulum_averages(E_dc, E_omega, omega, B, n_phase, h, n_rk):
    """(<v_dr>, <v_dr cos wt>, <v_dr sin wt>) of the zero-temperature pendulum model, eq. (44)-(46)."""
    out = np.zeros(3)
    _load().oracle_pendulum_averages(E_dc, E_omega, omega, B, n_phase, h, n_rk, out.ctypes.data)
    return tuple(float(x) for x in out)


def pendulum_trajectory(E_dc, E_omega, omega, B, t0, h, n_rk):
    px, py = np.zeros(n_rk + 1), np.zeros(n_rk + 1)
    _load().oracle_pendulum_trajectory(E_dc, E_omega, omega, B, t0, h, n_rk, px.ctypes.data, py.ctypes.data)
    return px, py


class OracleSim:
    """One system.  `params` is any object with the fields of workloads.Params."""

    def __init__(self, n_harm: int, n_phiy: int, dt: float, params, threads: int = 1, precision: int = 0):
        """precision: 0 = fp64, 1 = state stored in fp32 / fp64 arithmetic, 2 = fp32 throughout (NEXT-4)."""
        lib = _load()
        p = _Params(params.E_dc, params.E_omega, params.omega, params.B, params.mu, params.alpha,
                    params.phiy_min, params.phiy_max, params.kappa_scale,
                    int(params.n_steps_total), int(params.avg_start_step))
        self._h = lib.oracle_create(n_harm, n_phiy, dt, C.byref(p), threads)
        if not self._h:
            raise ValueError("oracle_create: invalid arguments")
        lib.oracle_set_precision(self._h, precision)
        self.N, self.M1, self.dt, self.threads = n_harm, n_phiy, dt, threads
        self.shape = (n_harm + 1, n_phiy)

    def close(self):
        if self._h:
            _load().oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def init_equilibrium(self):
        _load().oracle_init_equilibrium(self._h)

    def set_steady_policy(self, rel_tol: float, n_avg_periods: int, min_relax_periods: int = 0):
        """Steady-state detection and averaging policy (C23); rel_tol = 0 switches it off."""
        _load().oracle_set_steady_policy(self._h, float(rel_tol), int(n_avg_periods), int(min_relax_periods))

    def steady_info(self):
        st, ph = C.c_int64(), C.c_int32()
        _load().oracle_steady_info(self._h, C.byref(st), C.byref(ph))
        return int(st.value), int(ph.value)

    def startup_from_whole(self):
        _load().oracle_startup_from_whole(self._h)

    def step(self, n_steps: int, trace: bool = False):
        if trace:
            v = np.zeros(n_steps)
            nm = np.zeros(n_steps)
            _load().oracle_step(self._h, n_steps, v.ctypes.data, nm.ctypes.data)
            return v, nm
        _load().oracle_step(self._h, n_steps, None, None)
        return None

    def observables(self) -> OracleObs:
        o = _Obs()
        _load().oracle_observables(self._h, C.byref(o))
        return OracleObs(*[getattr(o, f[0]) for f in _Obs._fields_])

    def get_state(self, grid: int):
        a = np.empty(self.shape)
        b = np.empty(self.shape)
        _load().oracle_get_state(self._h, grid, a.ctypes.data, b.ctypes.data)
        return a, b

    def set_state(self, grid: int, a, b):
        a = np.ascontiguousarray(a, dtype=np.float64)
        b = np.ascontiguousarray(b, dtype=np.float64)
        assert a.shape == self.shape and b.shape == self.shape
        _load().oracle_set_state(self._h, grid, a.ctypes.data, b.ctypes.data)

    def equilibrium(self):
        phi = np.empty(self.M1)
        a0 = np.empty(self.shape)
        _load().oracle_get_equilibrium(self._h, phi.ctypes.data, a0.ctypes.data)
        return phi, a0

    def reconstruct_pdf(self, grid: int, n_phix: int):
        """f(phi_x, phi_y) of eq. (8) on phi_x = -pi + 2 pi i / n_phix; returns (n_phix, n_phiy)."""
        f = np.empty((n_phix, self.M1))
        _load().oracle_reconstruct_pdf(self._h, grid, n_phix, f.ctypes.data)
        return f

    def apply_T(self, target: int, delta: float, ta: float, tb: float):
        _load().oracle_apply_T(self._h, target, delta, ta, tb)
