"""Thin ctypes binding of libbte_b200.so (include/bte.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/.  PyTorch is used for exactly two things:
the device workspace (a uint8 tensor the library is handed) and the CUDA stream.  There is no CPU
fallback: if the shared library is missing or no CUDA device is present, construction raises.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import List, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbte_b200.so")

BTE_OK, BTE_EINVAL, BTE_EUNSTABLE, BTE_ENOMEM, BTE_ECUDA = 0, -1, -2, -3, -4

EXPORTS = ("bte_workspace_bytes", "bte_create", "bte_init_equilibrium", "bte_step", "bte_observables",
           "bte_destroy", "bte_get_state", "bte_set_state", "bte_get_state_batch", "bte_set_state_batch", "bte_get_option",
           "bte_reconstruct_pdf", "bte_pendulum_workspace_bytes",
           "bte_pendulum_averages", "bte_rs_workspace_bytes", "bte_rs_create", "bte_rs_init_equilibrium",
           "bte_rs_step", "bte_rs_observables", "bte_rs_get_state", "bte_rs_destroy", "bte_rs_evolve_static",
           "bte_set_option",
           "bte_launch_count", "bte_set_steady_policy", "bte_steady_info",
           "bte_last_error")


class BteError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libbte_b200 error {code}: {msg}")
        self.code = code


class bte_grid(C.Structure):
    _fields_ = [("n_harm", C.c_int32), ("n_phiy", C.c_int32), ("n_batch", C.c_int32),
                ("precision", C.c_int32), ("dt", C.c_double)]


class bte_rs_grid(C.Structure):
    _fields_ = [("n_phix", C.c_int32), ("n_phiy", C.c_int32), ("dt", C.c_double)]


class bte_params(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("E_dc", "E_omega", "omega", "B", "mu", "alpha", "phiy_min",
                                          "phiy_max", "kappa_scale")] + \
               [("n_steps_total", C.c_int64), ("avg_start_step", C.c_int64)]


class bte_obs(C.Structure):
    _fields_ = [("step", C.c_int64)] + [(k, C.c_double) for k in (
        "t", "norm", "v_dr", "sum_v_dt", "sum_vcos_dt", "sum_vsin_dt", "window", "edge_leak")]


@dataclass
class Obs:
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


def load_library(path: str = LIB_PATH) -> C.CDLL:
    """dlopen the C-ABI library and declare the prototypes of include/bte.h.  Fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise ImportError(f"{path} not found: build it with `python -m paper_1401_6047_b200.build` "
                          "(nvcc, sm_100a).  There is no CPU fallback.")
    lib = C.CDLL(path)
    lib.bte_workspace_bytes.restype = C.c_size_t
    lib.bte_workspace_bytes.argtypes = [C.POINTER(bte_grid)]
    lib.bte_create.restype = C.c_int
    lib.bte_create.argtypes = [C.POINTER(bte_grid), C.POINTER(bte_params), C.c_void_p, C.c_size_t,
                               C.c_void_p, C.POINTER(C.c_void_p)]
    for name in ("bte_init_equilibrium", "bte_destroy"):
        getattr(lib, name).restype = C.c_int
        getattr(lib, name).argtypes = [C.c_void_p]
    lib.bte_step.restype = C.c_int
    lib.bte_step.argtypes = [C.c_void_p, C.c_int64]
    lib.bte_observables.restype = C.c_int
    lib.bte_observables.argtypes = [C.c_void_p, C.POINTER(bte_obs)]
    lib.bte_get_state.restype = C.c_int
    lib.bte_get_state.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
    lib.bte_set_state.restype = C.c_int
    lib.bte_set_state.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
    for name in ("bte_get_state_batch", "bte_set_state_batch"):
        getattr(lib, name).restype = C.c_int
        getattr(lib, name).argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
    lib.bte_set_steady_policy.restype = C.c_int
    lib.bte_set_steady_policy.argtypes = [C.c_void_p, C.c_double, C.c_int32, C.c_int32]
    lib.bte_steady_info.restype = C.c_int
    lib.bte_steady_info.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int32)]
    lib.bte_get_option.restype = C.c_int
    lib.bte_get_option.argtypes = [C.c_void_p, C.c_char_p, C.POINTER(C.c_int64)]
    lib.bte_reconstruct_pdf.restype = C.c_int
    lib.bte_reconstruct_pdf.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_void_p]
    lib.bte_pendulum_workspace_bytes.restype = C.c_size_t
    lib.bte_pendulum_workspace_bytes.argtypes = [C.c_int32]
    lib.bte_pendulum_averages.restype = C.c_int
    lib.bte_pendulum_averages.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_double, C.c_int32, C.c_void_p,
                                          C.c_size_t, C.c_void_p, C.c_void_p]
    lib.bte_rs_workspace_bytes.restype = C.c_size_t
    lib.bte_rs_workspace_bytes.argtypes = [C.POINTER(bte_rs_grid)]
    lib.bte_rs_create.restype = C.c_int
    lib.bte_rs_create.argtypes = [C.POINTER(bte_rs_grid), C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p,
                                  C.POINTER(C.c_void_p)]
    for name in ("bte_rs_init_equilibrium", "bte_rs_destroy"):
        getattr(lib, name).restype = C.c_int
        getattr(lib, name).argtypes = [C.c_void_p]
    lib.bte_rs_step.restype = C.c_int
    lib.bte_rs_step.argtypes = [C.c_void_p, C.c_int64]
    lib.bte_rs_observables.restype = C.c_int
    lib.bte_rs_observables.argtypes = [C.c_void_p, C.POINTER(bte_obs)]
    lib.bte_rs_get_state.restype = C.c_int
    lib.bte_rs_get_state.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
    lib.bte_rs_evolve_static.restype = C.c_int
    lib.bte_rs_evolve_static.argtypes = [C.POINTER(bte_rs_grid), C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_void_p,
                                         C.c_void_p, C.c_void_p]
    lib.bte_set_option.restype = C.c_int
    lib.bte_set_option.argtypes = [C.c_void_p, C.c_char_p, C.c_int64]
    lib.bte_launch_count.restype = C.c_int
    lib.bte_launch_count.argtypes = [C.c_void_p, C.POINTER(C.c_int64)]
    lib.bte_last_error.restype = C.c_char_p
    lib.bte_last_error.argtypes = []
    _lib = lib
    return lib


def _check(rc: int):
    if rc != BTE_OK:
        raise BteError(rc, load_library().bte_last_error().decode())


def make_grid(n_harm: int, n_phiy: int, n_batch: int, dt: float, precision: int = 0) -> bte_grid:
    return bte_grid(int(n_harm), int(n_phiy), int(n_batch), int(precision), float(dt))


def make_params(ps: Sequence) -> C.Array:
    arr = (bte_params * len(ps))()
    for i, p in enumerate(ps):
        arr[i] = bte_params(p.E_dc, p.E_omega, p.omega, p.B, p.mu, p.alpha, p.phiy_min, p.phiy_max,
                            p.kappa_scale, int(p.n_steps_total), int(p.avg_start_step))
    return arr


def pendulum_averages(param_sets, n_phase: int = 64, h: float = 0.004, n_rk: int = 7500, device: str = "cuda:0"):
    """Zero-temperature pendulum model, eq. (44)-(46): param_sets = [(E_dc, E_omega, omega, B), ...]; returns a list
    of (v_mean, v_cos, v_sin).  Argument marshalling only: the integration runs in the library's kernel."""
    import torch
    lib = load_library()
    if not torch.cuda.is_available():
        raise RuntimeError("paper_1401_6047_b200 needs a CUDA device (no CPU fallback)")
    n = len(param_sets)
    arr = (C.c_double * (4 * n))(*[float(x) for ps in param_sets for x in ps])
    out = (C.c_double * (3 * n))()
    nbytes = int(lib.bte_pendulum_workspace_bytes(n))
    with torch.cuda.device(device):
        ws = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=device)
        stream = torch.cuda.current_stream().cuda_stream
        _check(lib.bte_pendulum_averages(arr, n, n_phase, h, n_rk, C.c_void_p(ws.data_ptr()), ws.numel(),
                                         C.c_void_p(stream), out))
    return [(out[3 * i], out[3 * i + 1], out[3 * i + 2]) for i in range(n)]


def workspace_bytes(n_harm: int, n_phiy: int, n_batch: int, dt: float) -> int:
    g = make_grid(n_harm, n_phiy, n_batch, dt)
    return int(load_library().bte_workspace_bytes(C.byref(g)))


def rs_evolve_static(n_phix: int, n_phiy: int, dt: float, params, f_in, step0: int, n_steps: int, f_out,
                     want_obs: bool = True, stream=None):
    """bte_rs_evolve_static (include/bte.h): n_steps real-space steps from f_in (CUDA float64 tensor [2, n_phix, n_phiy],
    contiguous; None = equilibrium) into f_out (same shape), in the library's static scratch array: no allocation, no
    workspace.  Returns an Obs when want_obs (synchronises), else None.  Argument marshalling only."""
    import torch
    lib = load_library()
    if not torch.cuda.is_available():
        raise RuntimeError("paper_1401_6047_b200 needs a CUDA device (B200, sm_100a); no CPU fallback")
    shape = (2, int(n_phix), int(n_phiy))
    for t in (f_in, f_out):
        if t is None and t is f_in:
            continue
        if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == shape):
            raise ValueError(f"need contiguous CUDA float64 tensors of shape {shape}")
    if f_in is not None and f_in.device != f_out.device:
        raise ValueError("f_in and f_out must live on the same device")
    g = bte_rs_grid(int(n_phix), int(n_phiy), float(dt))
    ps = make_params([params])
    o = bte_obs()
    with torch.cuda.device(f_out.device):
        st = stream if stream is not None else torch.cuda.current_stream(f_out.device)
        _check(lib.bte_rs_evolve_static(C.byref(g), C.cast(ps, C.c_void_p), C.c_void_p(f_in.data_ptr() if f_in is not None else None),
                                        C.c_int64(int(step0)), C.c_int64(int(n_steps)), C.c_void_p(f_out.data_ptr()),
                                        C.cast(C.byref(o), C.c_void_p) if want_obs else None,
                                        C.c_void_p(st.cuda_stream)))
    return Obs(*[getattr(o, f[0]) for f in bte_obs._fields_]) if want_obs else None


class RealSpaceSolver:
    """Thin wrapper of the bte_rs_* entry points (real-space-phi_x variant: one cyclic tridiagonal Crank-Nicolson solve
    per phi_y row; include/bte.h).  `params` is one object with the fields of bte_params."""

    def __init__(self, n_phix: int, n_phiy: int, dt: float, params, device: str = "cuda:0", stream=None):
        import torch
        lib = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1401_6047_b200 needs a CUDA device (B200, sm_100a); no CPU fallback")
        self._lib = lib
        self.grid = bte_rs_grid(int(n_phix), int(n_phiy), float(dt))
        self.shape = (int(n_phix), int(n_phiy))
        nbytes = int(lib.bte_rs_workspace_bytes(C.byref(self.grid)))
        if nbytes == 0:
            raise BteError(BTE_EINVAL, "invalid grid")
        self.device = torch.device(device)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self._params = make_params([params])
            h = C.c_void_p()
            _check(lib.bte_rs_create(C.byref(self.grid), self._params, C.c_void_p(self.workspace.data_ptr()),
                                     nbytes, C.c_void_p(self.stream.cuda_stream), C.byref(h)))
            self._h = h

    def _on_device(self):
        import torch
        return torch.cuda.device(self.device)      # the bte_rs_* calls launch on the current device

    def init_equilibrium(self):
        with self._on_device():
            _check(self._lib.bte_rs_init_equilibrium(self._h))

    def step(self, n_steps: int):
        with self._on_device():
            _check(self._lib.bte_rs_step(self._h, int(n_steps)))

    def observables(self) -> "Obs":
        o = bte_obs()
        with self._on_device():
            _check(self._lib.bte_rs_observables(self._h, C.byref(o)))
        return Obs(*[getattr(o, f[0]) for f in bte_obs._fields_])

    def get_state(self, grid_id: int):
        f = np.empty(self.shape)
        with self._on_device():
            _check(self._lib.bte_rs_get_state(self._h, grid_id, C.c_void_p(f.ctypes.data)))
        return f

    def destroy(self):
        if getattr(self, "_h", None):
            self._lib.bte_rs_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class Solver:
    """bte_create / bte_init_equilibrium / bte_step / bte_observables / bte_destroy with the same names.

    `grid` has n_harm, n_phiy, n_batch, dt; `params` is a sequence of objects with the fields of
    bte_params (e.g. workloads.Params).  The workspace tensor lives on `device` (default cuda:0).
    precision: 0 = fp64 (default), 1 = fp32 storage / fp64 arithmetic, 2 = fp32 throughout (bte_grid.precision).
    """

    def __init__(self, grid, params: Sequence, device: str = "cuda:0", stream=None, precision: int = 0):
        import torch  # device memory and streams only
        lib = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1401_6047_b200 needs a CUDA device (B200, sm_100a); no CPU fallback")
        if len(params) != grid.n_batch:
            raise ValueError("len(params) must equal grid.n_batch")
        self._lib = lib
        self.grid = make_grid(grid.n_harm, grid.n_phiy, grid.n_batch, grid.dt, precision)
        self.n_harm, self.n_phiy, self.n_batch, self.dt = grid.n_harm, grid.n_phiy, grid.n_batch, grid.dt
        self.shape = (grid.n_harm + 1, grid.n_phiy)
        nbytes = int(lib.bte_workspace_bytes(C.byref(self.grid)))
        if nbytes == 0:
            raise BteError(BTE_EINVAL, "invalid grid")
        self.device = torch.device(device)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._params = make_params(params)
        h = C.c_void_p()
        with torch.cuda.device(self.device):
            _check(lib.bte_create(C.byref(self.grid), self._params, C.c_void_p(self.workspace.data_ptr()),
                                  nbytes, C.c_void_p(self.stream.cuda_stream), C.byref(h)))
        self._h = h

    # -- the five calls of the boundary -------------------------------------------------------------
    def init_equilibrium(self):
        _check(self._lib.bte_init_equilibrium(self._h))

    def step(self, n_steps: int):
        _check(self._lib.bte_step(self._h, int(n_steps)))

    def observables(self) -> List[Obs]:
        out = (bte_obs * self.n_batch)()
        _check(self._lib.bte_observables(self._h, out))
        return [Obs(*[getattr(o, f[0]) for f in bte_obs._fields_]) for o in out]

    def destroy(self):
        if getattr(self, "_h", None):
            self._lib.bte_destroy(self._h)
            self._h = None

    close = destroy

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # -- state exchange / options ---------------------------------------------------------------------
    def get_state(self, system: int, grid_id: int, out_a=None, out_b=None):
        """Returns (a, b) numpy arrays of shape (n_harm+1, n_phiy); out_a/out_b may be preallocated
        (e.g. views of pinned torch tensors)."""
        a = np.empty(self.shape) if out_a is None else out_a
        b = np.empty(self.shape) if out_b is None else out_b
        _check(self._lib.bte_get_state(self._h, system, grid_id, C.c_void_p(a.ctypes.data),
                                       C.c_void_p(b.ctypes.data)))
        return a, b

    def set_state(self, system: int, grid_id: int, a, b):
        a = np.ascontiguousarray(a, dtype=np.float64)
        b = np.ascontiguousarray(b, dtype=np.float64)
        assert a.shape == self.shape and b.shape == self.shape
        _check(self._lib.bte_set_state(self._h, system, grid_id, C.c_void_p(a.ctypes.data),
                                       C.c_void_p(b.ctypes.data)))

    def reconstruct_pdf(self, system: int, grid_id: int, n_phix: int):
        """f(phi_x, phi_y) of eq. (8) on phi_x = -pi + 2 pi i / n_phix: a (n_phix, n_phiy) float64 tensor on the
        solver's device, written by the library's kernel on the solver's stream."""
        import torch
        f = torch.empty((n_phix, self.shape[1]), dtype=torch.float64, device=self.workspace.device)
        _check(self._lib.bte_reconstruct_pdf(self._h, system, grid_id, n_phix, C.c_void_p(f.data_ptr())))
        return f

    def get_state_batch(self, grid_id: int, out_a=None, out_b=None):
        """(a, b) of ALL systems: arrays of shape (n_batch, n_harm+1, n_phiy); one synchronisation."""
        shape = (self.n_batch,) + self.shape
        a = np.empty(shape) if out_a is None else out_a
        b = np.empty(shape) if out_b is None else out_b
        assert a.shape == shape and b.shape == shape and a.flags.c_contiguous and b.flags.c_contiguous
        _check(self._lib.bte_get_state_batch(self._h, grid_id, C.c_void_p(a.ctypes.data), C.c_void_p(b.ctypes.data)))
        return a, b

    def set_state_batch(self, grid_id: int, a, b):
        shape = (self.n_batch,) + self.shape
        a = np.ascontiguousarray(a, dtype=np.float64)
        b = np.ascontiguousarray(b, dtype=np.float64)
        assert a.shape == shape and b.shape == shape
        _check(self._lib.bte_set_state_batch(self._h, grid_id, C.c_void_p(a.ctypes.data), C.c_void_p(b.ctypes.data)))

    def set_option(self, key: str, value: int):
        _check(self._lib.bte_set_option(self._h, key.encode(), int(value)))

    def get_option(self, key: str) -> int:
        v = C.c_int64()
        _check(self._lib.bte_get_option(self._h, key.encode(), C.byref(v)))
        return int(v.value)

    def set_steady_policy(self, rel_tol: float, n_avg_periods: int, min_relax_periods: int = 0):
        _check(self._lib.bte_set_steady_policy(self._h, float(rel_tol), int(n_avg_periods), int(min_relax_periods)))

    def steady_info(self):
        """(steady_step, phase) per system."""
        nb = self.grid.n_batch
        st = (C.c_int64 * nb)()
        ph = (C.c_int32 * nb)()
        _check(self._lib.bte_steady_info(self._h, st, ph))
        return list(st), list(ph)

    def launch_count(self) -> int:
        n = C.c_int64()
        _check(self._lib.bte_launch_count(self._h, C.byref(n)))
        return int(n.value)

    def synchronize(self):
        self.stream.synchronize()
