"""The C-ABI boundary without a GPU: libbte_b200.so loads, exports every symbol include/bte.h declares, and
its argument validation (which runs before any CUDA call) behaves as the header says.  No compute calls."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "bte.h")


@pytest.fixture(scope="module")
def lib():
    from paper_1401_6047_b200 import binding, build
    return binding.load_library(build.build())


def declared_functions():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)                 # drop comments
    return sorted(set(re.findall(r"\b(bte_[a-z_]+)\s*\(", text)))


def test_header_declares_the_five_north_star_calls():
    names = declared_functions()
    for n in ("bte_create", "bte_init_equilibrium", "bte_step", "bte_observables", "bte_destroy"):
        assert n in names


def test_every_declared_symbol_is_exported(lib):
    from paper_1401_6047_b200 import binding
    names = declared_functions()
    assert len(names) >= 11
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/bte.h but not exported by libbte_b200.so"
    assert sorted(binding.EXPORTS) == names, "binding.EXPORTS must list exactly the header's functions"


def test_exported_symbols_are_exactly_the_header(lib):
    """-fvisibility=hidden + BTE_API: the dynamic symbol table of the .so holds the header's functions and nothing else."""
    import subprocess
    from paper_1401_6047_b200 import binding
    out = subprocess.run(["nm", "-D", "--defined-only", binding.LIB_PATH], capture_output=True, text=True, check=True).stdout
    exported = sorted(ln.split()[-1] for ln in out.splitlines() if len(ln.split()) >= 3 and ln.split()[-2] in ("T", "W", "B", "D"))
    exported = [n for n in exported if not n.startswith("_")]          # toolchain symbols (_init, _fini, ...)
    assert exported == declared_functions(), set(exported) ^ set(declared_functions())


def test_struct_layouts_match_header():
    from paper_1401_6047_b200 import binding
    assert C.sizeof(binding.bte_grid) == 24            # 4 x int32 + double
    assert C.sizeof(binding.bte_params) == 9 * 8 + 2 * 8
    assert C.sizeof(binding.bte_obs) == 8 + 8 * 8


def test_workspace_bytes_is_a_pure_function(lib):
    from paper_1401_6047_b200 import binding
    lib.bte_workspace_bytes.restype = C.c_size_t
    small = lib.bte_workspace_bytes(C.byref(binding.make_grid(20, 201, 1, 0.005)))
    big = lib.bte_workspace_bytes(C.byref(binding.make_grid(512, 32001, 1, 0.001)))
    assert 0 < small < big
    # state: 2 buffers x 2 grids x (N + 1 + ghost rows) x pitch x 16 B dominates
    assert big >= 2 * 2 * 513 * 32001 * 16 and big < 1.1 * 2 * 2 * 517 * 32008 * 16
    assert lib.bte_workspace_bytes(C.byref(binding.make_grid(0, 201, 1, 0.005))) == 0      # N < 1
    assert lib.bte_workspace_bytes(C.byref(binding.make_grid(20, 2, 1, 0.005))) == 0       # M+1 < 3
    assert lib.bte_workspace_bytes(C.byref(binding.make_grid(20, 201, 0, 0.005))) == 0     # n_batch < 1
    assert lib.bte_workspace_bytes(C.byref(binding.make_grid(20, 201, 1, 0.0))) == 0       # dt <= 0
    assert lib.bte_workspace_bytes(None) == 0
    # fp32 storage (bte_grid.precision 1, 2): half the bytes per lattice point; precision outside 0..2 is invalid
    half = lib.bte_workspace_bytes(C.byref(binding.make_grid(512, 32001, 1, 0.001, precision=2)))
    assert 0.49 * big < half < 0.52 * big
    assert lib.bte_workspace_bytes(C.byref(binding.make_grid(20, 201, 1, 0.005, precision=3))) == 0


def _create(lib, grid, params, ws=0x10000, nbytes=1 << 40):
    out = C.c_void_p()
    rc = lib.bte_create(C.byref(grid), params, C.c_void_p(ws), C.c_size_t(nbytes), None, C.byref(out))
    return rc, out


def test_create_validates_before_touching_cuda(lib):
    """Every rejection below happens in the argument checks of bte_create, i.e. before the first CUDA call,
    so it can be exercised on a box without a GPU (the fake workspace pointer is never dereferenced)."""
    from paper_1401_6047_b200 import binding, workloads as W
    lib.bte_last_error.restype = C.c_char_p
    w = W.small_case(N=4, M1=41, phiy_max=4.0)
    g, ps = binding.make_grid(4, 41, 1, w.grid.dt), binding.make_params(w.params)
    rc, out = _create(lib, g, ps, nbytes=16)
    assert rc == -3 and not out.value and b"workspace" in lib.bte_last_error()             # BTE_ENOMEM
    rc, out = _create(lib, g, ps, ws=0x10008)
    assert rc == -3 and not out.value                                                       # misaligned
    rc, out = _create(lib, g, None)
    assert rc == -1 and not out.value                                                       # NULL params
    bad = W.small_case(N=4, M1=41, mu=-1.0, phiy_max=4.0)
    rc, out = _create(lib, g, binding.make_params(bad.params))
    assert rc == -1 and not out.value                                                       # mu <= 0
    bad = W.small_case(N=4, M1=41, dt=0.5, B=4.0, phiy_max=4.0)                             # |B| dt/dphi = 10
    rc, out = _create(lib, binding.make_grid(4, 41, 1, 0.5), binding.make_params(bad.params))
    assert rc == -2 and not out.value and b"unstable" in lib.bte_last_error()               # BTE_EUNSTABLE
    assert lib.bte_step(None, 1) == -1 and lib.bte_destroy(None) == 0
    v = C.c_int64()
    assert lib.bte_get_option(None, b"variant", C.byref(v)) == -1
    assert lib.bte_get_state_batch(None, 0, None, None) == -1 and lib.bte_set_state_batch(None, 0, None, None) == -1


def test_product_path_fails_loudly_without_a_gpu():
    """No CPU fallback: on a box without CUDA the public API raises instead of computing."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    from paper_1401_6047_b200 import Solver, workloads as W
    w = W.small_case()
    with pytest.raises(Exception):
        Solver(w.grid, w.params)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1401_6047_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "bte_oracle" not in text, f


def test_rs_evolve_static_validates_before_any_cuda_call(lib):
    """bte_rs_evolve_static: NULL arguments, bad step arguments and grids beyond the static scratch limit (131072 points)
    are refused by host-side checks; the dummy device pointers below are never touched."""
    from paper_1401_6047_b200 import binding, workloads as W
    p = binding.make_params([W.small_case(N=2, M1=41, dt=0.004).params[0]])
    dummy = C.c_void_p(0x10000)

    def call(K, M1, f_in, step0, n_steps, f_out, params=p):
        g = binding.bte_rs_grid(K, M1, 0.004)
        return lib.bte_rs_evolve_static(C.byref(g), C.cast(params, C.c_void_p) if params is not None else None, f_in,
                                        C.c_int64(step0), C.c_int64(n_steps), f_out, None, None)

    assert call(64, 130, None, 0, 1, None) == -1                                   # no output
    assert call(64, 130, None, 0, 1, dummy, params=None) == -1                     # no parameters
    assert call(2, 130, None, 0, 1, dummy) == -1                                   # too few phi_x points
    assert call(64, 130, None, 0, -1, dummy) == -1 and call(64, 130, dummy, -1, 1, dummy) == -1
    assert call(64, 130, None, 5, 1, dummy) == -1                                  # equilibrium start needs step0 = 0
    assert call(256, 520, None, 0, 1, dummy) == -3                                 # 256 x 520 > 131072 points
    msg = lib.bte_last_error().decode()
    assert "131072" in msg and "bte_rs_create" in msg
    assert call(4096, 40, None, 0, 1, dummy) == -3                                 # 4096 x 40 = 163840 points
