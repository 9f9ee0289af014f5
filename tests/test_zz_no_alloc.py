"""bte_rs_evolve_static (include/bte.h): the real-space step in the library's static scratch array -- no allocation, no
workspace -- against the existing path (RealSpaceSolver = bte_rs_create / bte_rs_step with a caller-owned workspace),
on calls in a row that share the array.  Collected last on purpose (file name).  pytest -m gpu."""
import numpy as np
import pytest

from paper_1401_6047_b200 import workloads as W

pytestmark = pytest.mark.gpu

DT = 0.004
TOL = 1e-12          # relative to max |f|: the bound of tests/test_gpu_realspace.py


def existing_path(K, M1, p, n_steps):
    """[2, K, M1] state and observables after n_steps of the workspace-owning solver"""
    from paper_1401_6047_b200 import RealSpaceSolver
    s = RealSpaceSolver(K, M1, DT, p)
    s.init_equilibrium()
    s.step(n_steps)
    f = np.stack([s.get_state(0), s.get_state(1)])
    o = s.observables()
    s.destroy()
    return f, o


def close(f_static, f_ref):
    scale = np.abs(f_ref).max()
    assert np.isfinite(f_static).all()
    assert np.abs(f_static - f_ref).max() <= TOL * scale, np.abs(f_static - f_ref).max() / scale


def params(avg_start=3, **kw):
    return W.small_case(N=2, M1=41, dt=DT, avg_start=avg_start, **kw).params[0]


@pytest.mark.parametrize("K,M1", [(64, 130), (37, 41)])          # parallel cyclic reduction / Thomas sweeps
def test_static_scratch_two_calls_in_a_row_match_the_workspace_path(K, M1):
    import torch
    from paper_1401_6047_b200 import rs_evolve_static
    p = params()
    n1, n2 = 9, 7
    ref1, o1 = existing_path(K, M1, p, n1)
    ref2, o2 = existing_path(K, M1, p, n1 + n2)
    f1 = torch.full((2, K, M1), float("nan"), dtype=torch.float64, device="cuda:0")
    a1 = rs_evolve_static(K, M1, DT, p, None, 0, n1, f1)                    # call 1: from equilibrium
    close(f1.cpu().numpy(), ref1)
    assert a1.step == n1 and abs(a1.norm - o1.norm) <= 1e-12 and abs(a1.v_dr - o1.v_dr) <= 1e-12
    assert abs(a1.sum_vcos_dt - o1.sum_vcos_dt) <= 1e-12 and abs(a1.window - o1.window) <= 1e-12
    f2 = torch.empty_like(f1)
    a2 = rs_evolve_static(K, M1, DT, p, f1, n1, n2, f2)                     # call 2: continues from call 1's output
    close(f2.cpu().numpy(), ref2)
    assert a2.step == n1 + n2 and abs(a2.norm - o2.norm) <= 1e-12 and abs(a2.v_dr - o2.v_dr) <= 1e-12
    # running sums restart with every call: call 2 holds the difference of the long run's sums
    assert abs(a2.sum_vcos_dt - (o2.sum_vcos_dt - o1.sum_vcos_dt)) <= 1e-12
    assert abs(a2.sum_vsin_dt - (o2.sum_vsin_dt - o1.sum_vsin_dt)) <= 1e-12
    assert abs(a2.window - (o2.window - o1.window)) <= 1e-12
    rs_evolve_static(K, M1, DT, p, f1, n1, n2, f1, want_obs=False)          # in place, no host transfer
    torch.cuda.synchronize()
    assert torch.equal(f1, f2)


def test_static_scratch_keeps_nothing_between_shapes():
    """the array keeps the last call's contents: a different shape and different parameters right after must not see them"""
    import torch
    from paper_1401_6047_b200 import rs_evolve_static
    pa, pb = params(), params(avg_start=0, B=0.0, E_dc=1.3)
    out_a = torch.empty((2, 128, 257), dtype=torch.float64, device="cuda:0")
    out_b = torch.empty((2, 16, 5), dtype=torch.float64, device="cuda:0")
    rs_evolve_static(128, 257, DT, pa, None, 0, 12, out_a)
    b = rs_evolve_static(16, 5, DT, pb, None, 0, 30, out_b)
    ref_b, ob = existing_path(16, 5, pb, 30)
    close(out_b.cpu().numpy(), ref_b)
    assert abs(b.v_dr - ob.v_dr) <= 1e-12 and abs(b.sum_v_dt - ob.sum_v_dt) <= 1e-12
    a = rs_evolve_static(128, 257, DT, pa, None, 0, 12, out_a)
    ref_a, oa = existing_path(128, 257, pa, 12)
    close(out_a.cpu().numpy(), ref_a)
    assert abs(a.v_dr - oa.v_dr) <= 1e-12 and abs(a.norm - oa.norm) <= 1e-12


def test_static_scratch_refuses_what_does_not_fit():
    import torch
    from paper_1401_6047_b200 import BteError, rs_evolve_static
    p = params()
    big = torch.empty((2, 256, 520), dtype=torch.float64, device="cuda:0")      # 256 x 520 = 133120 > 131072 points
    with pytest.raises(BteError) as e:
        rs_evolve_static(256, 520, DT, p, None, 0, 1, big)
    assert e.value.code == -3 and "131072" in str(e.value) and "bte_rs_create" in str(e.value)
    ok = torch.empty((2, 256, 512), dtype=torch.float64, device="cuda:0")       # exactly the limit
    o = rs_evolve_static(256, 512, DT, p, None, 0, 2, ok)
    ref, oref = existing_path(256, 512, p, 2)
    close(ok.cpu().numpy(), ref)
    assert o.step == 2 and abs(o.norm - oref.norm) <= 1e-12
    with pytest.raises(BteError):
        rs_evolve_static(16, 5, DT, p, None, 3, 1, torch.empty((2, 16, 5), dtype=torch.float64, device="cuda:0"))
