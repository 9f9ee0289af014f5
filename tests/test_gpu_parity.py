"""GPU-vs-oracle parity through the C ABI (run on the B200 box: pytest -m gpu).

Element-by-element comparison of all four arrays (a, b on the whole and the fractional grid) and of the
observables, on the same generated inputs, at sizes that span several strips / row chunks with ragged
tails; then the BASELINE configs (full length where the oracle finishes in seconds, a step prefix
otherwise -- parity is asserted at the last common step).
"""
import numpy as np
import pytest

from paper_1401_6047_b200 import workloads as W

from parity_util import assert_obs_close, assert_state_close, oracle_run

pytestmark = pytest.mark.gpu

# name -> (variant, leap-frog steps fused per launch of the sweep kernel)
# (variant 3: shared-memory-ring kernel bte_sweep.cuh; variant 5: warp kernel bte_warpsweep.cuh, registers + tensor memory)
VARIANTS = {"split": (1, 0), "fused": (2, 0), "sweep1": (3, 1), "sweep2": (3, 2), "sweep3": (3, 3),
            "warp2": (5, 2), "warp3": (5, 3), "warp4": (5, 4), "resident": (4, 0), "auto": (0, 0)}
SWEEPS = ["sweep1", "sweep2", "sweep3", "warp2", "warp3", "warp4"]
ALL = ["split", "fused"] + SWEEPS + ["resident"]


def gpu_solver(w, variant="auto", graph_steps=None, tile_rows=None, ctas=None, res_ctas=None, threads=None):
    from paper_1401_6047_b200 import Solver
    s = Solver(w.grid, w.params)
    s.set_option("variant", VARIANTS[variant][0])
    s.set_option("sweep_steps", VARIANTS[variant][1])
    if graph_steps is not None:
        s.set_option("graph_steps", graph_steps)
    if tile_rows is not None:
        s.set_option("tile_rows", tile_rows)
    if ctas is not None:
        s.set_option("sweep_ctas", ctas)     # number of persistent CTAs of the sweep kernel
    if res_ctas is not None:
        s.set_option("resident_ctas", res_ctas)   # slabs of the resident kernel
    if threads is not None:
        s.set_option("sweep_threads", threads)    # 128 or 256 threads per CTA of the sweep kernel
    s.init_equilibrium()
    return s


def check(w, n_steps, variant, systems=None, graph_steps=None, tile_rows=None, chunks=None, ctas=None,
          res_ctas=None, threads=None):
    s = gpu_solver(w, variant, graph_steps, tile_rows, ctas, res_ctas, threads)
    if chunks:                      # several bte_step calls must equal one
        for c in chunks:
            s.step(c)
        assert sum(chunks) == n_steps
    else:
        s.step(n_steps)
    obs = s.observables()
    sims = oracle_run(w, n_steps, systems)
    worst = 0.0
    for i, sim in sims.items():
        what = f"{w.name}[{i}] {variant} steps={n_steps}"
        worst = max(worst, assert_state_close(s, sim, i, what=what))
        assert_obs_close(obs[i], sim.observables(), w.params[i], w.grid.dt, what=what)
    s.destroy()
    return worst


# -------------------------------------------------------------------------------------------------
# small / ragged shapes
# -------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", ALL)
def test_init_equilibrium_matches_oracle(variant):
    w = W.small_case(N=7, M1=45, n_steps=0)
    check(w, 0, variant)


@pytest.mark.parametrize("variant", ALL)
@pytest.mark.parametrize("N,M1", [(1, 3), (2, 5), (5, 126), (12, 127), (9, 128), (33, 253), (40, 801)])
def test_small_shapes(variant, N, M1):
    """M+1 around the strip width (126 columns) and its multiples, N around the chunk length."""
    w = W.small_case(N=N, M1=M1, dt=0.004, n_steps=23, B=1.5 if M1 > 3 else 0.2, avg_start=5)
    check(w, 23, variant)


@pytest.mark.parametrize("tile_rows", [2, 3, 7, 16])
def test_fused_row_chunking(tile_rows):
    """Row chunks with halo recompute, ragged last chunk, chunk boundaries next to rows 0/1."""
    w = W.small_case(N=21, M1=300, dt=0.004, n_steps=17, avg_start=3)
    check(w, 17, "fused", tile_rows=tile_rows)


@pytest.mark.parametrize("ctas", [1, 2, 3, 5, 7, 16, 40, 0])
@pytest.mark.parametrize("variant", SWEEPS)
def test_sweep_partition(ctas, variant):
    """Linearised static partition: CTA ranges that cut strips at arbitrary rows (segments that start at
    row 0, 1, 2, ..., one-row segments, ranges spanning several strips), every sweep depth S; 17 steps
    is not a multiple of S = 2, 3, so the trailing shorter launch is covered too."""
    w = W.small_case(N=21, M1=300, dt=0.004, n_steps=17, avg_start=3)
    check(w, 17, variant, ctas=ctas)


@pytest.mark.parametrize("ctas", [1, 3, 11, 0])
@pytest.mark.parametrize("variant", SWEEPS)
def test_sweep_wide_ctas(ctas, variant):
    """256-thread CTAs (strips of 254 / 250 / 246 columns): several strips with a ragged last one, segments cut
    at arbitrary rows, single and batched."""
    w = W.small_case(N=21, M1=600, dt=0.004, n_steps=10, avg_start=3)
    check(w, 10, variant, ctas=ctas, threads=256)
    wb = W.random_batch(n_batch=5, N=9, M1=300, dt=0.004, seed=78, periods=0.15)
    check(wb, wb.n_steps + 2, variant, ctas=ctas, threads=256)
    if variant == "sweep1":                       # 512-thread CTAs exist for the one-step pass only
        w = W.small_case(N=21, M1=1100, dt=0.004, n_steps=10, avg_start=3)
        check(w, 10, variant, ctas=ctas, threads=512)


@pytest.mark.parametrize("ctas", [1, 3, 9, 0])
@pytest.mark.parametrize("variant", SWEEPS)
def test_sweep_partition_batched(ctas, variant):
    """Ranges spanning several systems, with systems freezing at different steps (on-the-fly compaction)."""
    w = W.random_batch(n_batch=7, N=9, M1=140, dt=0.004, seed=77, periods=0.2)
    n = w.n_steps + 3
    s = gpu_solver(w, variant, ctas=ctas)
    s.step(n)
    obs = s.observables()
    sims = oracle_run(w, n)
    for i, sim in sims.items():
        assert obs[i].step == w.params[i].n_steps_total
        assert_state_close(s, sim, i, what=f"linbatch[{i}] ctas={ctas}")
        assert_obs_close(obs[i], sim.observables(), w.params[i], w.grid.dt, what=f"linbatch[{i}] ctas={ctas}")


@pytest.mark.parametrize("res_ctas", [1, 2, 3, 4, 5, 8, 16, 17, 40, 148, 0])
def test_resident_slabs(res_ctas):
    """Resident kernel: one CTA, clusters of 2..16 CTAs (edge columns through distributed shared memory),
    cooperative grids (edge columns through L2), ragged last slab; one launch per bte_step call."""
    w = W.small_case(N=21, M1=300 if res_ctas != 1 else 150, dt=0.004, n_steps=17, avg_start=3)
    s = gpu_solver(w, "resident", res_ctas=res_ctas)
    n0 = s.launch_count()
    s.step(9); s.step(1); s.step(7)
    assert s.launch_count() - n0 == 3
    obs = s.observables()
    sim = oracle_run(w, 17)[0]
    assert_state_close(s, sim, 0, what=f"resident ctas={res_ctas}")
    assert_obs_close(obs[0], sim.observables(), w.params[0], w.grid.dt, what=f"resident ctas={res_ctas}")
    s.destroy()


@pytest.mark.parametrize("halo", [1, 2, 3, 4])
@pytest.mark.parametrize("res_ctas", [17, 37, 75])
def test_resident_grid_halo_width(res_ctas, halo):
    """Cooperative-grid mode with 1..4 halo columns per side: the slabs exchange edge columns once per `halo`
    half-updates and update the halo columns redundantly in between (trapezoid in time); odd and even step counts,
    launches that end in the middle of an exchange group."""
    w = W.small_case(N=21, M1=300, dt=0.004, n_steps=23, avg_start=3)
    s = gpu_solver(w, "resident", res_ctas=res_ctas)
    s.set_option("resident_halo", halo)
    s.step(5); s.step(1); s.step(10); s.step(7)
    obs = s.observables()
    sim = oracle_run(w, 23)[0]
    assert_state_close(s, sim, 0, what=f"resident grid ctas={res_ctas} halo={halo}")
    assert_obs_close(obs[0], sim.observables(), w.params[0], w.grid.dt, what=f"resident grid ctas={res_ctas} halo={halo}")
    s.destroy()


@pytest.mark.parametrize("res_ctas", [1, 2, 4, 0])
def test_resident_batched_with_budgets(res_ctas):
    """A batch on the resident kernel: one CTA / one cluster per system, every system ends at its own step budget;
    several bte_step calls; more systems than SMs would also just queue (clusters are independent)."""
    w = W.random_batch(n_batch=9, N=9, M1=140, dt=0.004, seed=31, periods=0.2)
    n = w.n_steps + 3
    s = gpu_solver(w, "resident", res_ctas=res_ctas)
    n0 = s.launch_count()
    s.step(n // 3); s.step(n - n // 3)
    assert s.launch_count() - n0 == 2
    obs = s.observables()
    sims = oracle_run(w, n)
    for i, sim in sims.items():
        assert obs[i].step == w.params[i].n_steps_total
        assert_state_close(s, sim, i, what=f"resident batch[{i}] ctas={res_ctas}")
        assert_obs_close(obs[i], sim.observables(), w.params[i], w.grid.dt, what=f"resident batch[{i}] ctas={res_ctas}")
    s.destroy()


def test_resident_batch_of_many_small_systems_auto():
    """200 systems of 5 x 33 points (more clusters than SMs), automatic variant choice = resident; a sample is
    compared with the oracle."""
    w = W.random_batch(n_batch=200, N=4, M1=33, dt=0.004, seed=5, periods=0.0, n_steps=60)
    s = gpu_solver(w, "auto")
    n0 = s.launch_count()
    s.step(60)
    assert s.launch_count() - n0 == 1
    obs = s.observables()
    for i, sim in oracle_run(w, 60, systems=[0, 57, 131, 199]).items():
        assert_state_close(s, sim, i, what=f"many small[{i}]")
        assert_obs_close(obs[i], sim.observables(), w.params[i], w.grid.dt, what=f"many small[{i}]")
    s.destroy()


@pytest.mark.parametrize("N,M1", [(1, 3), (1, 4000), (300, 7), (600, 50), (3, 129), (40, 16), (97, 1025)])
def test_odd_shapes_through_the_automatic_path(N, M1):
    """Tall / narrow / tiny lattices through the automatic variant choice (resident CTA, cluster, grid, or sweep),
    two bte_step calls of different lengths (>= 4 steps: resident where it fits; < 4: sweep)."""
    w = W.small_case(N=N, M1=M1, dt=0.004, n_steps=14, avg_start=2)
    check(w, 14, "auto", chunks=[11, 3])


def test_resident_interleaves_with_sweep_and_budget():
    """The resident kernel and the streaming kernels share the state: alternate them; a step budget freezes
    the system exactly at n_steps_total."""
    w = W.small_case(N=12, M1=190, dt=0.004, n_steps=40, avg_start=5)
    w.params[0].n_steps_total = 33
    s = gpu_solver(w, "auto")
    s.step(10)                          # resident (>= 4 steps)
    s.set_option("variant", 3); s.step(3)
    s.set_option("variant", 4); s.step(2)
    s.set_option("variant", 1); s.step(5)
    s.set_option("variant", 0); s.step(50)      # runs into the budget
    obs = s.observables()
    assert obs[0].step == 33
    sim = oracle_run(w, 70)[0]
    assert_state_close(s, sim, 0, what="resident/sweep interleaved")
    assert_obs_close(obs[0], sim.observables(), w.params[0], w.grid.dt, what="resident/sweep interleaved")
    s.destroy()


@pytest.mark.parametrize("variant", ALL)
def test_graph_replay_equals_plain_launches(variant):
    w = W.small_case(N=10, M1=140, n_steps=50, avg_start=7)
    check(w, 50, variant, graph_steps=8)             # 6 graph replays + 2 plain steps
    check(w, 50, variant, graph_steps=0)
    check(w, 50, variant, chunks=[1, 2, 30, 17])


def test_fused_equals_split_bitwise_state():
    """The variants that form mu = n * (beta dt/2) evaluate the same per-point expression in the same operation order:
    their states must be bit-identical (this stands in for a race detector: any ordering bug changes bits).  The warp
    kernel forms mu = fma(n, B phi dt/2, n E dt/2) (no per-column table of the half-step times): it differs from the
    others in the last bits of mu only, so it must agree with them to a few ulps, and its three depths (same expression,
    different decomposition into strips, stages and segments) with each other bit for bit (36 steps: a multiple of every
    depth, so that no single-step launch of the ring kernel, which forms mu the other way, is mixed in)."""
    w = W.small_case(N=14, M1=260, n_steps=36)
    a = gpu_solver(w, "split"); a.step(36)
    ref = [a.get_state(0, g) for g in (0, 1)]
    scale = max(np.abs(x).max() for pair in ref for x in pair)
    warp = {}
    for other in ["fused", "resident"] + SWEEPS:
        b = gpu_solver(w, other); b.step(36)
        for g in (0, 1):
            ya, yb = b.get_state(0, g)
            if other.startswith("warp"):
                assert max(np.abs(ya - ref[g][0]).max(), np.abs(yb - ref[g][1]).max()) <= 1e-14 * scale, other
                warp.setdefault(g, []).append((ya, yb))
            else:
                assert np.array_equal(ref[g][0], ya) and np.array_equal(ref[g][1], yb), other
    for g in (0, 1):
        assert len(warp[g]) == 3                     # the three depths of the warp kernel: bit for bit
        for other in warp[g][1:]:
            assert np.array_equal(warp[g][0][0], other[0]) and np.array_equal(warp[g][0][1], other[1])


@pytest.mark.parametrize("variant", ALL)
def test_batched_with_step_budgets(variant):
    """Config-3-shaped batch: per-system parameters, phi_y ranges and step budgets (systems freeze)."""
    w = W.random_batch(n_batch=6, N=10, M1=150, dt=0.004, seed=123, periods=0.25)
    n = w.n_steps + 5                   # run past the longest budget
    s = gpu_solver(w, variant)
    s.step(n)
    obs = s.observables()
    sims = oracle_run(w, n)
    for i, sim in sims.items():
        assert obs[i].step == w.params[i].n_steps_total
        assert_state_close(s, sim, i, what=f"batch[{i}] {variant}")
        assert_obs_close(obs[i], sim.observables(), w.params[i], w.grid.dt, what=f"batch[{i}] {variant}")


def test_alpha_and_kappa_scale():
    w = W.small_case(N=8, M1=90, alpha=0.9496, kappa_scale=0.9496, n_steps=20)
    for v in ALL:
        check(w, 20, v)


def test_set_state_roundtrip_and_step():
    rng = np.random.default_rng(5)
    w = W.small_case(N=6, M1=70, n_steps=9)
    s = gpu_solver(w, "auto")
    shape = (7, 70)
    ha, hb, fa, fb = (rng.standard_normal(shape) for _ in range(4))
    hb[0] = 0; fb[0] = 0
    s.set_state(0, 0, ha, hb); s.set_state(0, 1, fa, fb)
    ga, gb = s.get_state(0, 0)
    assert np.array_equal(ga, ha) and np.array_equal(gb, hb)
    from oracle import OracleSim
    sim = OracleSim(6, 70, w.grid.dt, w.params[0])
    sim.set_state(0, ha, hb); sim.set_state(1, fa, fb)
    s.step(9); sim.step(9)
    assert_state_close(s, sim, 0, what="set_state")


def test_batch_state_exchange_equals_per_system_calls():
    """bte_get_state_batch / bte_set_state_batch: one synchronisation for the whole batch; systems whose live
    ping-pong buffers differ (frozen systems stop toggling) are handled on the device."""
    w = W.random_batch(n_batch=7, N=9, M1=140, dt=0.004, seed=77, periods=0.2)
    s = gpu_solver(w, "sweep3")
    s.step(w.n_steps // 2 + 1)            # some systems frozen already, odd and even launch counts mixed
    per = [[s.get_state(i, g) for g in (0, 1)] for i in range(7)]
    for g in (0, 1):
        a, b = s.get_state_batch(g)
        for i in range(7):
            assert np.array_equal(a[i], per[i][g][0]) and np.array_equal(b[i], per[i][g][1])
    # round trip through set_state_batch into a fresh solver, then both continue identically
    t = gpu_solver(w, "sweep3")
    t.step(w.n_steps // 2 + 1)
    rng = np.random.default_rng(3)
    new = [[rng.standard_normal((7, 10, 140)) for _ in range(2)] for _ in range(2)]
    for g in (0, 1):
        new[g][1][:, 0, :] = 0.0
        s.set_state_batch(g, new[g][0], new[g][1])
        for i in range(7):
            t.set_state(i, g, new[g][0][i], new[g][1][i])
    s.step(5); t.step(5)
    for g in (0, 1):
        a, b = s.get_state_batch(g)
        for i in range(7):
            ra, rb = t.get_state(i, g)
            assert np.array_equal(a[i], ra) and np.array_equal(b[i], rb)
    os_, ot = s.observables(), t.observables()
    assert [o.step for o in os_] == [o.step for o in ot]
    assert s.get_option("device") == 0 and s.get_option("effective_variant") == 3 and s.get_option("effective_sweep_steps") == 3


# -------------------------------------------------------------------------------------------------
# error behaviour of the boundary
# -------------------------------------------------------------------------------------------------
def test_create_rejects_unstable_and_invalid():
    from paper_1401_6047_b200 import BteError, Solver
    w = W.small_case(N=4, M1=41, dt=0.5, B=4.0, phiy_max=4.0)       # B dt/dphi = 10
    with pytest.raises(BteError) as e:
        Solver(w.grid, w.params)
    assert e.value.code == -2
    w = W.small_case(N=4, M1=41, mu=-1.0, phiy_max=4.0)
    with pytest.raises(BteError) as e:
        Solver(w.grid, w.params)
    assert e.value.code == -1


# -------------------------------------------------------------------------------------------------
# BASELINE configs
# -------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", ALL)
def test_config0_full(variant):
    from scipy import special
    w = W.config0()
    s = gpu_solver(w, variant)
    s.step(w.n_steps)
    o = s.observables()[0]
    want = special.ive(1, 1.0) / special.ive(0, 1.0) * 0.5
    assert abs(o.v_dr - want) / want < 5e-9 and abs(o.norm - 1) < 1e-12
    sim = oracle_run(w, w.n_steps)[0]
    assert_state_close(s, sim, 0, what="config0")
    assert_obs_close(o, sim.observables(), w.params[0], w.grid.dt, what="config0")


def test_config1_prefix():
    """Prefix of 3000 steps: full state parity (full length: tests/test_gpu_full_size.py)."""
    w = W.config1()
    check(w, 3000, "auto")


def test_config2_prefix():
    w = W.config2()
    check(w, 300, "auto")


def test_config3_subset_prefix():
    """All 512 systems advance together on the GPU; 8 of them (0, 73, 146, ...) are checked."""
    w = W.config3()
    check(w, 200, "auto", systems=list(range(0, 512, 73)))


def test_paper_table1_prefix():
    """The paper's own Table 1 run (mu = 116, sharp f0; 121 x 4000 lattice), 60 steps, fp64, automatic variant."""
    w = W.get(5)
    check(w, 60, "auto")


def test_config4_prefix():
    """Bandwidth-stress grid in the launch configuration bench.py times; 4 steps, full state compare."""
    w = W.config4()
    check(w, 4, "auto")
