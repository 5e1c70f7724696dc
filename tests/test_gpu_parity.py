"""Parity of the CUDA path (through the C-ABI, via the ctypes binding) with the CPU oracle, element by element
on the same seeded inputs.  Tolerances:
  * a, jerk: per-particle vector-norm relative error <= 1e-12 (north_star) against the oracle's compensated sums;
  * predictor, corrector, time steps given identical inputs: bit-exact (both round every operation separately);
  * active lists, block levels, times: bit-exact;
  * energy: |dK/K|, |dU/U| <= 1e-13.
"""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from paper_1702_00440_b200 import workloads as W


@pytest.fixture(scope="module")
def gd():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (the product has no CPU fallback)")
    from paper_1702_00440_b200 import binding
    binding.load()
    return binding


def relnorm(u, ref):
    u, ref = np.asarray(u, dtype=np.float64), np.asarray(ref, dtype=np.float64)
    den = np.linalg.norm(ref, axis=-1)
    den = np.where(den == 0, 1.0, den)
    return np.linalg.norm(u - ref, axis=-1) / den


def cpu(t):
    return t.detach().cpu().numpy()


TOL = 1e-12


# ------------------------------------------------------------------------------------------- force / jerk
@pytest.mark.parametrize("n", [1, 2, 3, 31, 257, 1000])
@pytest.mark.parametrize("eps", [0.0, 1e-4])
def test_force_small_and_ragged(gd, n, eps):
    # tiny and ragged sizes: one tile with a tail, padding records, eps = 0 self-pair masking
    w = W.random_cluster(n, seed=20 + n, eps=eps)
    a, j = gd.force_jerk_host(w.m, w.x, w.v, eps)
    a_ref, j_ref = oracle.pairsum(w.m, w.x, w.v, eps)
    assert relnorm(a, a_ref).max() <= TOL and relnorm(j, j_ref).max() <= TOL
    assert np.isfinite(a).all() and np.isfinite(j).all()


def test_force_hand_example(gd):
    # the paper-formula hand example of tests/golden/pairsum_hand_example.txt
    from conftest import read_golden_table
    m = np.array([0.0, 1.0])
    x = np.array([[0, 0, 0], [3, 4, 0.0]])
    v = np.array([[0, 0, 0], [1, 2, 0.0]])
    for eps2, *ref in read_golden_table("pairsum_hand_example.txt"):
        a, j = gd.force_jerk_host(m, x, v, math.sqrt(eps2))
        assert np.allclose(a[0], ref[:3], rtol=1e-15, atol=1e-18) and np.allclose(j[0], ref[3:], rtol=2e-15, atol=1e-18)
        assert not a[1].any() and not j[1].any()


@pytest.mark.parametrize("cfg,n", [(1, 1024), (2, 16384), (4, 5000), (5, 3000)])
def test_force_all_active_configs(gd, cfg, n):
    # all-active evaluation on the config inputs (C4: Kroupa masses; C5: central point mass, N = n + 1 ragged)
    w = W.config(cfg, n=n)
    a, j = gd.force_jerk_host(w.m, w.x, w.v, w.eps)
    a_ref, j_ref = oracle.pairsum(w.m, w.x, w.v, w.eps)
    ea, ej = relnorm(a, a_ref), relnorm(j, j_ref)
    assert ea.max() <= TOL and ej.max() <= TOL, (ea.max(), ej.max())


KERNEL_OPTIONS = {   # force one of the four force kernels regardless of n_act
    "ipar": {"slice_max_nact": 0, "jsplit_max_nact": 0, "ipar_small_max_nact": 0},
    "ipar_small": {"slice_max_nact": 0, "jsplit_max_nact": 0, "ipar_small_max_nact": 1 << 30},
    "jsplit": {"slice_max_nact": 0, "jsplit_max_nact": 1 << 30},   # capped by the library at 32 sinks x the clusters of its grid
    "slice": {"slice_max_nact": 1 << 30},
    "slice3": {"slice_max_nact": 1 << 30, "slice_passes": 3},     # three slices per CTA, as for systems beyond shared memory
}


@pytest.mark.parametrize("kernel", ["ipar", "ipar_small", "jsplit", "slice", "slice3"])
@pytest.mark.parametrize("n_act", [1, 5, 16, 96, 97, 100, 256, 1000, 4096])
def test_force_active_subsets_all_kernels(gd, kernel, n_act):
    # C3-style index sets on a smaller sphere, forced through each kernel; all must agree with the oracle
    import torch
    if kernel == "jsplit" and n_act > 1000:
        pytest.skip("beyond the j-split kernel's grid (32 sinks per cluster)")
    if kernel == "slice3" and n_act > 2048:
        pytest.skip("beyond the partial-sum scratch of three slices per CTA at this N")
    w = W.config(3, n=8192 + 77)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    for key, val in KERNEL_OPTIONS[kernel].items():
        h.set_option(key, val)
    h.predict(0.0)
    idx = W.active_indices(w.n, n_act)
    a, j = h.force_jerk(torch.from_numpy(idx).cuda())
    assert h.last_force_kernel == kernel.rstrip("3")
    if kernel.startswith("slice"):
        assert h.last_force_geometry[3] == (3 if kernel == "slice3" else 1)
    a_ref, j_ref = oracle.pairsum(w.m, w.x, w.v, w.eps, idx=idx)
    assert relnorm(cpu(a), a_ref).max() <= TOL and relnorm(cpu(j), j_ref).max() <= TOL
    # run-to-run identical (fixed combination order)
    a2, j2 = h.force_jerk(torch.from_numpy(idx).cuda())
    assert torch.equal(a, a2) and torch.equal(j, j2)
    h.close()


def test_force_unsorted_and_repeated_indices(gd):
    import torch
    w = W.config(1)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    h.predict(0.0)
    idx = np.array([1023, 0, 5, 5, 512, 0], dtype=np.int32)
    a, j = h.force_jerk(torch.from_numpy(idx).cuda())
    a_ref, j_ref = oracle.pairsum(w.m, w.x, w.v, w.eps, idx=idx)
    assert relnorm(cpu(a), a_ref).max() <= TOL and relnorm(cpu(j), j_ref).max() <= TOL
    h.close()


# ------------------------------------------------------------------------------ init, predictor, corrector
@pytest.mark.parametrize("seed", [1, 2, 3])
def test_division_by_constants_is_the_correctly_rounded_quotient(gd, seed):
    # gd_div_const (x / 6, x / 24, x / 120 as a multiply and two FMAs) against the division routine, bit for bit,
    # on 2^26 random operands per constant; the oracle divides (oracle/hermite_oracle.c), so must the device
    assert gd.selftest_div_const(1 << 26, seed) == 0


def test_init_matches_oracle(gd):
    w = W.config(1)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    o = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta)
    s = {k: cpu(v) for k, v in h.state().items()}
    assert np.array_equal(s["x"], w.x) and np.array_equal(s["v"], w.v)
    assert relnorm(s["a"], o.a).max() <= TOL and relnorm(s["j"], o.j).max() <= TOL
    assert np.array_equal(s["dt"], o.dt) and not s["t"].any()
    h.close()


def test_predictor_bit_exact_given_same_state(gd):
    # advance the GPU a few steps, then predict both from the GPU's own state: identical inputs -> identical bits
    w = W.config(1, n=700)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    h.step(25)
    s = {k: cpu(v) for k, v in h.state().items()}
    t = h.t + 2.0 ** -9
    h.predict(t)
    xp, vp = (cpu(u) for u in h.predicted())
    xp_ref, vp_ref = oracle.predict(t, s["x"], s["v"], s["a"], s["j"], s["t"])
    assert np.array_equal(xp, xp_ref) and np.array_equal(vp, vp_ref)
    h.close()


def test_corrector_bit_exact_given_same_inputs(gd):
    import torch
    w = W.config(4, n=900)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    h.step(10)
    before = {k: cpu(v) for k, v in h.state().items()}
    t_next, n_act = h.next_block()
    act = cpu(h.active())
    h.predict(t_next)
    xp, vp = (cpu(u) for u in h.predicted())
    a1 = torch.empty((n_act, 3), dtype=torch.float64, device="cuda")
    j1 = torch.empty_like(a1)
    h.force_jerk(None, a1, j1)            # explicit outputs: a copy of what the corrector will consume
    h.force_jerk(None)
    h.correct_and_timestep()
    after = {k: cpu(v) for k, v in h.state().items()}
    ref = oracle.correct(act, t_next, w.eta, before["x"], before["v"], before["a"], before["j"], before["t"],
                         before["dt"], xp, vp, cpu(a1), cpu(j1))
    for k, r in zip(("x", "v", "a", "j", "t", "dt"), ref):
        assert np.array_equal(after[k], r), k
    h.close()


# ----------------------------------------------------------------------------------------- active sets
@pytest.mark.parametrize("n,steps", [(3000, 30), (10000, 12), (40000, 8), (70000, 6)])
def test_next_block_against_oracle_on_synthetic_times(gd, n, steps):
    # drive the compaction with many different patterns by stepping a system; every list must be the ascending
    # exact-equality set of the oracle's definition applied to the GPU's own t, dt.  The sizes cover the three
    # single-CTA variants (chunks of 4, 16, 64 per thread) and the two-kernel path for large systems.
    w = W.config(1, n=n)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    for _ in range(steps):
        s = h.state(("t", "dt"))
        t_ref, act_ref = oracle.next_block(cpu(s["t"]), cpu(s["dt"]))
        t_next, n_act = h.next_block()
        assert t_next == t_ref and n_act == len(act_ref)
        assert np.array_equal(cpu(h.active()), act_ref)
        h.predict(t_next)
        h.force_jerk(None)
        h.correct_and_timestep()
    h.close()


@pytest.mark.parametrize("cfg,n", [(1, 1024), (2, 16384), (3, 4096), (4, 6000), (5, 2047)])
def test_first_100_block_steps_bit_exact_schedule(gd, cfg, n):
    # north_star: active-set and block-time-step indices bit-exact over the first 100 block steps
    w = W.config(cfg, n=n)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    o = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta)
    for k in range(100):
        t_next, n_act = h.next_block()
        act = cpu(h.active())
        h.predict(t_next)
        h.force_jerk(None)
        h.correct_and_timestep()
        o.step()
        assert t_next == o.t and np.array_equal(act, o.active), f"step {k}"
    s = {k: cpu(v) for k, v in h.state(("x", "t", "dt")).items()}
    assert np.array_equal(s["t"], o.t_i) and np.array_equal(s["dt"], o.dt)
    assert np.abs(s["x"] - o.x).max() < 1e-12
    hist, diag = h.level_histogram()
    assert np.array_equal(hist, o.level_hist) and diag[0] == o.nan_count and diag[1] == o.dtmin_clamps
    assert h.block_steps == 100 and h.particle_steps == o.particle_steps
    assert o.min_margin > 1e-10, "a time-step decision sat on a threshold: bit-exactness would be luck"
    h.close()


# ---------------------------------------------------------------------------------------------- energy
@pytest.mark.parametrize("cfg,n", [(1, 1024), (4, 3001), (5, 4096)])
def test_energy_matches_oracle(gd, cfg, n):
    w = W.config(cfg, n=n)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    K, U = h.energy()
    K_ref, U_ref = oracle.energy(w.m, w.x, w.v, w.eps)
    assert abs(K / K_ref - 1) < 1e-13 and abs(U / U_ref - 1) < 1e-13
    h.close()


def test_energy_off_sync_uses_predicted_state(gd):
    w = W.config(1, n=512)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    o = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta)
    h.step(37)
    o.run(max_steps=37)
    K, U = h.energy()
    K_ref, U_ref = o.energy()
    assert abs(K / K_ref - 1) < 1e-11 and abs(U / U_ref - 1) < 1e-11
    h.close()


def test_c1_integration_energy_error_matches_oracle(gd):
    # C1: integrate to t = 0.125; same schedule statistics; |dE/E| within 10 % of the oracle's (north_star),
    # with an absolute floor at the rounding level of E itself (|dE/E| ~ 1e-9 here is ~1e7 ulp: well resolved)
    w = W.config(1)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    o = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta)
    K0, U0 = h.energy()
    K0r, U0r = o.energy()
    steps, psteps = h.run_until(w.t_end)
    o.run(w.t_end)
    assert h.t == o.t == w.t_end
    assert steps == o.block_steps and psteps == o.particle_steps
    K, U = h.energy()
    Kr, Ur = o.energy()
    de = abs((K + U) / (K0 + U0) - 1)
    de_ref = abs((Kr + Ur) / (K0r + U0r) - 1)
    assert abs(de - de_ref) <= 0.1 * de_ref + 1e-13, (de, de_ref)
    h.close()


# ----------------------------------------------------------------------------------------- edge cases
def test_single_particle_and_two_body(gd):
    z = np.zeros((1, 3))
    h = gd.Hermite(np.array([1.0]), z, np.array([[1.0, 0, 0]]), 1e-4, 0.01)
    assert cpu(h.state(("dt",))["dt"])[0] == 0.125
    h.run_until(0.5)
    s = h.state_host(("x", "a"))
    assert h.block_steps == 4 and np.allclose(s["x"][0], [0.5, 0, 0], atol=1e-16) and not s["a"].any()
    h.close()
    w = W.two_body(0.5, 0.5, 1.0, 0.0)
    h = gd.Hermite(w.m, w.x, w.v, 0.0, 0.01)
    o = oracle.HermiteOracle(w.m, w.x, w.v, 0.0, 0.01)
    h.run_until(1.0)
    o.run(1.0)
    assert h.block_steps == o.block_steps
    assert np.abs(h.state_host(("x",))["x"] - o.x).max() < 1e-14
    h.close()


def test_errors_are_reported(gd):
    w = W.config(1, n=64)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    with pytest.raises(gd.GravidyError) as e:
        h.correct_and_timestep()
    assert e.value.code == gd.GD_ESTATE
    with pytest.raises(gd.GravidyError):
        h.set_option("no_such_key", 1)
    with pytest.raises(gd.GravidyError) as e:
        gd.Hermite(w.m, w.x, w.v, w.eps, -1.0)
    assert e.value.code == gd.GD_EINVAL
    h.close()


def test_host_init_equals_device_init(gd):
    w = W.config(4, n=1500)
    h1 = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    h2 = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta, host=True)
    h1.step(5)
    h2.step(5)
    s1, s2 = h1.state_host(), h2.state_host()
    for k in s1:
        assert np.array_equal(s1[k], s2[k]), k
    h1.close()
    h2.close()


# ------------------------------------------------------------------------------ the captured block-step graph
@pytest.mark.parametrize("slice_on", [True, False])
@pytest.mark.parametrize("cfg,n", [(1, 1024), (4, 3000), (5, 2047)])
def test_graph_replay_equals_explicit_calls(gd, cfg, n, slice_on):
    # gd_run_until / gd_step replay a captured graph whose kernels read n_act and t_next from device memory;
    # the explicit call sequence passes them from the host.  Same kernels, same arithmetic: identical bits.
    w = W.config(cfg, n=n)
    hg = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    he = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    hg.set_option("loop_max_nact", 0)            # stage kernels only: the persistent loop sums in another order
    he.set_option("use_graph", 0)
    if slice_on:
        for u in (hg, he):
            u.set_option("slice_passes", 3)      # k_force_slice with three slices per CTA, as at C5's size
    else:
        for u in (hg, he):
            u.set_option("slice_max_nact", 0)    # k_force_jsplit / k_force_ipar take every step
    for steps in (40, 70):                       # 70 is not a multiple of the graph's step count
        pg = hg.step(steps)
        pe = he.step(steps)
        assert pg == pe and hg.t == he.t and hg.block_steps == he.block_steps == (40 if steps == 40 else 110)
    sg, se = hg.state_host(), he.state_host()
    for k in sg:
        assert np.array_equal(sg[k], se[k]), k
    hg.close(); he.close()


def test_graph_run_until_matches_oracle_schedule(gd):
    w = W.config(1)
    t_end = 2.0 ** -5
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    steps, psteps = h.run_until(t_end)
    o = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta)
    o.run(t_end)
    assert h.t == o.t == t_end and steps == o.block_steps and psteps == o.particle_steps
    hist, diag = h.level_histogram()
    assert hist.sum() == psteps
    s = h.state_host(("t", "dt"))
    assert np.array_equal(s["t"], o.t_i) and np.array_equal(s["dt"], o.dt)
    # a second call continues from where the first stopped; max_steps bounds it
    steps2, _ = h.run_until(1.0, max_steps=5)
    assert steps2 == 5 and h.block_steps == steps + 5
    h.close()


# ------------------------------------------------------------------------------ the persistent block-step loop
@pytest.mark.parametrize("cfg,n", [(1, 1024), (2, 16384), (3, 4096), (4, 6000), (5, 2047), (1, 100), (4, 40000)])
def test_loop_first_100_block_steps_bit_exact_schedule(gd, cfg, n):
    # gd_step through the graph whose first node is k_block_loop (small active sets are taken inside the persistent
    # kernel, larger ones by the stage kernels behind it): the schedule must equal the oracle's bit for bit.
    w = W.config(cfg, n=n)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    o = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta)
    psteps = h.step(100)
    for _ in range(100):
        o.step()
    assert h.t == o.t and h.block_steps == 100 and psteps == o.particle_steps
    s = h.state_host(("x", "v", "a", "j", "t", "dt"))
    assert np.array_equal(s["t"], o.t_i) and np.array_equal(s["dt"], o.dt)
    assert np.abs(s["x"] - o.x).max() < 1e-12 and np.abs(s["v"] - o.v).max() < 1e-12
    assert relnorm(s["a"], o.a).max() < 1e-12 and relnorm(s["j"], o.j).max() < 1e-12
    hist, diag = h.level_histogram()
    assert np.array_equal(hist, o.level_hist) and diag[0] == o.nan_count and diag[1] == o.dtmin_clamps
    lp = h.loop_profile()
    assert lp["block_steps"] == 100 and lp["particle_steps"] == psteps, "the persistent loop did not take the steps"
    h.close()


@pytest.mark.parametrize("hi,small", [(1, 96), (3, 96), (8, 2), (64, 0), (1024, 96), (1 << 30, 0), (1 << 30, 7), (1 << 30, 256)])
def test_loop_threshold_sweep_same_schedule(gd, hi, small):
    # whatever share of the steps the loop takes (hi = largest active set it accepts), the schedule is the same
    w = W.config(1)
    t_end = 2.0 ** -5
    ref = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    ref.set_option("loop_max_nact", 0)
    ref.run_until(t_end)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    h.set_option("loop_max_nact", hi)
    h.set_option("loop_small_nact", small)
    steps, psteps = h.run_until(t_end)
    assert h.t == ref.t == t_end and steps == ref.block_steps and psteps == ref.particle_steps
    a, b = h.state_host(), ref.state_host()
    assert np.array_equal(a["t"], b["t"]) and np.array_equal(a["dt"], b["dt"])
    assert np.abs(a["x"] - b["x"]).max() < 1e-12
    ha, _ = h.level_histogram(); hb, _ = ref.level_histogram()
    assert np.array_equal(ha, hb)
    h.close(); ref.close()


def test_loop_is_run_to_run_identical(gd):
    w = W.config(2, n=4096)
    out = []
    for _ in range(2):
        h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
        h.step(200)
        out.append(h.state_host())
        h.close()
    for k in out[0]:
        assert np.array_equal(out[0][k], out[1][k]), k


def test_loop_tiny_systems_and_eps0(gd):
    # N = 1, 2, 3: most CTAs own nothing; eps = 0 exercises the masked self pair inside the loop
    z = np.zeros((1, 3))
    h = gd.Hermite(np.array([1.0]), z, np.array([[1.0, 0, 0]]), 1e-4, 0.01)
    h.run_until(0.5)
    assert h.block_steps == 4 and h.loop_profile()["block_steps"] == 4
    h.close()
    w = W.two_body(0.5, 0.5, 1.0, 0.5)
    h = gd.Hermite(w.m, w.x, w.v, 0.0, 0.01)
    o = oracle.HermiteOracle(w.m, w.x, w.v, 0.0, 0.01)
    steps, psteps = h.run_until(2.0)
    o.run(2.0)
    assert steps == o.block_steps and psteps == o.particle_steps and h.loop_profile()["block_steps"] == steps
    s = h.state_host(("x", "v", "t", "dt"))
    assert np.array_equal(s["t"], o.t_i) and np.array_equal(s["dt"], o.dt)
    assert np.abs(s["x"] - o.x).max() < 1e-13 and np.abs(s["v"] - o.v).max() < 1e-13
    h.close()
    rng = np.random.default_rng(7)
    m, x, v = np.array([0.5, 0.3, 0.2]), rng.normal(size=(3, 3)), 0.3 * rng.normal(size=(3, 3))
    h = gd.Hermite(m, x, v, 1e-4, 0.01)
    o = oracle.HermiteOracle(m, x, v, 1e-4, 0.01)
    steps, _ = h.run_until(0.25)
    o.run(0.25)
    s = h.state_host(("x", "t", "dt"))
    assert steps == o.block_steps and np.array_equal(s["dt"], o.dt) and np.abs(s["x"] - o.x).max() < 1e-13
    h.close()


def test_loop_timers_are_off_by_default_and_change_nothing(gd):
    # the default instantiation of k_block_loop has no timers: step counts are kept, every ns stays 0 and nothing is
    # binned; "loop_timers" switches to the instantiation with timers, which must take the very same steps
    w = W.config(1, n=900)
    plain = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    timed = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    timed.set_option("loop_timers", 1)
    plain.step(150); timed.step(150)
    lp, lt = plain.loop_profile(), timed.loop_profile()
    assert lp["block_steps"] == lt["block_steps"] == 150 and lp["particle_steps"] == lt["particle_steps"]
    assert all(v == 0 for k, v in lp.items() if k.startswith("ns")) and plain.loop_histogram() == []
    assert lt["ns"] > 0 and lt["ns_force"] > 0
    rows = timed.loop_histogram()
    assert sum(r["block_steps"] for r in rows) == 150 and sum(r["particle_steps"] for r in rows) == lt["particle_steps"]
    a, b = plain.state_host(), timed.state_host()
    for k in a:
        assert np.array_equal(a[k], b[k]), k
    timed.set_option("loop_timers", 0)          # back to the plain instantiation: the graph is rebuilt, the bins stop growing
    timed.step(50); plain.step(50)
    assert sum(r["block_steps"] for r in timed.loop_histogram()) == 150 and timed.loop_profile()["block_steps"] == 200
    a, b = plain.state_host(), timed.state_host()
    for k in a:
        assert np.array_equal(a[k], b[k]), k
    plain.close(); timed.close()


def test_loop_resumes_and_honours_max_steps(gd):
    w = W.config(1, n=700)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    ref = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    ref.set_option("loop_max_nact", 0)
    total = 0
    for n in (17, 40, 33):                       # three launches of the loop, each bounded by max_steps
        h.step(n); ref.step(n); total += n
        assert h.block_steps == ref.block_steps == total and h.t == ref.t
    steps, _ = h.run_until(h.t + 2.0 ** -6, max_steps=10 ** 6)
    steps_r, _ = ref.run_until(ref.t + 2.0 ** -6, max_steps=10 ** 6)
    assert steps == steps_r and h.t == ref.t
    a, b = h.state_host(), ref.state_host()
    assert np.array_equal(a["t"], b["t"]) and np.array_equal(a["dt"], b["dt"]) and np.abs(a["x"] - b["x"]).max() < 1e-12
    assert h.loop_profile()["block_steps"] == h.block_steps
    h.close(); ref.close()


def test_c2_energy_error_after_one_time_unit_matches_oracle(gd):
    # north_star: the same |dE/E| to within 10 % after one N-body time unit (C2).  The oracle's side is stored
    # (5 minutes of host time): tests/golden/c2_t1_energy.txt, written by tests/golden/make_c2_t1_energy.py.
    import os
    gold = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "c2_t1_energy.txt")):
        if not line.startswith("#"):
            k, v = line.split()
            gold[k] = float(v)
    w = W.config(2)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    k0, u0 = h.energy()
    steps, psteps = h.run_until(1.0)
    k1, u1 = h.energy()
    h.close()
    # chaotic dynamics: the schedules need not stay identical for 30 k block steps (they do as of round 1)
    assert abs(steps - gold["block_steps"]) <= 1e-3 * gold["block_steps"]
    assert abs(psteps - gold["particle_steps"]) <= 1e-3 * gold["particle_steps"]
    err = abs((k1 + u1) / (k0 + u0) - 1.0)
    err_ref = abs(gold["e1"] / gold["e0"] - 1.0)
    assert abs(k0 + u0 - gold["e0"]) <= 1e-13 * abs(gold["e0"])
    assert abs(err - err_ref) <= 0.1 * err_ref, (err, err_ref)


# ------------------------------------------------------------------------------ diagnostics: Lagrange radii
@pytest.mark.parametrize("cfg,n", [(1, 1024), (2, 16384), (4, 6000), (5, 2047), (1, 3)])
def test_lagrange_radii_match_oracle(gd, cfg, n):
    from oracle import lagrange
    w = W.config(cfg, n=n)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    fr = [0.005, 0.01, 0.02, 0.03, 0.04, 0.05, 0.06, 0.75, 0.90, 0.5, 1.0]    # Fig. 9 + half mass + all
    r, c, mtot = h.lagrange_radii(fr)
    r_ref, c_ref = lagrange.lagrange_radii(w.m, w.x, fr)
    assert abs(mtot - w.m.sum()) <= 1e-14 * w.m.sum() and np.abs(c - c_ref).max() < 1e-14
    # (C5's central particle sits on the centre of mass: its distance is the rounding noise of the centre)
    assert np.all(np.abs(r - r_ref) <= 1e-12 * r_ref + 1e-14), (r, r_ref)
    # and directly against the definition of P:306 written out (plain float cumulative mass, no fixed point): on these
    # inputs it names the same particle per fraction as the fixed-point count, so the device gives that particle's radius
    r_plain, c_plain, who = lagrange.lagrange_radii_plain(w.m, w.x, fr)
    assert np.array_equal(r_plain, r_ref), "the fixed-point and the plain cumulative mass name different particles here"
    assert np.abs(c - c_plain).max() < 1e-14 and np.all(np.abs(r - r_plain) <= 1e-12 * r_plain + 1e-14), (r, r_plain)
    assert np.allclose(np.linalg.norm(w.x[who] - c, axis=1), r, rtol=1e-12, atol=1e-14)
    # about a given centre the centre drops out of the comparison: identical bits
    r2, c2, _ = h.lagrange_radii(fr, center=[0.05, -0.1, 0.2])
    r2_ref, _ = lagrange.lagrange_radii(w.m, w.x, fr, centre=[0.05, -0.1, 0.2])
    assert np.array_equal(r2, r2_ref) and np.array_equal(c2, [0.05, -0.1, 0.2])
    assert np.array_equal(r2, lagrange.lagrange_radii_plain(w.m, w.x, fr, centre=[0.05, -0.1, 0.2])[0])
    h.close()


def test_lagrange_radii_follow_the_predicted_state_and_reject_bad_fractions(gd):
    from oracle import lagrange
    w = W.config(1)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    o = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta)
    h.step(37)
    for _ in range(37):
        o.step()
    xp, _ = oracle.predict(o.t, o.x, o.v, o.a, o.j, o.t_i)
    r, _, _ = h.lagrange_radii([0.1, 0.5, 0.9])
    r_ref, _ = lagrange.lagrange_radii(w.m, xp, [0.1, 0.5, 0.9])
    assert np.abs(r / r_ref - 1.0).max() < 1e-11
    for bad in ([0.0], [1.5], [float("nan")], list(np.linspace(0.01, 0.9, 17))):
        with pytest.raises(gd.GravidyError):
            h.lagrange_radii(bad)
    h.close()


# ------------------------------------------------------------------------------------------- boundary behaviour
def test_init_host_arrays_may_be_reused_at_once(gd):
    # gd_init_host waits for its host-to-device copies (and the repacking kernel) before it returns: scribbling over the
    # caller's arrays right after the call must not change the initial conditions the library took
    import torch
    w = W.config(1)
    ref = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    m, x, v = (torch.from_numpy(u.copy()).pin_memory().numpy() for u in (w.m, w.x, w.v))
    h = gd.Hermite(m, x, v, w.eps, w.eta, host=True)
    m[:] = 7.0; x[:] = np.nan; v[:] = -1.0
    a, b = h.state_host(("x", "v", "a", "j", "dt")), ref.state_host(("x", "v", "a", "j", "dt"))
    for k in a:
        assert np.array_equal(a[k], b[k]), k
    h.close(); ref.close()


def test_level_options_void_the_step_in_flight(gd):
    # changing dt_level_min / max rewrites every dt_i: an active list or force result from before is void, and while the
    # two levels are out of order every stage call is refused
    w = W.config(1, n=300)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    t_next, _ = h.next_block()
    h.predict(t_next)
    h.force_jerk(None)
    h.set_option("dt_level_max", 12)
    with pytest.raises(gd.GravidyError) as e:
        h.correct_and_timestep()
    assert e.value.code == gd.GD_ESTATE
    h.set_option("dt_level_min", 14)                         # min > max: transient
    for call in (h.next_block, lambda: h.predict(0.0), lambda: h.step(1)):
        with pytest.raises(gd.GravidyError) as e:
            call()
        assert e.value.code == gd.GD_ESTATE
    h.set_option("dt_level_max", 16)
    o = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta, dt_min=2.0 ** -16, dt_max=2.0 ** -14)
    assert np.array_equal(h.state_host(("dt",))["dt"], o.dt)
    h.step(20)
    for _ in range(20):
        o.step()
    assert h.t == o.t and np.array_equal(h.state_host(("dt",))["dt"], o.dt)
    h.close()


# --------------------------------------------------- the paper's further applications, Newtonian part
def _further_workload(kind):
    if kind == "two_clusters":
        return W.two_cluster_collision(3000, seed=11, mass_ratio=2.0)          # P:390 "the collision of two clusters"
    return W.central_massive_particle(2500, seed=21, m_central=0.05)          # P:392 "a central massive particle", eps = 1e-5


@pytest.mark.parametrize("kind", ["two_clusters", "central_massive"])
def test_further_workloads_match_oracle(gd, kind):
    # same bar as the five configs: a, jerk 1e-12 and dt bit-exact at init, the first 100 block steps bit-exact, the
    # energy error at the end of a short run within 10 % of the oracle's
    w = _further_workload(kind)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    o = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta)
    s = h.state_host(("a", "j", "dt"))
    assert relnorm(s["a"], o.a).max() < 1e-12 and relnorm(s["j"], o.j).max() < 1e-12 and np.array_equal(s["dt"], o.dt)
    k0, u0 = h.energy()
    K0, U0 = o.energy()
    assert abs(k0 / K0 - 1) < 1e-13 and abs(u0 / U0 - 1) < 1e-13
    for k in range(100):
        t_next, cnt = h.next_block()
        act = h.active().cpu().numpy()
        o.step()
        assert t_next == o.t and np.array_equal(act, o.active), f"schedule differs at block step {k}"
        h.predict(t_next)
        h.force_jerk(None)
        h.correct_and_timestep()
    s = h.state_host(("x", "t", "dt"))
    assert np.array_equal(s["t"], o.t_i) and np.array_equal(s["dt"], o.dt) and np.abs(s["x"] - o.x).max() < 1e-12
    # on through the persistent loop to the workload's end time
    steps, psteps = h.run_until(w.t_end)
    o.run(w.t_end)
    assert h.block_steps == o.block_steps and h.particle_steps == o.particle_steps and h.t == o.t == w.t_end
    k1, u1 = h.energy()
    K1, U1 = o.energy()
    err, err_ref = abs((k1 + u1) / (k0 + u0) - 1), abs((K1 + U1) / (K0 + U0) - 1)
    assert err_ref < 1e-5 and abs(err / err_ref - 1.0) < 0.10, (err, err_ref)
    s = h.state_host(("t", "dt"))
    assert np.array_equal(s["t"], o.t_i) and np.array_equal(s["dt"], o.dt)
    h.close()


# ------------------------------------------------------------------ time-step census, density centre, core radius
@pytest.mark.parametrize("cfg,n", [(1, 1024), (4, 3000), (5, 2047), (2, 257)])
def test_level_census_matches_oracle(gd, cfg, n):
    # P:343 / Fig. 13: particles per CURRENT block step, at t = 0 and after 60 block steps (not the steps-taken histogram)
    from oracle import structure
    w = W.config(cfg, n=n)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    o = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta)
    c0 = h.level_census()
    assert np.array_equal(c0, structure.level_census(o.dt)) and c0.sum() == w.n
    h.step(60)
    for _ in range(60):
        o.step()
    c1 = h.level_census()
    assert np.array_equal(c1, structure.level_census(o.dt)) and c1.sum() == w.n
    assert not np.array_equal(c1, h.level_histogram()[0])
    h.close()


@pytest.mark.parametrize("cfg,n,k", [(1, 1024, 6), (4, 3000, 6), (4, 700, 2), (5, 2047, 8), (2, 300, 6)])
def test_core_radius_matches_oracle(gd, cfg, n, k):
    # P:341 / Fig. 12, reading R25 (Casertano & Hut 1985): rho_i element by element, density centre and core radius
    from oracle import structure
    w = W.config(cfg, n=n)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    rc, xd, rho = h.core_radius(k, want_rho=True)
    rc_ref, xd_ref, rho_ref = structure.core_radius(w.m, w.x, k)
    rho = rho.cpu().numpy()
    # every operation of rho_i is rounded as the definition writes it: the same K neighbours, the same doubles
    assert np.abs(rho / rho_ref - 1.0).max() <= 4e-16, np.abs(rho / rho_ref - 1.0).max()
    assert abs(rc / rc_ref - 1.0) < 1e-12 and np.abs(xd - xd_ref).max() < 1e-12 * max(1.0, np.abs(w.x).max())
    # off a synchronisation time the predicted positions are what is looked at
    o = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta)
    h.step(33)
    for _ in range(33):
        o.step()
    xp, _ = oracle.predict(o.t, o.x, o.v, o.a, o.j, o.t_i)
    rc2, xd2 = h.core_radius(k)
    rc2_ref, xd2_ref, _ = structure.core_radius(w.m, xp, k)
    assert abs(rc2 / rc2_ref - 1.0) < 1e-10 and np.abs(xd2 - xd2_ref).max() < 1e-10
    for bad in (1, 9):
        with pytest.raises(gd.GravidyError):
            h.core_radius(bad)
    h.close()


def test_core_radius_reports_coincident_particles(gd):
    # a particle with K others on its own point: r_iK = 0, the density estimate is infinite and the weighted means NaN --
    # an error, not GD_OK
    w = W.config(1, n=300)
    x = w.x.copy()
    x[10:16] = x[10]                       # six coincident particles: each has five neighbours at distance 0
    h = gd.Hermite(w.m, x, w.v, 1e-2, w.eta)
    for k in (8, 6):                       # the 6th neighbour is somewhere else: fine
        rc, _ = h.core_radius(k)
        assert np.isfinite(rc) and rc > 0
    for k in (5, 2):
        with pytest.raises(gd.GravidyError, match="coincident"):
            h.core_radius(k)
    h.close()


# ------------------------------------------------------------------------------ options that change the schedule
@pytest.mark.parametrize("use_loop", [True, False])
def test_single_halving_variant_matches_oracle(gd, use_loop):
    # DESIGN.md reading R7: the block rule's variant "a single halving per step" (halving_mode 0) on both sides
    w = W.config(4, n=1500)                      # the variants part ways at block step 53 of this input
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    h.set_option("halving_mode", 0)
    if not use_loop:
        h.set_option("loop_max_nact", 0)
    o = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta, halving_mode=0)
    psteps = h.step(150)
    for _ in range(150):
        o.step()
    s = h.state_host(("x", "t", "dt"))
    assert h.t == o.t and psteps == o.particle_steps
    assert np.array_equal(s["t"], o.t_i) and np.array_equal(s["dt"], o.dt) and np.abs(s["x"] - o.x).max() < 1e-12
    # the two variants do differ on this input (otherwise the test would not tell them apart)
    o1 = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta, halving_mode=1)
    for _ in range(150):
        o1.step()
    assert o1.particle_steps != o.particle_steps or not np.array_equal(o1.dt, o.dt)
    h.close()


@pytest.mark.parametrize("level", [6, 9])
def test_shared_step_special_case_matches_oracle(gd, level):
    # SURVEY 8(c) pin 7: dt_min = dt_max makes the scheme the shared-step 4th-order Hermite integrator; every particle
    # is active in every step.  Device: options dt_level_min = dt_level_max; oracle: dt_min = dt_max = 2^-level.
    w = W.config(4, n=1500)
    dt = 2.0 ** -level
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    h.set_option("dt_level_min", level)
    h.set_option("dt_level_max", level)
    o = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta, dt_min=dt, dt_max=dt)
    for k in range(12):
        t_next, n_act = h.next_block()
        assert n_act == w.n and t_next == (k + 1) * dt
        h.predict(t_next)
        h.force_jerk(None)
        h.correct_and_timestep()
        o.step()
    s = h.state_host()
    assert np.array_equal(s["t"], o.t_i) and np.array_equal(s["dt"], o.dt)
    assert np.abs(s["x"] - o.x).max() < 1e-12 and np.abs(s["v"] - o.v).max() < 1e-12
    assert relnorm(s["a"], o.a).max() < 1e-11 and relnorm(s["j"], o.j).max() < 1e-11
    k1, u1 = h.energy()
    k2, u2 = o.energy()
    assert abs((k1 + u1) / (k2 + u2) - 1.0) < 1e-11
    with pytest.raises(gd.GravidyError):
        h.set_option("dt_level_max", level + 1)          # levels can only change before the first step
    h.close()
