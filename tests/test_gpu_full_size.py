"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (default options: gd_init's
all-active evaluation, gd_step through the captured graph / persistent loop, gd_force_jerk's own kernel choice).

The oracle computes what it can one by one: sampled sinks against all N sources (C4, C5), the whole of C3, and --
stored, because the full-size INIT is minutes to an hour of host time -- the first 100 block steps of C3, C4, C5
(tests/golden/c<k>_full_schedule.txt, written by tests/golden/make_full_size_schedule.py from oracle/ only).
Everything else is a property that holds at any size (momentum sums, scheduler invariants).
"""
import zlib

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from conftest import GOLDEN
from paper_1702_00440_b200 import workloads as W

TOL = 1e-12


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


def crc(a) -> int:
    return zlib.crc32(np.ascontiguousarray(a).tobytes()) & 0xFFFFFFFF


# ----------------------------------------------------------------------------------- C3: the isolated sweep
def test_c3_full_size_force_sweep(gd):
    # BASELINE.json configs[2]: N = 65536, n_act in {1, 16, 256, 4096, 65536}, the kernels gd_force_jerk picks itself
    import torch
    w = W.config(3)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    h.predict(0.0)
    kernels = {}
    for n_act in (1, 16, 256, 4096, 65536):
        idx = W.active_indices(w.n, n_act)
        a, j = h.force_jerk(torch.from_numpy(idx).cuda())
        kernels[n_act] = h.last_force_kernel
        a_ref, j_ref = oracle.pairsum(w.m, w.x, w.v, w.eps, idx=idx)
        ea, ej = relnorm(cpu(a), a_ref), relnorm(cpu(j), j_ref)
        assert ea.max() <= TOL and ej.max() <= TOL, (n_act, ea.max(), ej.max())
        if n_act == w.n:
            # pairwise antisymmetry (SURVEY 8c pin 2) on the GPU's own full output
            ma = (w.m[:, None] * cpu(a)).sum(axis=0)
            assert np.abs(ma).max() <= 1e-13 * (w.m * np.linalg.norm(cpu(a), axis=1)).sum()
            # gd_init's evaluation (step a0) is the same sum
            s = h.state(("a", "j"))
            assert relnorm(cpu(s["a"]), a_ref).max() <= TOL and relnorm(cpu(s["j"]), j_ref).max() <= TOL
    assert kernels[65536] == "ipar" and kernels[1] in ("slice", "jsplit")
    h.close()


# ------------------------------------------------------- C4, C5: all-active evaluation, sampled sinks one by one
@pytest.mark.parametrize("cfg", [4, 5])
def test_full_size_all_active_sampled_sinks(gd, cfg):
    w = W.config(cfg)
    assert w.n == {4: 262144, 5: 1048577}[cfg]
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)          # a0: all-active force/jerk + initial time steps
    s = {k: cpu(v) for k, v in h.state(("a", "j", "t", "dt")).items()}
    idx = W.active_indices(w.n, 509, seed=900 + cfg)
    if cfg == 5:
        idx = np.concatenate([idx[idx != w.n - 1], [w.n - 1]]).astype(np.int32)     # the central point mass too
    a_ref, j_ref = oracle.pairsum(w.m, w.x, w.v, w.eps, idx=idx)
    ea, ej = relnorm(s["a"][idx], a_ref), relnorm(s["j"][idx], j_ref)
    assert ea.max() <= TOL and ej.max() <= TOL, (ea.max(), ej.max())
    assert np.array_equal(s["dt"][idx], oracle.initial_dt(a_ref, j_ref, w.eta)) and not s["t"].any()
    # properties at any size: finite, momentum sums vanish to rounding, every dt a power of two inside the clamps
    assert np.isfinite(s["a"]).all() and np.isfinite(s["j"]).all()
    for u in (s["a"], s["j"]):
        tot = (w.m[:, None] * u).sum(axis=0)
        assert np.abs(tot).max() <= 1e-12 * (w.m * np.linalg.norm(u, axis=1)).sum()
    mant, _ = np.frexp(s["dt"])
    assert np.all(mant == 0.5) and s["dt"].max() <= oracle.DT_MAX and s["dt"].min() >= oracle.DT_MIN
    h.close()


def test_c4_all_active_steps_inside_the_block_loop_match_oracle(gd):
    # The path that does most of C4's arithmetic: k_block_loop with tens of thousands of sinks per step (lanes over
    # sinks, 148 partial rows per sink, owners fold and correct).  A shared step (dt_level_min = dt_level_max) makes every
    # block step all-active at N = 262144; gd_run_until takes them inside the loop.  Sampled sinks one by one: a, jerk of
    # the second step against the oracle's sums over the state the device held before it (predicted by the oracle, which
    # the predictor parity test shows bit-identical), and the corrected x, v, t, dt against the oracle's corrector.
    w = W.config(4)
    lvl = 12
    dt = 2.0 ** -lvl
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    h.set_option("dt_level_min", lvl)
    h.set_option("dt_level_max", lvl)
    steps, psteps = h.run_until(dt)
    assert (steps, psteps) == (1, w.n) and h.loop_profile()["block_steps"] == 1
    s1 = h.state_host()
    assert np.all(s1["t"] == dt) and np.all(s1["dt"] == dt)
    steps, psteps = h.run_until(2 * dt)
    assert (steps, psteps) == (1, w.n) and h.loop_profile()["block_steps"] == 2 and h.loop_profile()["particle_steps"] == 2 * w.n
    s2 = h.state_host()
    h.close()
    idx = W.active_indices(w.n, 509, seed=904)
    xp, vp = oracle.predict(2 * dt, s1["x"], s1["v"], s1["a"], s1["j"], s1["t"])
    a_ref, j_ref = oracle.pairsum(w.m, xp, vp, w.eps, idx=idx)
    ea, ej = relnorm(s2["a"][idx], a_ref), relnorm(s2["j"][idx], j_ref)
    assert ea.max() <= TOL and ej.max() <= TOL, (ea.max(), ej.max())
    ref = oracle.correct(idx, 2 * dt, w.eta, s1["x"], s1["v"], s1["a"], s1["j"], s1["t"], s1["dt"], xp, vp, a_ref, j_ref,
                         dt_min=dt, dt_max=dt)
    for k, r in zip(("x", "v", "t", "dt"), (ref[0], ref[1], ref[4], ref[5])):
        if k in ("t", "dt"):
            assert np.array_equal(s2[k][idx], r[idx]), k
        else:
            assert np.abs(s2[k][idx] - r[idx]).max() <= 1e-12 * max(1.0, np.abs(r[idx]).max()), k
    # the whole output: finite, momentum of the accelerations vanishes to rounding
    assert np.isfinite(s2["a"]).all() and np.isfinite(s2["j"]).all()
    tot = (w.m[:, None] * s2["a"]).sum(axis=0)
    assert np.abs(tot).max() <= 1e-12 * (w.m * np.linalg.norm(s2["a"], axis=1)).sum()


# ------------------------------------------------------------------ first 100 block steps at full size (stored)
def read_schedule(cfg):
    steps, kv, samples = [], {}, []
    for line in (GOLDEN / f"c{cfg}_full_schedule.txt").read_text().splitlines():
        tok = line.split("#", 1)[0].split()
        if not tok:
            continue
        if tok[0] == "step":
            steps.append((float.fromhex(tok[1]), int(tok[2]), int(tok[3], 16)))
        elif tok[0] == "sample":
            samples.append((int(tok[1]), np.array([float.fromhex(u) for u in tok[2:]])))
        else:
            kv[tok[0]] = tok[1:]
    return steps, kv, samples


def check_invariants(s, t_now):
    # SURVEY 8c pin 8: t_i = 0 (mod dt_i); t_i <= t <= t_i + dt_i; dt_i a power of two inside the clamps
    t_i, dt = s["t"], s["dt"]
    mant, _ = np.frexp(dt)
    assert np.all(mant == 0.5) and dt.max() <= oracle.DT_MAX and dt.min() >= oracle.DT_MIN
    assert not np.any(np.fmod(t_i, dt)) and np.all(t_i <= t_now) and np.all(t_now <= t_i + dt)


@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_full_size_first_100_block_steps_match_stored_oracle_schedule(gd, cfg):
    if not (GOLDEN / f"c{cfg}_full_schedule.txt").exists():
        pytest.fail(f"tests/golden/c{cfg}_full_schedule.txt missing: run tests/golden/make_full_size_schedule.py {cfg}")
    steps, kv, samples = read_schedule(cfg)
    assert len(steps) == 100 and float(kv["min_margin"][0]) > 1e-10
    w = W.config(cfg)
    # (1) stage by stage through the boundary's per-step calls: every active list
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    for k, (t_ref, n_ref, crc_ref) in enumerate(steps):
        t_next, n_act = h.next_block()
        assert (t_next, n_act) == (t_ref, n_ref), f"step {k}"
        assert crc(cpu(h.active()).astype(np.int32)) == crc_ref, f"step {k}"
        h.predict(t_next)
        h.force_jerk(None)
        h.correct_and_timestep()
    # (2) the path bench.py times: gd_step (captured graph: persistent loop where the slice fits, stage kernels else)
    g = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    psteps = g.step(100)
    for hh in (h, g):
        s = hh.state_host()
        assert hh.t == steps[-1][0] and hh.block_steps == 100
        assert hh.particle_steps == int(kv["particle_steps"][0]) == sum(n for _, n, _ in steps)
        assert crc(s["t"]) == int(kv["crc_t"][0], 16) and crc(s["dt"]) == int(kv["crc_dt"][0], 16)
        hist, diag = hh.level_histogram()
        assert np.array_equal(hist, np.array([int(c) for c in kv["level_hist"]]))
        assert diag[0] == int(kv["nan_count"][0]) and diag[1] == int(kv["dtmin_clamps"][0])
        check_invariants(s, hh.t)
        for i, ref in samples:
            assert np.abs(s["x"][i] - ref[0:3]).max() < 1e-12 and np.abs(s["v"][i] - ref[3:6]).max() < 1e-12
            assert relnorm(s["a"][i], ref[6:9]) <= TOL and relnorm(s["j"][i], ref[9:12]) <= TOL
    assert psteps == int(kv["particle_steps"][0])
    h.close(); g.close()


def test_c5_workload_all_active_plus_10_block_steps_invariants(gd):
    # BASELINE.json configs[4] exactly as bench.py runs it: init + 10 block steps; properties that hold at any size,
    # and the active list of the next step against the definition applied to the device's own (t_i, dt_i)
    w = W.config(5)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    k0, u0 = h.energy()
    psteps = h.step(10)
    s = h.state_host(("t", "dt"))
    check_invariants(s, h.t)
    hist, _ = h.level_histogram()
    assert hist.sum() == psteps == h.particle_steps and h.block_steps == 10
    t_ref, act_ref = oracle.next_block(s["t"], s["dt"])
    t_next, n_act = h.next_block()
    assert t_next == t_ref and n_act == len(act_ref) and np.array_equal(cpu(h.active()), act_ref)
    k1, u1 = h.energy()
    assert abs((k1 + u1) / (k0 + u0) - 1.0) < 1e-9      # 10 tiny block steps: the energy has not moved
    h.close()


def test_contexts_of_different_sizes_coexist(gd):
    # the dynamic shared-memory limit is a property of the kernel function, not of a context: a small context created
    # after a large one must not shrink what the large one may launch with (k_force_slice: 160 KB of source records
    # per CTA at N = 200000; k_block_loop likewise)
    import torch
    big = W.config(4, n=200000)
    small = W.config(1)
    hb = gd.Hermite(big.m, big.x, big.v, big.eps, big.eta)
    hs = gd.Hermite(small.m, small.x, small.v, small.eps, small.eta)
    hb.predict(0.0)
    idx = W.active_indices(big.n, 100, seed=11)
    a, j = hb.force_jerk(torch.from_numpy(idx).cuda())
    assert hb.last_force_kernel == "slice"
    a_ref, j_ref = oracle.pairsum(big.m, big.x, big.v, big.eps, idx=idx)
    assert relnorm(cpu(a), a_ref).max() <= TOL and relnorm(cpu(j), j_ref).max() <= TOL
    assert hb.step(40) > 0 and hs.step(40) > 0 and hb.step(40) > 0       # both persistent loops, interleaved
    assert hb.loop_profile()["block_steps"] == 80 and hs.loop_profile()["block_steps"] == 40
    check_invariants(hb.state_host(("t", "dt")), hb.t)
    hb.close(); hs.close()


@pytest.mark.parametrize("n", [70001, 600000, 1300000])
def test_next_block_one_kernel_form_at_every_chunk_width(gd, n):
    # gd_next_block of mid-size systems is one cooperative kernel whose threads keep 4, 8 or 16 values of t_i + dt_i in
    # registers (65 537 .. 606 208 / .. 1 212 416 / .. 2 424 832 particles on 148 SMs): the three widths against the
    # definition applied to the device's own (t_i, dt_i), on the first block and after some block steps, and in
    # the all-active case (shared step)
    w = W.config(2, n=n)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    for stage in range(3):
        s = h.state_host(("t", "dt"))
        t_ref, act_ref = oracle.next_block(s["t"], s["dt"])
        t_next, n_act = h.next_block()
        assert t_next == t_ref and n_act == len(act_ref) and np.array_equal(cpu(h.active()), act_ref)
        h.next_block()                                       # a second call re-arms its counters correctly
        assert np.array_equal(cpu(h.active()), act_ref)
        if stage == 0:
            h.step(3)
        elif stage == 1 and n <= 600000:
            h.step(20)                                       # through the persistent loop or the graph of stage kernels
    h.close()
    if n == 70001:                                           # every particle active at once: the ordered write of the whole list
        h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
        h.set_option("dt_level_min", 9)
        h.set_option("dt_level_max", 9)
        t_next, n_act = h.next_block()
        assert t_next == 2.0 ** -9 and n_act == n and np.array_equal(cpu(h.active()), np.arange(n, dtype=np.int32))
        h.close()
