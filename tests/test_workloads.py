"""Input generators against the closed forms the paper states."""
import math

import numpy as np
import pytest

from paper_1702_00440_b200 import workloads as W
from conftest import read_golden_table


def test_plummer_deterministic_and_centred():
    m1, x1, v1 = W.plummer(2048, seed=7)
    m2, x2, v2 = W.plummer(2048, seed=7)
    assert np.array_equal(x1, x2) and np.array_equal(v1, v2) and np.array_equal(m1, m2)
    _, x3, _ = W.plummer(2048, seed=8)
    assert not np.array_equal(x1, x3)
    assert abs(m1.sum() - 1.0) < 1e-14
    assert np.abs((m1[:, None] * x1).sum(0)).max() < 1e-15
    assert np.abs((m1[:, None] * v1).sum(0)).max() < 1e-15
    assert x1.flags.c_contiguous and x1.dtype == np.float64


def test_plummer_half_mass_radius_matches_closed_form_and_paper():
    a, r_h, *_rest, t_rh, n_p, gamma = read_golden_table("plummer_constants.txt")[0]
    assert abs(a - 3 * math.pi / 16) < 1e-8
    assert abs(r_h - a / math.sqrt(2 ** (2 / 3) - 1)) < 1e-6
    m, x, v = W.plummer(65536, seed=3)
    r = np.sort(np.linalg.norm(x, axis=1))
    rh = r[len(r) // 2]
    assert abs(rh - r_h) < 0.01                       # closed form
    assert abs(rh - 0.8) < 0.05                       # P:233 "half-mass radius of 0.8"
    # Eq. 5 with the printed T_rh = 112.186 for N = 8192 implies r_h ~ 0.762
    rh_paper = (t_rh * math.log(gamma * n_p) / 0.138) ** (2 / 3) / n_p ** (2 / 3)
    assert abs(rh - rh_paper) < 0.02


def test_plummer_nbody_units_energy_and_virial():
    # direct O(N^2) sums with scipy (not the oracle): E = -1/4, K/|U| = 1/2 up to sampling noise
    from scipy.spatial.distance import pdist
    n = 4096
    m, x, v = W.plummer(n, seed=1)
    K = 0.5 * (m * (v * v).sum(1)).sum()
    iu = np.triu_indices(n, 1)
    U = -(m[iu[0]] * m[iu[1]] / pdist(x)).sum()
    assert abs(K + U + 0.25) < 0.02
    assert abs(K / abs(U) - 0.5) < 0.03


def test_plummer_velocity_below_escape_speed():
    m, x, v = W.plummer(8192, seed=2)
    a = 3 * math.pi / 16
    # undo CoM shift influence: tiny; v_esc^2 = 2 / sqrt(r^2 + a^2)
    r2 = (x * x).sum(1)
    assert np.all((v * v).sum(1) <= 2.0 / np.sqrt(r2 + a * a) * (1 + 1e-3) + 1e-3)


def test_kroupa_segments():
    n = 200000
    m = W.kroupa_masses(n, seed=40)
    assert abs(m.sum() - 1.0) < 1e-12
    raw = m / m.min() * 0.1                      # smallest sample sits at ~m_lo
    assert raw.max() <= 100.0 * 1.01

    def seg(a, lo, hi, k):
        return (hi ** (k - a) - lo ** (k - a)) / (k - a)
    w1, w2 = seg(1.3, .1, .5, 1), 0.5 * seg(2.3, .5, 100, 1)
    p1 = w1 / (w1 + w2)
    assert abs((raw < 0.5).mean() - p1) < 5e-3   # ~0.729
    # slope inside each segment from log-binned counts
    for lo, hi, alpha in ((0.1, 0.5, 1.3), (0.5, 20.0, 2.3)):
        edges = np.geomspace(lo, hi, 9)
        cnt, _ = np.histogram(raw, edges)
        mid = np.sqrt(edges[1:] * edges[:-1])
        slope = np.polyfit(np.log(mid), np.log(cnt / np.diff(edges)), 1)[0]
        assert abs(slope + alpha) < 0.08


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5])
def test_configs_shapes(k):
    n_small = 512
    w = W.config(k, n=n_small)
    n = n_small + (1 if k == 5 else 0)
    assert w.n == n and w.x.shape == (n, 3) and w.v.shape == (n, 3)
    assert w.eps == 1e-4 and w.eta == 0.01
    if k == 5:
        assert w.m[-1] == 0.01 and not w.x[-1].any() and not w.v[-1].any()
        assert abs(w.m.sum() - 1.01) < 1e-12
    else:
        assert abs(w.m.sum() - 1.0) < 1e-12
    if k == 4:
        assert w.m.max() / w.m.min() > 20


def test_config_full_sizes_listed():
    assert W.CONFIG_N == {1: 1024, 2: 16384, 3: 65536, 4: 262144, 5: 1048576}


def test_active_indices():
    for n_act in (1, 16, 256, 4096, 65536):
        idx = W.active_indices(65536, n_act)
        assert idx.dtype == np.int32 and idx.shape == (n_act,)
        assert np.all(np.diff(idx) > 0) and idx.min() >= 0 and idx.max() < 65536
    assert np.array_equal(W.active_indices(65536, 16), W.active_indices(65536, 16))


def test_two_body_closed_form_setup():
    w = W.two_body(0.5, 0.5, 1.0, 0.0)
    assert abs(w.meta["period"] - 2 * math.pi) < 1e-14
    vrel = np.linalg.norm(w.v[1] - w.v[0])
    assert abs(vrel - 1.0) < 1e-14               # circular: v^2 = M/r
    assert np.abs((w.m[:, None] * w.v).sum(0)).max() < 1e-16


@pytest.mark.parametrize("cfg,n", [(3, 65536), (4, 262144), (5, 1048577)])
def test_stored_full_size_schedules_are_well_formed(cfg, n):
    # tests/golden/c<k>_full_schedule.txt (the oracle's first 100 block steps at full size, written by
    # tests/golden/make_full_size_schedule.py): times strictly increasing dyadic values, counts consistent with the
    # totals, the level histogram sums to the particle steps, 64 samples inside the system
    from conftest import GOLDEN
    steps, kv, samples = [], {}, []
    for line in (GOLDEN / f"c{cfg}_full_schedule.txt").read_text().splitlines():
        tok = line.split("#", 1)[0].split()
        if not tok:
            continue
        if tok[0] == "step":
            steps.append((float.fromhex(tok[1]), int(tok[2])))
        elif tok[0] == "sample":
            samples.append(int(tok[1]))
        else:
            kv[tok[0]] = tok[1:]
    assert len(steps) == 100 and len(samples) == 64 and all(0 <= i < n for i in samples)
    t = np.array([s[0] for s in steps])
    assert np.all(np.diff(t) > 0) and np.all(t * 2.0 ** 23 == np.round(t * 2.0 ** 23))
    assert all(1 <= s[1] <= n for s in steps)
    assert sum(s[1] for s in steps) == int(kv["particle_steps"][0]) == sum(int(c) for c in kv["level_hist"])
    assert float(kv["min_margin"][0]) > 1e-10 and int(kv["nan_count"][0]) == 0


# ------------------------------------------------------------- the paper's further applications, Newtonian
def test_two_cluster_collision_generator():
    from scipy.spatial.distance import pdist
    w = W.two_cluster_collision(3000, seed=11, mass_ratio=2.0, apocentre=3.0, ecc=0.5)
    n1, n2 = w.meta["n1"], w.meta["n2"]
    assert n1 == 2000 and n2 == 1000 and w.n == 3000 and abs(w.m.sum() - 1.0) < 1e-14
    M1, M2 = w.meta["M1"], w.meta["M2"]
    assert abs(M1 - 2.0 / 3.0) < 1e-15 and abs(M2 - 1.0 / 3.0) < 1e-15
    # whole system: centre of mass at rest at the origin
    assert np.abs((w.m[:, None] * w.x).sum(0)).max() < 1e-14 and np.abs((w.m[:, None] * w.v).sum(0)).max() < 1e-14
    # the two centres: apocentre separation along x, apocentre speed of the Kepler orbit along y
    c1, c2 = w.x[:n1].mean(0), w.x[n1:].mean(0)
    u1, u2 = w.v[:n1].mean(0), w.v[n1:].mean(0)
    assert np.allclose(c2 - c1, [3.0, 0, 0], atol=1e-13)
    vrel = math.sqrt(1.0 * (1 - 0.5) / 3.0)
    assert np.allclose(u2 - u1, [0, vrel, 0], atol=1e-13) and abs(w.meta["vrel"] - vrel) < 1e-15
    # orbital energy and angular momentum of two point masses on that orbit: E = -M1 M2 / 2a, a = d / (1 + e)
    mu = M1 * M2 / (M1 + M2)
    E_orb = 0.5 * mu * vrel ** 2 - M1 * M2 / 3.0
    assert abs(E_orb - (-M1 * M2 / (2.0 * w.meta["semi_major"]))) < 1e-15
    # each cluster alone is a Plummer sphere of its mass in virial equilibrium: 2K/|U| = 1 in its own frame
    for sl, M in ((slice(0, n1), M1), (slice(n1, None), M2)):
        m, x, v = w.m[sl], w.x[sl], w.v[sl] - w.v[sl].mean(0)
        K = 0.5 * (m * (v * v).sum(1)).sum()
        iu = np.triu_indices(len(m), 1)
        U = -(m[iu[0]] * m[iu[1]] / pdist(x)).sum()
        assert abs(2 * K / abs(U) - 1.0) < 0.06
        assert abs((K + U) / (-0.25 * M * M) - 1.0) < 0.08      # E = -M^2 / 4 at unit length scale
    # deterministic, and a different seed differs
    w2 = W.two_cluster_collision(3000, seed=11, mass_ratio=2.0)
    assert np.array_equal(w.x, w2.x) and not np.array_equal(w.x, W.two_cluster_collision(3000, seed=12, mass_ratio=2.0).x)


def test_central_massive_particle_generator():
    w = W.central_massive_particle(2048, seed=21, m_central=0.05)
    assert w.n == 2049 and abs(w.m.sum() - 1.0) < 1e-14 and w.m[-1] == 0.05
    assert abs(w.m[-1] / w.m[0] - 0.05 * 2048 / 0.95) < 1e-9          # ~108 stellar masses
    assert np.abs((w.m[:, None] * w.x).sum(0)).max() < 1e-15 and np.abs((w.m[:, None] * w.v).sum(0)).max() < 1e-15
    # the heavy particle starts (almost) at rest at the centre: displaced only by the removal of the centre of mass
    assert np.linalg.norm(w.x[-1]) < 1e-12 and np.linalg.norm(w.v[-1]) < 1e-12
    assert w.eps == 1e-5 and w.eps < 1e-4                              # "small epsilon"
    # the stars: a Plummer sphere of mass 0.95 at the unit-mass length scale (half-mass radius 0.7686)
    r = np.sort(np.linalg.norm(w.x[:-1], axis=1))
    assert abs(r[1024] - 0.7686) < 0.05
