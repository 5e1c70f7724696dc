"""Pins for the oracle's PAIRSUM and ENERGY (Eq. 3, P:188 fn. 11, Eq. 2).

Each test fixes the oracle against something other than itself: hand-computed numbers, invariants,
a finite difference of the acceleration, a gradient of the potential taken by mpmath, and
extended-precision brute force.
"""
import math

import mpmath as mp
import numpy as np
import pytest

import oracle
from paper_1702_00440_b200 import workloads as W
from conftest import read_golden_table


def relnorm(u, ref):
    u, ref = np.asarray(u, dtype=np.float64), np.asarray(ref, dtype=np.float64)
    return np.linalg.norm(u - ref, axis=-1) / np.linalg.norm(ref, axis=-1)


def test_hand_example():
    m = np.array([0.0, 1.0])
    x = np.array([[0, 0, 0], [3, 4, 0.0]])
    v = np.array([[0, 0, 0], [1, 2, 0.0]])
    for eps2, *ref in read_golden_table("pairsum_hand_example.txt"):
        for mode in ("plain", "compensated"):
            a, j = oracle.pairsum(m, x, v, math.sqrt(eps2), mode=mode)
            assert np.allclose(a[0], ref[:3], rtol=4e-16, atol=0)
            assert np.allclose(j[0], ref[3:], rtol=1e-15, atol=0)
        assert not a[1].any() and not j[1].any()        # the only other source is massless


def test_two_bodies_attract():
    # sign convention (Eq. 1): each body accelerates toward the other
    w = W.two_body(0.3, 0.7, 2.0)
    a, _ = oracle.pairsum(w.m, w.x, w.v, 0.0)
    d = w.x[1] - w.x[0]
    assert np.dot(a[0], d) > 0 and np.dot(a[1], d) < 0
    assert np.allclose(np.linalg.norm(a[0]), 0.7 / 4.0, rtol=1e-15)
    assert np.allclose(np.linalg.norm(a[1]), 0.3 / 4.0, rtol=1e-15)


@pytest.mark.parametrize("eps", [0.0, 1e-4, 0.1])
def test_momentum_invariants(eps):
    # pairwise antisymmetry: sum m a = 0 and sum m jerk = 0
    w = W.random_cluster(300, seed=11)
    a, j = oracle.pairsum(w.m, w.x, w.v, eps)
    scale_a = (w.m[:, None] * np.abs(a)).sum()
    scale_j = (w.m[:, None] * np.abs(j)).sum()
    assert np.abs((w.m[:, None] * a).sum(0)).max() < 1e-14 * scale_a
    assert np.abs((w.m[:, None] * j).sum(0)).max() < 1e-14 * scale_j


@pytest.mark.parametrize("eps", [1e-4, 0.05])
def test_jerk_is_time_derivative_of_acceleration(eps):
    # jerk = d/dt a(x + v t) at t = 0, central difference, velocities frozen
    w = W.random_cluster(64, seed=5)
    _, j = oracle.pairsum(w.m, w.x, w.v, eps)
    h = 1e-5
    ap, _ = oracle.pairsum(w.m, w.x + h * w.v, w.v, eps)
    am, _ = oracle.pairsum(w.m, w.x - h * w.v, w.v, eps)
    fd = (ap - am) / (2 * h)
    assert relnorm(fd, j).max() < 1e-6


def _mp_potential_derivatives(w, eps, i):
    """a_i = -grad_i Phi and jerk_i = d/dt of that along x + v t, from the potential only (50 digits)."""
    mp.mp.dps = 50
    n = w.n
    X = [[mp.mpf(float(c)) for c in w.x[k]] for k in range(n)]
    V = [[mp.mpf(float(c)) for c in w.v[k]] for k in range(n)]
    M = [mp.mpf(float(c)) for c in w.m]
    e2 = mp.mpf(eps) ** 2

    def phi_i(pos_i, t):
        s = mp.mpf(0)
        for k in range(n):
            if k == i:
                continue
            d2 = sum((X[k][c] + V[k][c] * t - pos_i[c]) ** 2 for c in range(3)) + e2
            s -= M[k] / mp.sqrt(d2)
        return s

    def acc(t, comp):
        base = [X[i][c] + V[i][c] * t for c in range(3)]

        def f(u):
            p = list(base)
            p[comp] = u
            return phi_i(p, t)
        return -mp.diff(f, base[comp])

    a = [acc(mp.mpf(0), c) for c in range(3)]
    j = [mp.diff(lambda t, c=c: acc(t, c), mp.mpf(0)) for c in range(3)]
    return np.array([float(u) for u in a]), np.array([float(u) for u in j])


@pytest.mark.parametrize("eps", [0.0, 1e-2])
def test_against_gradient_of_potential_mpmath(eps):
    w = W.random_cluster(5, seed=3)
    a, j = oracle.pairsum(w.m, w.x, w.v, eps)
    for i in (0, 3):
        a_ref, j_ref = _mp_potential_derivatives(w, eps, i)
        assert relnorm(a[i], a_ref) < 1e-14
        assert relnorm(j[i], j_ref) < 1e-13


@pytest.mark.parametrize("eps", [0.0, 1e-4, 0.1])
@pytest.mark.parametrize("n", [2, 17, 64])
def test_long_double_brute_force(n, eps):
    w = W.random_cluster(n, seed=100 + n)
    a_ld, j_ld = oracle.pairsum_longdouble(w.m, w.x, w.v, eps)
    for mode in ("plain", "compensated"):
        a, j = oracle.pairsum(w.m, w.x, w.v, eps, mode=mode)
        # a few u, times the cancellation between pair terms (|sum| can be ~10x below sum|terms|)
        assert relnorm(a, a_ld.astype(np.float64)).max() < 1e-14
        assert relnorm(j, j_ld.astype(np.float64)).max() < 3e-14


def test_long_double_brute_force_itself_vs_mpmath():
    # the extended-precision routine is pinned too: 30-digit evaluation of the definition at N = 4
    mp.mp.dps = 30
    w = W.random_cluster(4, seed=9)
    a_ld, j_ld = oracle.pairsum_longdouble(w.m, w.x, w.v, 1e-4)
    a_ref, j_ref = _mp_potential_derivatives(w, 1e-4, 2)
    assert relnorm(a_ld[2].astype(np.float64), a_ref) < 1e-15
    assert relnorm(j_ld[2].astype(np.float64), j_ref) < 1e-15


def test_plain_and_compensated_agree_to_sqrtN_u():
    w = W.config(1)
    a0, j0 = oracle.pairsum(w.m, w.x, w.v, w.eps, mode="plain")
    a1, j1 = oracle.pairsum(w.m, w.x, w.v, w.eps, mode="compensated")
    u = 2.0 ** -53
    assert 0 < relnorm(a0, a1).max() < 40 * math.sqrt(w.n) * u
    assert 0 < relnorm(j0, j1).max() < 400 * math.sqrt(w.n) * u


def test_subset_rows_equal_full_rows():
    w = W.config(1)
    idx = W.active_indices(w.n, 16)
    a, j = oracle.pairsum(w.m, w.x, w.v, w.eps)
    a_s, j_s = oracle.pairsum(w.m, w.x, w.v, w.eps, idx=idx)
    assert np.array_equal(a_s, a[idx]) and np.array_equal(j_s, j[idx])


def test_thread_count_independent():
    w = W.random_cluster(257, seed=1)
    nt = oracle.num_threads()
    try:
        oracle.set_num_threads(1)
        a1, j1 = oracle.pairsum(w.m, w.x, w.v, 1e-4, mode="plain")
        oracle.set_num_threads(max(2, nt))
        a2, j2 = oracle.pairsum(w.m, w.x, w.v, 1e-4, mode="plain")
    finally:
        oracle.set_num_threads(nt)
    assert np.array_equal(a1, a2) and np.array_equal(j1, j2)


def test_single_particle_and_coincident_softened():
    a, j = oracle.pairsum(np.array([1.0]), np.zeros((1, 3)), np.zeros((1, 3)), 1e-4)
    assert not a.any() and not j.any()
    # two coincident particles with softening: zero separation gives exactly zero force
    a, j = oracle.pairsum(np.array([.5, .5]), np.zeros((2, 3)), np.array([[0, 0, 0], [1., 0, 0]]), 1e-2)
    assert not a.any()
    assert np.allclose(j[0], [0.5 / 1e-6, 0, 0])


# ------------------------------------------------------------------------------------------ energy
def test_energy_two_body_closed_form():
    w = W.two_body(0.5, 0.5, 1.0, 0.0)
    K, U = oracle.energy(w.m, w.x, w.v, 0.0)
    assert abs(U + 0.25) < 1e-16 and abs(K - 0.125) < 1e-16      # E = -1/8 = -G m1 m2 / 2a
    K, U = oracle.energy(w.m, w.x, w.v, 0.75 ** 0.5)               # softened: 1/sqrt(1 + 0.75)
    assert abs(U + 0.25 / math.sqrt(1.75)) < 1e-16


def test_energy_against_scipy_pdist():
    from scipy.spatial.distance import pdist
    w = W.config(1)
    K, U = oracle.energy(w.m, w.x, w.v, w.eps)
    iu = np.triu_indices(w.n, 1)
    U_ref = -(w.m[iu[0]] * w.m[iu[1]] / np.sqrt(pdist(w.x) ** 2 + w.eps ** 2)).sum()
    K_ref = 0.5 * (w.m * (w.v ** 2).sum(1)).sum()
    assert abs(U - U_ref) < 1e-13 * abs(U_ref) and abs(K - K_ref) < 1e-14 * K_ref


def test_force_is_gradient_of_energy():
    # the softened potential (reading R8) is the one whose gradient is Eq. 3: dU/dx_i = -m_i a_i
    w = W.random_cluster(40, seed=2, eps=0.05)
    a, _ = oracle.pairsum(w.m, w.x, w.v, w.eps)
    h = 1e-6
    for i, c in ((0, 0), (7, 2), (39, 1)):
        xp, xm = w.x.copy(), w.x.copy()
        xp[i, c] += h
        xm[i, c] -= h
        dU = (oracle.energy(w.m, xp, w.v, w.eps)[1] - oracle.energy(w.m, xm, w.v, w.eps)[1]) / (2 * h)
        assert abs(dU + w.m[i] * a[i, c]) < 1e-7 * abs(w.m[i] * a[i, c]) + 1e-10
