"""Pins of oracle/structure.py: the time-step census (Fig. 13) and the density centre / core radius
(Fig. 12; reading R25 = Casertano & Hut 1985) -- against what the definitions fix, not a re-run of the code."""
import math

import numpy as np
import pytest

import oracle
from oracle import structure
from paper_1702_00440_b200 import workloads as W


# ------------------------------------------------------------------------------------------- census
def test_level_census_hand_example():
    dt = np.array([0.125, 0.125, 2.0 ** -10, 2.0 ** -23, 0.25, 1.0, 0.3, 2.0 ** -10])
    c = structure.level_census(dt)
    assert c[3] == 2 and c[10] == 2 and c[23] == 1 and c[2] == 1 and c[0] == 1
    assert c.sum() == 7                                      # 0.3 is not a block step: not counted


def test_level_census_of_an_integration():
    # at every time the census counts every particle once, inside the clamps; the census is NOT the histogram of steps taken
    w = W.config(1)
    o = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta)
    c0 = structure.level_census(o.dt)
    lev = np.round(-np.log2(o.dt)).astype(int)
    assert np.array_equal(c0, np.bincount(lev, minlength=64)) and c0.sum() == w.n
    assert c0[:3].sum() == 0 and c0[24:].sum() == 0
    # "the initial distribution of time steps ... has a log-normal distribution": one hump in log2(dt), i.e.
    # in the level k, whose mean and median agree and whose tails are thin
    k = np.arange(64)
    mean = (k * c0).sum() / w.n
    sd = math.sqrt(((k - mean) ** 2 * c0).sum() / w.n)
    assert abs(mean - np.median(lev)) < 0.75 and 0.5 < sd < 3.0
    assert c0[int(round(mean))] >= 0.15 * w.n
    o.run(0.0625)
    c1 = structure.level_census(o.dt)
    assert c1.sum() == w.n and not np.array_equal(o.level_hist, c1)


# ------------------------------------------------------------------------------------- density / core
def test_knn_density_hand_example():
    # particles on the x axis at 0, 1, 3, 7, 15 with masses 1, 2, 4, 8, 16; K = 2: one neighbour's mass inside the sphere
    # through the second neighbour
    x = np.zeros((5, 3))
    x[:, 0] = [0.0, 1.0, 3.0, 7.0, 15.0]
    m = np.array([1.0, 2.0, 4.0, 8.0, 16.0])
    rho, rk = structure.knn_density(m, x, k=2)
    # i = 0: neighbours at 1 (m 2), 3 -> r_K = 3, mass 2;  i = 1: 0 (m 1) at 1, 3 at 2 -> r_K = 2, mass 1
    # i = 2: 1 (m 2) at 2, 0 at 3 -> r_K = 3, mass 2;      i = 3: 3 (m 4) at 4, 1 at 6 -> r_K = 6, mass 4
    # i = 4: 7 (m 8) at 8, 3 at 12 -> r_K = 12, mass 8
    assert rk.tolist() == [3.0, 2.0, 3.0, 6.0, 12.0]
    vol = lambda r: 4.0 * math.pi / 3.0 * r ** 3
    assert np.allclose(rho, [2 / vol(3), 1 / vol(2), 2 / vol(3), 4 / vol(6), 8 / vol(12)], rtol=1e-15)


def test_kth_neighbour_against_scipy_kdtree():
    from scipy.spatial import cKDTree
    w = W.config(4, n=1500)                                  # unequal masses
    rho, rk = structure.knn_density(w.m, w.x, k=6)
    dist, idx = cKDTree(w.x).query(w.x, k=7)                 # column 0 is the particle itself
    assert np.allclose(rk, dist[:, 6], rtol=1e-14)
    mass = w.m[idx[:, 1:6]].sum(axis=1)
    assert np.allclose(rho, mass / (4.0 * math.pi / 3.0 * dist[:, 6] ** 3), rtol=1e-13)


def test_core_radius_transformations():
    w = W.config(4, n=800)
    rc, xd, rho = structure.core_radius(w.m, w.x)
    shift = np.array([3.0, -2.0, 0.5])
    rc1, xd1, rho1 = structure.core_radius(w.m, w.x + shift)
    assert abs(rc1 / rc - 1) < 1e-12 and np.allclose(xd1 - shift, xd, atol=1e-12) and np.allclose(rho1, rho, rtol=1e-11)
    th = 0.7
    R = np.array([[math.cos(th), -math.sin(th), 0], [math.sin(th), math.cos(th), 0], [0, 0, 1.0]])
    rc2, xd2, _ = structure.core_radius(w.m, w.x @ R.T)
    assert abs(rc2 / rc - 1) < 1e-12 and np.allclose(xd2, R @ xd, atol=1e-12)
    rc3, xd3, rho3 = structure.core_radius(5.0 * w.m, 2.0 * w.x)       # lengths x 2: rho x 5 / 8, r_c x 2, centre x 2
    assert abs(rc3 / (2 * rc) - 1) < 1e-12 and np.allclose(xd3, 2 * xd, atol=1e-12) and np.allclose(rho3, rho * 5 / 8, rtol=1e-12)
    # permuting the particles changes nothing but the order of the sums
    perm = np.random.default_rng(3).permutation(w.n)
    rc4, xd4, rho4 = structure.core_radius(w.m[perm], w.x[perm])
    assert abs(rc4 / rc - 1) < 1e-12 and np.allclose(rho4, rho[perm], rtol=1e-13)


def test_core_radius_plummer_closed_form():
    # rho(r) ~ (1 + r^2/a^2)^(-5/2); with weights rho_i^2 over particles (density rho): r_c^2 = int rho^3 r^2 d^3r / int rho^3 d^3r
    #   = a^2 B(5/2, 5) / B(3/2, 6) = a^2 (3/2)(1/5) = 3 a^2 / 10, a = 3 pi / 16 in N-body units  ->  r_c = 0.3226
    w = W.config(2, n=8192)
    rc, xd, rho = structure.core_radius(w.m, w.x)
    a = 3.0 * math.pi / 16.0
    assert abs(rc / (a * math.sqrt(0.3)) - 1.0) < 0.10, rc
    assert np.linalg.norm(xd) < 0.05                          # the density centre of a centred sphere
    # density of the model: 3 M / (4 pi a^3) (1 + r^2/a^2)^(-5/2); the six-neighbour estimate is noisy per particle
    # (~45 %) but right on average: over the ~250 particles inside r = 0.2
    r = np.linalg.norm(w.x, axis=1)
    sel = r < 0.2
    model = 3.0 / (4.0 * math.pi * a ** 3) * (1.0 + r[sel] ** 2 / a ** 2) ** -2.5
    assert abs(rho[sel].mean() / model.mean() - 1.0) < 0.15
