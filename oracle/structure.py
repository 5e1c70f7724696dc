"""Structure diagnostics of the paper's validation plots -- TEST INFRASTRUCTURE, not product (plain numpy; shares
nothing with the CUDA path).

1. Time-step census ("the distribution of the time steps ... the initial distribution of time steps in the system
   has a log-normal distribution"; Fig. 13 P:363 plots it at four times): how many particles hold each block step
   dt = 2^-k AT ONE TIME.  (The per-level count of particle STEPS taken since t = 0 is a different thing: level_hist of
   the integrator.)  The definition written out: counts[k] = #{ i : dt_i = 2^-k }.

2. Core radius and density centre ("the core radius as calculated at T=0"; Fig. 12 P:359 "The blue circle
   depict the core radius at T = 0").  The paper prints no definition.  Reading R25: the estimator of
   Casertano & Hut (1985) in the form the direct-summation codes the paper compares itself with use (NBODY6):
     rho_i  = (sum of the masses of the K - 1 nearest neighbours of i) / (4 pi / 3 r_iK^3),  r_iK = distance from i to its
              K-th nearest neighbour, K = 6; neither particle i nor the K-th neighbour is counted in the mass;
     x_d    = sum_i rho_i x_i / sum_i rho_i                                      (density centre)
     r_c    = sqrt( sum_i rho_i^2 |x_i - x_d|^2 / sum_i rho_i^2 )               (core radius)
   Written out exactly so: all N - 1 distances of every particle, sorted.  O(N^2 log N); N up to a few 10^4.

Parity: pinned by tests/test_oracle_structure.py (hand examples, scipy's k-d tree as the library routine for the K-th
neighbour, translation / rotation / scale behaviour, the closed form for a Plummer sphere, r_c = a sqrt(3/10)).
"""
from __future__ import annotations

import math

import numpy as np


def level_census(dt, levels: int = 64):
    """counts[k] = number of particles whose current step is exactly 2^-k (k = 0 .. levels-1)."""
    dt = np.asarray(dt, dtype=np.float64)
    counts = np.zeros(levels, dtype=np.int64)
    for h in dt:
        mant, e = math.frexp(float(h))               # h = mant 2^e, mant in [0.5, 1): a power of two has mant = 0.5
        k = 1 - e
        if mant == 0.5 and 0 <= k < levels:
            counts[k] += 1
    return counts


def knn_density(m, x, k: int = 6):
    """rho_i of Casertano & Hut (1985) from the K nearest neighbours; -> (rho[n], r_K[n])."""
    m = np.asarray(m, dtype=np.float64)
    x = np.asarray(x, dtype=np.float64)
    n = m.shape[0]
    assert n > k, "need more than K particles"
    rho, rk = np.empty(n), np.empty(n)
    for i in range(n):
        d = x - x[i]
        r2 = (d[:, 0] * d[:, 0] + d[:, 1] * d[:, 1]) + d[:, 2] * d[:, 2]
        r2[i] = np.inf                                # j != i
        order = np.argsort(r2, kind="stable")[:k]     # the K nearest, nearest first
        mass = 0.0
        for j in order[: k - 1]:                      # the K - 1 nearest, nearest first
            mass += m[j]
        r = math.sqrt(r2[order[k - 1]])
        rk[i] = r
        rho[i] = mass / (4.0 * math.pi / 3.0 * r * r * r)
    return rho, rk


def core_radius(m, x, k: int = 6):
    """-> (r_c, x_d[3], rho[n]): density centre and core radius as defined in the header."""
    x = np.asarray(x, dtype=np.float64)
    rho, _ = knn_density(m, x, k)
    s = 0.0
    c = np.zeros(3)
    for i in range(x.shape[0]):                       # index order
        s += rho[i]
        c += rho[i] * x[i]
    xd = c / s
    num = den = 0.0
    for i in range(x.shape[0]):
        d = x[i] - xd
        w = rho[i] * rho[i]
        num += w * ((d[0] * d[0] + d[1] * d[1]) + d[2] * d[2])
        den += w
    return math.sqrt(num / den), xd, rho
