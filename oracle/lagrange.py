"""Lagrange radii -- TEST INFRASTRUCTURE, not product (plain numpy; shares nothing with the CUDA path).

P:306: "the so-called Lagrange radii (the radii of spheres containing a certain mass fraction of the system)";
Fig. 9 and Fig. 11 plot them for 0.5, 1, 2, 3, 4, 5, 6, 75 and 90 % of the total mass.
The definition written out: sort the particles by distance from the centre, accumulate their masses in that order,
and take the distance of the first particle at which the accumulated mass reaches the fraction.

Readings of what the paper leaves open (R23, R24):
  centre  the centre of mass, sum m x / sum m (or a centre given by the caller);
  masses  accumulated in fixed point, w_i = rint(m_i 2^e), e = 62 - ceil(log2 n) - (floor(log2 max m) + 1), so that the
          accumulated mass is an exact integer and "reaches the fraction" means  cum >= max(1, trunc(f * float(W))),
          W = sum w_i (at most W).  With exact sums the answer does not depend on any summation order.
Parity: pinned by tests/test_oracle_lagrange.py (hand example, equal-mass k-th distance, the Plummer closed form).
"""
from __future__ import annotations

import math

import numpy as np


def centre_of_mass(m, x):
    m = np.asarray(m, dtype=np.float64)
    x = np.asarray(x, dtype=np.float64)
    return (m[:, None] * x).sum(axis=0) / m.sum()


def fixed_point_weights(m):
    """w_i = rint(m_i 2^e) as Python-exact uint64, and e."""
    m = np.asarray(m, dtype=np.float64)
    n = m.shape[0]
    lg = 0
    while (1 << lg) < n:
        lg += 1
    e = 62 - lg - (math.frexp(float(m.max()))[1])          # frexp exponent = floor(log2 max m) + 1
    w = np.rint(np.ldexp(m, e)).astype(np.uint64)
    return w, e


def lagrange_radii(m, x, fractions, centre=None):
    """-> (radii[len(fractions)], centre[3]).  x: [n,3] positions, m: [n] masses."""
    m = np.asarray(m, dtype=np.float64)
    x = np.asarray(x, dtype=np.float64)
    c = centre_of_mass(m, x) if centre is None else np.asarray(centre, dtype=np.float64)
    d = x - c
    r2 = (d[:, 0] * d[:, 0] + d[:, 1] * d[:, 1]) + d[:, 2] * d[:, 2]
    w, _ = fixed_point_weights(m)
    order = np.argsort(r2, kind="stable")
    cum = np.cumsum(w[order], dtype=np.uint64)               # exact: W < 2^63 by the choice of e
    W = int(cum[-1])
    out = np.empty(len(fractions))
    for k, f in enumerate(fractions):
        target = min(max(1, int(float(f) * float(W))), W)
        i = int(np.searchsorted(cum, np.uint64(target), side="left"))   # first index with cum >= target
        out[k] = math.sqrt(r2[order[i]])
    return out, c
