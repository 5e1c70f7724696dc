"""Lagrange radii -- TEST INFRASTRUCTURE, not product (plain numpy; shares nothing with the CUDA path).

P:306: "the so-called Lagrange radii (the radii of spheres containing a certain mass fraction of the system)";
Fig. 9 and Fig. 11 plot them for 0.5, 1, 2, 3, 4, 5, 6, 75 and 90 % of the total mass.
The definition written out: sort the particles by distance from the centre, accumulate their masses in that order,
and take the distance of the first particle at which the accumulated mass reaches the fraction.

Two functions:
  lagrange_radii_plain  THE DEFINITION, nothing else: a plain float cumulative mass in order of distance, and the
          radius of fraction f is the distance of the first particle at which that cumulative mass reaches f * M.
  lagrange_radii        the same with the masses counted in fixed point (R24): w_i = rint(m_i 2^e),
          e = 62 - ceil(log2 n) - (floor(log2 max m) + 1), so that the accumulated mass is an exact integer and "reaches
          the fraction" means  cum >= max(1, trunc(f * float(W))),  W = sum w_i.  With exact sums the answer does not
          depend on any summation order, which is what an element-by-element comparison with a parallel device
          selection needs.  It is a documented VARIANT of the definition, not the definition: the two name the same
          particle unless f * M falls within rounding (~n u M) of one of the cumulative masses -- an exact tie such as
          f n integer for equal masses -- where they may differ by one particle in the order of distance
          (tests/test_oracle_lagrange.py::test_fixed_point_variant_names_the_particle_of_the_plain_definition).
Reading of what the paper leaves open (R23): the centre is the centre of mass, sum m x / sum m, or a centre
given by the caller.
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


def lagrange_radii_plain(m, x, fractions, centre=None):
    """The definition of P:306 written out: particles in order of distance from the centre, plain float cumulative
    mass, radius of fraction f = distance of the first particle at which the cumulative mass is >= f * M.
    -> (radii[len(fractions)], centre[3], index of that particle per fraction)."""
    m = np.asarray(m, dtype=np.float64)
    x = np.asarray(x, dtype=np.float64)
    c = centre_of_mass(m, x) if centre is None else np.asarray(centre, dtype=np.float64)
    r = np.sqrt(((x - c) ** 2).sum(axis=1))
    order = np.argsort(r, kind="stable")
    cum = np.cumsum(m[order])
    M = cum[-1]
    radii, who = np.empty(len(fractions)), np.empty(len(fractions), dtype=np.int64)
    for k, f in enumerate(fractions):
        i = min(int(np.searchsorted(cum, float(f) * M, side="left")), len(cum) - 1)
        radii[k], who[k] = r[order[i]], order[i]
    return radii, c, who
