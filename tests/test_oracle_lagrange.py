"""Pins of oracle/lagrange.py (Fig. 9): what the definition fixes, not a re-run of its own code."""
import math

import numpy as np

from oracle import lagrange
from paper_1702_00440_b200 import workloads as W

PAPER_FRACTIONS = [0.005, 0.01, 0.02, 0.03, 0.04, 0.05, 0.06, 0.75, 0.90]      # Fig. 9


def test_hand_example_unequal_masses():
    # five particles on the x axis about a fixed centre; masses 1, 2, 3, 2, 2 (total 10), distances 1, 2, 3, 4, 5
    x = np.array([[3.0, 0, 0], [-1.0, 0, 0], [0, 2.0, 0], [0, 0, -5.0], [4.0, 0, 0]])
    m = np.array([3.0, 1.0, 2.0, 2.0, 2.0])
    # sorted by distance: d=1 (m 1, cum 1), d=2 (m 2, cum 3), d=3 (m 3, cum 6), d=4 (m 2, cum 8), d=5 (m 2, cum 10)
    r, _ = lagrange.lagrange_radii(m, x, [0.05, 0.1, 0.11, 0.3, 0.31, 0.6, 0.75, 0.8, 0.81, 1.0], centre=[0, 0, 0])
    assert r.tolist() == [1.0, 1.0, 2.0, 2.0, 3.0, 3.0, 4.0, 4.0, 5.0, 5.0]


def test_equal_masses_is_the_kth_smallest_distance():
    rng = np.random.default_rng(11)
    n = 1000
    x = rng.normal(size=(n, 3))
    m = np.full(n, 1.0 / n)
    c = np.array([0.1, -0.2, 0.3])
    d = np.sort(np.linalg.norm(x - c, axis=1))
    fr = [0.001, 0.01, 0.0105, 0.25, 0.5, 0.9, 0.999, 1.0]
    r, _ = lagrange.lagrange_radii(m, x, fr, centre=c)
    for f, rk in zip(fr, r):
        k = max(1, math.floor(f * n + 1e-9))                 # the k-th particle completes the fraction (f n integer: exactly)
        assert abs(rk - d[k - 1]) <= 1e-15 * d[k - 1] or abs(rk - d[min(k, n - 1)]) <= 1e-15 * d[k], (f, k)
    assert r[-1] == np.linalg.norm(x - c, axis=1).max() or abs(r[-1] - d[-1]) < 1e-15


def test_centre_of_mass_default_and_translation_invariance():
    rng = np.random.default_rng(5)
    x = rng.normal(size=(300, 3))
    m = rng.uniform(0.5, 2.0, size=300)
    r0, c0 = lagrange.lagrange_radii(m, x, [0.1, 0.5, 0.9])
    assert np.allclose(c0, (m[:, None] * x).sum(0) / m.sum(), rtol=0, atol=1e-15)
    shift = np.array([10.0, -3.0, 7.0])
    r1, c1 = lagrange.lagrange_radii(m, x + shift, [0.1, 0.5, 0.9])
    assert np.allclose(c1 - shift, c0, atol=1e-13) and np.allclose(r1, r0, rtol=1e-12)
    # scaling all masses by a constant changes nothing
    r2, _ = lagrange.lagrange_radii(7.0 * m, x, [0.1, 0.5, 0.9])
    assert np.array_equal(r2, r0)


def test_plummer_closed_form():
    # Plummer sphere with scale a = 3 pi / 16 (N-body units): M(<r)/M = (1 + a^2/r^2)^(-3/2)  =>  r_f = a / sqrt(f^(-2/3) - 1);
    # the sampling of workloads.py truncates the mass fraction at 0.999, so fractions are rescaled by that factor.
    w = W.config(2)
    a = 3.0 * math.pi / 16.0
    fr = [0.1, 0.25, 0.5, 0.75, 0.9]
    r, c = lagrange.lagrange_radii(w.m, w.x, fr)
    assert np.abs(c).max() < 1e-12                          # the generator removes the centre of mass
    for f, rk in zip(fr, r):
        exact = a / math.sqrt((0.999 * f) ** (-2.0 / 3.0) - 1.0)
        assert abs(rk / exact - 1.0) < 0.04, (f, rk, exact)   # N = 16384: sampling noise ~ 1 / sqrt(f N) on the mass
    # half-mass radius of the untruncated model: 0.7686 (SURVEY.md pin 9; the paper quotes "0.8")
    assert abs(r[2] - 0.7686) < 0.03


def test_weights_are_exact_integers_and_fit():
    w = W.config(4, n=5000)                                  # Kroupa-like masses over three decades
    wi, e = lagrange.fixed_point_weights(w.m)
    assert int(wi.sum(dtype=np.uint64)) < 2 ** 63 and int(wi.max()) >= 2 ** (62 - 13 - 1)
    assert np.all(np.ldexp(wi.astype(np.float64), -e) == w.m) or np.abs(np.ldexp(wi.astype(np.float64), -e) / w.m - 1).max() < 2.0 ** -40
    fr = PAPER_FRACTIONS
    r, _ = lagrange.lagrange_radii(w.m, w.x, fr)
    assert np.all(np.diff(r) >= 0) and r[0] > 0


def test_plain_definition_on_the_hand_example():
    # the same five particles: the definition itself (float cumulative mass) gives the same radii
    x = np.array([[3.0, 0, 0], [-1.0, 0, 0], [0, 2.0, 0], [0, 0, -5.0], [4.0, 0, 0]])
    m = np.array([3.0, 1.0, 2.0, 2.0, 2.0])
    r, _, who = lagrange.lagrange_radii_plain(m, x, [0.05, 0.11, 0.31, 0.75, 0.81, 1.0], centre=[0, 0, 0])
    assert r.tolist() == [1.0, 2.0, 3.0, 4.0, 5.0, 5.0] and who.tolist() == [1, 2, 0, 4, 3, 3]


def test_fixed_point_variant_names_the_particle_of_the_plain_definition():
    # R24's fixed-point masses are a variant that makes the device comparison independent of summation order; away from
    # exact ties (f M within rounding of a cumulative mass) it must pick the very particle the plain definition picks
    w = W.config(4, n=20000)                                 # Kroupa-like masses: no two cumulative masses coincide
    rng = np.random.default_rng(17)
    fr = np.sort(np.concatenate([PAPER_FRACTIONS, rng.uniform(0.001, 0.999, 200)]))
    c = np.zeros(3)
    rp, _, who = lagrange.lagrange_radii_plain(w.m, w.x, fr, centre=c)
    rf, _ = lagrange.lagrange_radii(w.m, w.x, fr, centre=c)
    d = np.sort(np.linalg.norm(w.x - c, axis=1))
    exact = rp == rf
    # a fraction may land within ~n u M of a cumulative mass: then the two may differ by ONE particle in distance order
    for k in np.nonzero(~exact)[0]:
        i = int(np.searchsorted(d, rp[k]))
        assert rf[k] in (d[max(i - 1, 0)], d[min(i + 1, len(d) - 1)]), (fr[k], rp[k], rf[k])
    assert exact.mean() > 0.98
    # equal masses and f n not an integer: no tie is possible, the two agree exactly
    w2 = W.config(1)
    fr2 = [(k + 0.5) / w2.n for k in (0, 3, 100, 511, 1000, 1022)]
    rp2, _, _ = lagrange.lagrange_radii_plain(w2.m, w2.x, fr2, centre=c)
    rf2, _ = lagrange.lagrange_radii(w2.m, w2.x, fr2, centre=c)
    assert np.array_equal(rp2, rf2)
