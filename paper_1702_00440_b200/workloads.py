"""Seeded synthetic inputs shaped like the paper's workloads.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
path.  It holds none of the method's arithmetic (no forces, no energies, no
integrator): it only draws initial conditions.

The paper's runs start from McLuster-generated equal-mass Plummer spheres in
N-body units (§3.1) and, for the mass-spectrum
experiment, a Kroupa IMF (§4.2.2).  Those input files are not
available, so the same *distributions* are sampled here from
``numpy.random.Generator(PCG64(seed))``:

* Plummer sphere by the Aarseth-Henon-Wielen (1974, cited PAPER.md:516) recipe,
  scaled analytically to N-body units (G = M = 1, E = -1/4: positions x 3pi/16,
  velocities x sqrt(16/(3pi))), centre of mass removed.  No exact rescale to
  E = -1/4 is applied (that would need the method's energy sum); the paper's own
  input had E = -0.256.
* Kroupa-like two-segment power law (alpha = 1.3 on [0.1, 0.5), 2.3 on
  [0.5, 100], continuous at 0.5) by inverse CDF, normalised to total mass 1.

``config(k)`` builds the five BASELINE.json configs C1..C5.

Two further workloads from the paper's list of applications (section 6: "the collision of two
clusters", "a central massive particle"), Newtonian only (the post-Newtonian pair of PAPER.md:351-355 has no equations
in the reference): ``two_cluster_collision`` and ``central_massive_particle``.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

__all__ = [
    "Workload", "plummer", "kroupa_masses", "config", "active_indices",
    "CONFIG_N", "two_body", "random_cluster", "two_cluster_collision", "central_massive_particle",
]

#: particle counts of BASELINE.json configs C1..C5 (C5 has one extra central particle)
CONFIG_N = {1: 1024, 2: 16384, 3: 65536, 4: 262144, 5: 1048576}


@dataclass
class Workload:
    """Initial conditions: masses [n], positions [n,3], velocities [n,3] (float64, C order)."""
    name: str
    m: np.ndarray
    x: np.ndarray
    v: np.ndarray
    eps: float = 1e-4
    eta: float = 0.01
    t_end: float = 0.0
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.m.shape[0])


def _isotropic(rng: np.random.Generator, n: int) -> np.ndarray:
    """n unit vectors, uniform on the sphere (cos(theta) uniform, phi uniform)."""
    c = 1.0 - 2.0 * rng.random(n)
    s = np.sqrt(np.maximum(0.0, 1.0 - c * c))
    phi = 2.0 * math.pi * rng.random(n)
    return np.stack([s * np.cos(phi), s * np.sin(phi), c], axis=1)


def _plummer_speed_fraction(rng: np.random.Generator, n: int) -> np.ndarray:
    """q = v/v_esc by von Neumann rejection on g(q) = q^2 (1-q^2)^(7/2), g_max < 0.1.

    Draws are consumed in fixed-size batches and accepted values are taken in
    draw order, so the result depends only on the seed.
    """
    out = np.empty(n, dtype=np.float64)
    filled = 0
    while filled < n:
        batch = max(1024, 2 * (n - filled))
        q = rng.random(batch)
        y = 0.1 * rng.random(batch)
        ok = q[y < q * q * (1.0 - q * q) ** 3.5]
        take = min(ok.size, n - filled)
        out[filled:filled + take] = ok[:take]
        filled += take
    return out


def plummer(n: int, seed: int, m: np.ndarray | None = None) -> tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Plummer sphere in N-body units; returns (m, x, v).

    ``m`` defaults to equal masses 1/n.  Mass fraction is drawn from (0, 0.999]
    so that the outermost radius stays finite (r_max ~ 38.7 Plummer radii).
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    if m is None:
        m = np.full(n, 1.0 / n, dtype=np.float64)
    m = np.ascontiguousarray(m, dtype=np.float64)
    assert m.shape == (n,)
    frac = 0.999 * (1.0 - rng.random(n))          # (0, 0.999]
    r = 1.0 / np.sqrt(frac ** (-2.0 / 3.0) - 1.0)
    x = r[:, None] * _isotropic(rng, n)
    q = _plummer_speed_fraction(rng, n)
    speed = q * math.sqrt(2.0) * (1.0 + r * r) ** (-0.25)
    v = speed[:, None] * _isotropic(rng, n)
    lscale = 3.0 * math.pi / 16.0
    x *= lscale
    v *= 1.0 / math.sqrt(lscale)
    mtot = m.sum()
    x -= (m[:, None] * x).sum(axis=0) / mtot
    v -= (m[:, None] * v).sum(axis=0) / mtot
    return m, np.ascontiguousarray(x), np.ascontiguousarray(v)


def kroupa_masses(n: int, seed: int, m_lo: float = 0.1, m_br: float = 0.5, m_hi: float = 100.0,
                  a1: float = 1.3, a2: float = 2.3) -> np.ndarray:
    """Two-segment power-law masses dN/dm ~ m^-a1 (m<m_br), ~ m^-a2 (m>=m_br), sum normalised to 1."""
    rng = np.random.Generator(np.random.PCG64(seed))
    # segment weights with continuity at m_br: f1 = m^-a1, f2 = m_br^(a2-a1) m^-a2
    def seg(a, lo, hi):
        return (hi ** (1.0 - a) - lo ** (1.0 - a)) / (1.0 - a)
    w1 = seg(a1, m_lo, m_br)
    w2 = m_br ** (a2 - a1) * seg(a2, m_br, m_hi)
    p1 = w1 / (w1 + w2)
    u = rng.random(n)
    first = u < p1
    t = np.where(first, u / p1, (u - p1) / (1.0 - p1))
    lo = np.where(first, m_lo, m_br)
    hi = np.where(first, m_br, m_hi)
    a = np.where(first, a1, a2)
    m = (lo ** (1.0 - a) + t * (hi ** (1.0 - a) - lo ** (1.0 - a))) ** (1.0 / (1.0 - a))
    return m / m.sum()


def config(k: int, n: int | None = None) -> Workload:
    """BASELINE.json config C<k>.  ``n`` overrides the particle count (for scaled-down tests)."""
    if k not in CONFIG_N:
        raise ValueError(f"unknown config {k}")
    n = CONFIG_N[k] if n is None else int(n)
    if k in (1, 2, 3):
        m, x, v = plummer(n, seed=k)
        t_end = {1: 0.125, 2: 1.0, 3: 0.0}[k]
        return Workload(f"C{k}-plummer-{n}", m, x, v, 1e-4, 0.01, t_end, {"config": k, "seed": k})
    if k == 4:
        m = kroupa_masses(n, seed=40)
        m, x, v = plummer(n, seed=4, m=m)
        return Workload(f"C4-plummer-kroupa-{n}", m, x, v, 1e-4, 0.01, 0.25,
                        {"config": 4, "seed": 4, "mass_seed": 40})
    # k == 5: equal masses 1/n plus a central point mass 0.01 at rest at the origin (index n)
    m, x, v = plummer(n, seed=5)
    m = np.concatenate([m, [0.01]])
    x = np.concatenate([x, np.zeros((1, 3))])
    v = np.concatenate([v, np.zeros((1, 3))])
    return Workload(f"C5-plummer-central-{n}+1", np.ascontiguousarray(m), np.ascontiguousarray(x),
                    np.ascontiguousarray(v), 1e-4, 0.01, 0.0, {"config": 5, "seed": 5})


def active_indices(n: int, n_act: int, seed: int | None = None) -> np.ndarray:
    """C3's active sets: n_act distinct indices drawn uniformly, ascending, int32."""
    if n_act >= n:
        return np.arange(n, dtype=np.int32)
    if seed is None:
        seed = 300 + int(round(math.log2(max(n_act, 1))))
    rng = np.random.Generator(np.random.PCG64(seed))
    return np.sort(rng.choice(n, size=n_act, replace=False)).astype(np.int32)


def two_body(m1: float = 0.5, m2: float = 0.5, sep: float = 1.0, ecc: float = 0.0) -> Workload:
    """Two bodies at apocentre-free start: separation ``sep`` = pericentre distance a(1-e), in the
    centre-of-mass frame, orbit in the x-y plane.  Used for Kepler closed-form pins (eps = 0)."""
    mt = m1 + m2
    a = sep / (1.0 - ecc)
    vrel = math.sqrt(mt * (1.0 + ecc) / (a * (1.0 - ecc)))   # speed at pericentre, G = 1
    x = np.array([[-m2 / mt * sep, 0.0, 0.0], [m1 / mt * sep, 0.0, 0.0]])
    v = np.array([[0.0, -m2 / mt * vrel, 0.0], [0.0, m1 / mt * vrel, 0.0]])
    return Workload(f"two-body-e{ecc}", np.array([m1, m2]), x, v, 0.0, 0.01, 0.0,
                    {"semi_major": a, "ecc": ecc, "period": 2.0 * math.pi * math.sqrt(a ** 3 / mt)})


def random_cluster(n: int, seed: int, eps: float = 1e-4) -> Workload:
    """Small unstructured test input: uniform positions/velocities in a cube, random masses."""
    rng = np.random.Generator(np.random.PCG64(seed))
    m = rng.random(n) + 0.1
    m /= m.sum()
    x = rng.random((n, 3)) * 2.0 - 1.0
    v = (rng.random((n, 3)) * 2.0 - 1.0) * 0.5
    return Workload(f"random-{n}", m, np.ascontiguousarray(x), np.ascontiguousarray(v), eps, 0.01, 0.0,
                    {"seed": seed})


def two_cluster_collision(n: int, seed: int, mass_ratio: float = 1.0, apocentre: float = 3.0, ecc: float = 0.5,
                          eps: float = 1e-4, t_end: float = 0.25) -> Workload:
    """"The collision of two clusters": two Plummer spheres with n1 : n2 = M1 : M2 = mass_ratio : 1
    (equal particle masses, total mass 1), each sampled like C1-C3 and scaled to its own mass at unchanged length
    scale (velocities x sqrt(M_k)), set on a bound Kepler orbit of their centres of mass: they start at the apocentre
    distance ``apocentre`` along x, moving along +-y with the two-body apocentre speed of eccentricity ``ecc``, so that
    point masses would pass at apocentre (1 - ecc) / (1 + ecc) -- inside each other for the defaults.  The centre of
    mass of the whole system is at rest at the origin.  Particles 0 .. n1-1 are cluster 1."""
    n1 = int(round(n * mass_ratio / (1.0 + mass_ratio)))
    n1 = min(max(n1, 1), n - 1)
    n2 = n - n1
    mp = 1.0 / n
    M1, M2 = n1 * mp, n2 * mp
    _, x1, v1 = plummer(n1, seed=seed)
    _, x2, v2 = plummer(n2, seed=seed + 1)
    v1 = v1 * math.sqrt(M1)
    v2 = v2 * math.sqrt(M2)
    # relative orbit of the centres: separation d at apocentre, speed sqrt(M (1 - e) / d), G = M = 1
    d = float(apocentre)
    vrel = math.sqrt((M1 + M2) * (1.0 - ecc) / d)
    x1 = x1 + np.array([-M2 * d, 0.0, 0.0])
    x2 = x2 + np.array([M1 * d, 0.0, 0.0])
    v1 = v1 + np.array([0.0, -M2 * vrel, 0.0])
    v2 = v2 + np.array([0.0, M1 * vrel, 0.0])
    m = np.full(n, mp, dtype=np.float64)
    x = np.ascontiguousarray(np.concatenate([x1, x2]))
    v = np.ascontiguousarray(np.concatenate([v1, v2]))
    return Workload(f"two-clusters-{n1}+{n2}", m, x, v, eps, 0.01, t_end,
                    {"seed": seed, "n1": n1, "n2": n2, "M1": M1, "M2": M2, "apocentre": d, "ecc": ecc, "vrel": vrel,
                     "semi_major": d / (1.0 + ecc)})


def central_massive_particle(n: int, seed: int, m_central: float = 0.05, eps: float = 1e-5, t_end: float = 0.125) -> Workload:
    """"A central massive particle" with a small softening: an equal-mass Plummer sphere of n particles
    and total mass 1 - m_central, scaled from the unit-mass sample at unchanged length scale (velocities x
    sqrt(1 - m_central)), plus ONE particle of mass m_central (index n: m_central n / (1 - m_central) stellar masses) at
    rest at the origin; the centre of mass of the whole system is then put at rest at the origin.  Not an equilibrium:
    the stars inside the heavy particle's sphere of influence fall towards it, and it wanders -- it takes part in the
    dynamics, unlike the 0.01 point mass of the throughput config C5."""
    _, x, v = plummer(n, seed=seed)
    ms = (1.0 - m_central) / n
    v = v * math.sqrt(1.0 - m_central)
    m = np.concatenate([np.full(n, ms), [m_central]])
    x = np.concatenate([x, np.zeros((1, 3))])
    v = np.concatenate([v, np.zeros((1, 3))])
    x = x - (m[:, None] * x).sum(axis=0) / m.sum()
    v = v - (m[:, None] * v).sum(axis=0) / m.sum()
    return Workload(f"central-massive-{n}+1", np.ascontiguousarray(m), np.ascontiguousarray(x), np.ascontiguousarray(v),
                    eps, 0.01, t_end, {"seed": seed, "m_central": m_central, "m_star": ms})
