"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module only *draws inputs*.  It holds none of the method's arithmetic (no accelerations,
no gradient term, no time-steps, no integrator) and imports neither ``oracle`` nor the CUDA
package.  Every generator is a pure function of its arguments: random numbers come from numpy's
counter-based Philox bit generator keyed by ``seed``, so the same call gives the same bits in the
oracle process and in the GPU process.

Workload recipes (stand-ins for the paper's McLuster/SSE clusters,
PAPER.md:680, 984-1005, which are not available offline):

* ``plummer``       -- Plummer sphere in Henon units (G = M = 1, a = 3*pi/16), equal masses,
                       positions from the inverted cumulative mass profile Eq. (A2), speeds by
                       rejection from q^2 (1-q^2)^{7/2} (from f(E) ~ E^{7/2}, Eq. A4).
* ``active_subset`` -- config 4's random sorted active index set.
* ``star_cluster``  -- config 5: Kroupa-like two-segment IMF, central point mass, hard binaries.
* ``kepler_binary`` / ``solar_system`` -- small analytic systems for the oracle pins.

Layout convention (same as include/frost.h): positions and velocities are C-contiguous float64
arrays of shape (3, ld) -- three SoA planes -- with ld == n here.
"""
from __future__ import annotations

import math
import os
from typing import Tuple

import numpy as np

PLUMMER_A = 3.0 * math.pi / 16.0  # Henon units: virial radius 1  <=>  a = 3 pi / 16


def _rng(seed: int, stream: int = 0) -> np.random.Generator:
    """Counter-based generator: one independent Philox stream per (seed, stream)."""
    return np.random.Generator(np.random.Philox(key=[int(seed) & 0xFFFFFFFFFFFFFFFF, int(stream)]))


def _isotropic(rng: np.random.Generator, n: int) -> np.ndarray:
    """n unit vectors, uniform on the sphere, shape (3, n)."""
    cz = rng.uniform(-1.0, 1.0, n)
    ph = rng.uniform(0.0, 2.0 * math.pi, n)
    s = np.sqrt(np.maximum(0.0, 1.0 - cz * cz))
    return np.stack([s * np.cos(ph), s * np.sin(ph), cz])


def _plummer_xv(rng: np.random.Generator, n: int, a: float = PLUMMER_A, G: float = 1.0,
                M: float = 1.0) -> Tuple[np.ndarray, np.ndarray]:
    """Positions and velocities of n stars drawn from the Plummer DF (not yet centred)."""
    # radius: invert M(r)/M = (1 + a^2/r^2)^{-3/2} = X  (Eq. A2); X <= 0.999
    X = rng.uniform(0.0, 0.999, n)
    X = np.maximum(X, 1e-12)
    r = a / np.sqrt(X ** (-2.0 / 3.0) - 1.0)
    pos = _isotropic(rng, n) * r
    # speed: v = q * v_esc, q ~ q^2 (1 - q^2)^{7/2} on [0,1] by rejection (max of g is < 0.1)
    q = np.empty(n)
    todo = np.arange(n)
    while todo.size:
        q1 = rng.uniform(0.0, 1.0, todo.size)
        y = rng.uniform(0.0, 0.1, todo.size)
        ok = y < q1 * q1 * (1.0 - q1 * q1) ** 3.5
        q[todo[ok]] = q1[ok]
        todo = todo[~ok]
    vesc = np.sqrt(2.0 * G * M / np.sqrt(r * r + a * a))  # from phi(r), Eq. A1
    vel = _isotropic(rng, n) * (q * vesc)
    return pos, vel


def _recentre(pos: np.ndarray, vel: np.ndarray, mass: np.ndarray) -> None:
    mt = mass.sum()
    pos -= (pos * mass).sum(axis=1, keepdims=True) / mt
    vel -= (vel * mass).sum(axis=1, keepdims=True) / mt


def plummer(n: int, seed: int) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Equal-mass Plummer sphere (configs 1-4).  Returns pos(3,n), vel(3,n), mass(n)."""
    rng = _rng(seed)
    pos, vel = _plummer_xv(rng, n)
    mass = np.full(n, 1.0 / n)
    _recentre(pos, vel, mass)
    return np.ascontiguousarray(pos), np.ascontiguousarray(vel), mass


def active_subset(n: int, fraction: float, seed: int) -> np.ndarray:
    """Config 4: round(fraction*n) distinct uniformly random indices, sorted, int32."""
    k = int(round(fraction * n))
    rng = _rng(seed, stream=1)
    idx = rng.choice(n, size=k, replace=False)
    return np.sort(idx).astype(np.int32)


def _kroupa_masses(rng: np.random.Generator, n: int, m_lo=0.08, m_br=0.5, m_hi=100.0,
                   a1=1.3, a2=2.3) -> np.ndarray:
    """Two-segment power law dN/dm ~ m^-a1 on [m_lo,m_br], ~ m^-a2 on [m_br,m_hi], continuous."""
    def seg(alpha, lo, hi):
        return (hi ** (1 - alpha) - lo ** (1 - alpha)) / (1 - alpha)
    k2 = m_br ** (a2 - a1)  # continuity at the break
    w1, w2 = seg(a1, m_lo, m_br), k2 * seg(a2, m_br, m_hi)
    u = rng.uniform(0.0, 1.0, n)
    first = u < w1 / (w1 + w2)
    m = np.empty(n)
    u1 = u[first] * (w1 + w2) / w1
    m[first] = (m_lo ** (1 - a1) + u1 * (m_br ** (1 - a1) - m_lo ** (1 - a1))) ** (1 / (1 - a1))
    u2 = (u[~first] * (w1 + w2) - w1) / w2
    m[~first] = (m_br ** (1 - a2) + u2 * (m_hi ** (1 - a2) - m_br ** (1 - a2))) ** (1 / (1 - a2))
    return m


def _solve_kepler(M: np.ndarray, e: np.ndarray) -> np.ndarray:
    """Eccentric anomaly from mean anomaly (Newton iterations; input construction only)."""
    E = np.where(e < 0.8, M, np.pi * np.ones_like(M))
    for _ in range(60):
        f = E - e * np.sin(E) - M
        E = E - f / (1.0 - e * np.cos(E))
    return E


def _orbit_relative(rng, mtot, a, e, G=1.0):
    """Relative position/velocity (3,k) of k two-body orbits: random phase and orientation."""
    k = a.size
    Mano = rng.uniform(0.0, 2.0 * math.pi, k)
    E = _solve_kepler(Mano, e)
    cosE, sinE = np.cos(E), np.sin(E)
    b = np.sqrt(1.0 - e * e)
    xp = a * (cosE - e)
    yp = a * b * sinE
    nmean = np.sqrt(G * mtot / a ** 3)
    rr = a * (1.0 - e * cosE)
    vxp = -a * a * nmean * sinE / rr
    vyp = a * a * nmean * b * cosE / rr
    # random orthonormal frame (p, q): p isotropic, q perpendicular
    p = _isotropic(rng, k)
    t = _isotropic(rng, k)
    qv = np.cross(p.T, t.T).T
    qv /= np.linalg.norm(qv, axis=0, keepdims=True)
    return p * xp + qv * yp, p * vxp + qv * vyp


def star_cluster(n: int, seed: int, binary_fraction: float = 0.05, central_mass: float = 0.01,
                 a_lo: float = 1e-5, a_hi: float = 1e-3, e_max: float = 0.99):
    """Config 5 (stand-in for PAPER.md:680-684 with primordial binaries added as a stress test).

    Index 0 is a point mass ``central_mass`` at rest at the origin; the other n-1 stars share
    1-central_mass with Kroupa-like masses (0.08-100 before normalisation), Plummer x and v;
    floor(binary_fraction*n/2) disjoint random pairs become binaries with log-uniform semi-major
    axis in [a_lo,a_hi], thermal eccentricities (capped at e_max; config 5: 0.99) and random
    phase; the pair's centre of mass takes the primary's Plummer phase-space point.  Returns pos(3,n), vel(3,n), mass(n),
    pairs(k,2) int32.
    """
    rng = _rng(seed)
    ns = n - 1
    m = _kroupa_masses(rng, ns)
    m *= (1.0 - central_mass) / m.sum()
    pos_s, vel_s = _plummer_xv(rng, ns)
    nb = int(binary_fraction * n / 2.0)
    perm = rng.permutation(ns)[: 2 * nb].reshape(nb, 2)
    if nb:
        i1, i2 = perm[:, 0], perm[:, 1]
        mt = m[i1] + m[i2]
        sma = np.exp(rng.uniform(math.log(a_lo), math.log(a_hi), nb))
        ecc = np.sqrt(rng.uniform(0.0, 1.0, nb))
        ecc = np.minimum(ecc, e_max)
        xr, vr = _orbit_relative(rng, mt, sma, ecc)
        xc, vc = pos_s[:, i1].copy(), vel_s[:, i1].copy()
        pos_s[:, i1] = xc - xr * (m[i2] / mt)
        vel_s[:, i1] = vc - vr * (m[i2] / mt)
        pos_s[:, i2] = xc + xr * (m[i1] / mt)
        vel_s[:, i2] = vc + vr * (m[i1] / mt)
    pos = np.concatenate([np.zeros((3, 1)), pos_s], axis=1)
    vel = np.concatenate([np.zeros((3, 1)), vel_s], axis=1)
    mass = np.concatenate([[central_mass], m])
    # recentre the stars only, so that the central mass stays at the origin at rest
    ms = mass[1:]
    pos[:, 1:] -= (pos[:, 1:] * ms).sum(axis=1, keepdims=True) / ms.sum()
    vel[:, 1:] -= (vel[:, 1:] * ms).sum(axis=1, keepdims=True) / ms.sum()
    return (np.ascontiguousarray(pos), np.ascontiguousarray(vel), mass,
            (perm + 1).astype(np.int32))


def kepler_binary(m1: float, m2: float, a: float, e: float, G: float = 1.0):
    """Two bodies at apocentre on the x axis, orbit in the xy plane, COM at rest at the origin.

    Returns pos(3,2), vel(3,2), mass(2), period.  (PAPER.md:644 uses m1=m2, a=10 AU.)
    """
    mt = m1 + m2
    r = a * (1.0 + e)
    v = math.sqrt(G * mt * (1.0 - e) / (a * (1.0 + e)))
    pos = np.zeros((3, 2))
    vel = np.zeros((3, 2))
    pos[0, 0], pos[0, 1] = -r * m2 / mt, r * m1 / mt
    vel[1, 0], vel[1, 1] = -v * m2 / mt, v * m1 / mt
    period = 2.0 * math.pi * math.sqrt(a ** 3 / (G * mt))
    return pos, vel, np.array([m1, m2], dtype=np.float64), period


GAUSS_K = 0.01720209895  # Gaussian gravitational constant; G = k^2 in AU^3 / (Msun day^2)


def solar_system(path: str | None = None):
    """Sun + four giant planets from tests/golden/solar_system_tables_A1_A2.txt
    (Tables A1/A2).  Returns pos(3,5) [AU], vel(3,5) [AU/day], mass(5) [Msun],
    G = k^2 (reading 18: the paper prints no G)."""
    if path is None:
        path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "..", "tests", "golden",
                            "solar_system_tables_A1_A2.txt")
    rows = [ln.split() for ln in open(path) if ln.strip() and not ln.startswith("#")]
    mass = np.array([float(r[1]) for r in rows])
    pos = np.array([[float(v) for v in r[2:5]] for r in rows]).T.copy()
    vel = np.array([[float(v) for v in r[5:8]] for r in rows]).T.copy()
    return pos, vel, mass, GAUSS_K ** 2
