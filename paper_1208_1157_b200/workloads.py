"""Seeded synthetic ensembles shaped like the paper's workloads (BASELINE.json ``configs`` 0-4; §5.1).

This module holds NO arithmetic of the method (no force law, no integrator, no energy): it only draws
orbital elements from a counter-based generator and converts them to Cartesian initial conditions with
numpy.  It is the one module both the CUDA path's callers (tests, bench.py) and the oracle's callers
use, so that both sides read the same arrays.  Recipe: G = 1, star m0 = 1 at the
heliocentric origin at rest; each planet from (a, e, i, Omega, omega, M) -> E - e sin E = M ->
heliocentric Cartesian with mu = G (m0 + m_k) -> subtract centre-of-mass position and velocity.

Random numbers: u(seed, system, draw) = top 53 bits of a splitmix64-style hash of the three counters, so
any subset of systems [offset, offset + n_sys) is reproducible on its own.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

HERMITE, MVS = 0, 1
_DRAWS_PER_BODY = 16  # slots 0..6: m, a, e, i, Omega, omega, M; 8..15: resamples of e


def _mix(z: np.ndarray) -> np.ndarray:
    z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
    z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    return z ^ (z >> np.uint64(31))


def uniform(seed: int, system: np.ndarray, draw: int) -> np.ndarray:
    """U[0,1) with 53 random bits, a pure function of (seed, system index, draw index)."""
    with np.errstate(over="ignore"):
        s = np.asarray(system, dtype=np.uint64)
        k = _mix(np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + np.uint64(0x9E3779B97F4A7C15))
        z = _mix(k ^ _mix(s + np.uint64(0xD1B54A32D192ED03)))
        z = _mix(z ^ _mix(np.uint64(draw) * np.uint64(0x8CB92BA72F3D8DD7) + np.uint64(1)))
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def _rayleigh(seed, system, body, sigma):
    """Rayleigh(sigma) = sigma sqrt(-2 ln(1-U)); resample (next draw slot) while >= 0.9."""
    base = body * _DRAWS_PER_BODY
    e = sigma * np.sqrt(-2.0 * np.log1p(-uniform(seed, system, base + 2)))
    for k in range(8, 16):
        bad = e >= 0.9
        if not bad.any():
            break
        e = np.where(bad, sigma * np.sqrt(-2.0 * np.log1p(-uniform(seed, system, base + k))), e)
    return np.minimum(e, 0.9 - 1e-9)


def _solve_kepler(M, e):
    E = M + e * np.sin(M)
    for _ in range(60):
        dE = (E - e * np.sin(E) - M) / (1.0 - e * np.cos(E))
        E = E - dE
        if np.max(np.abs(dE)) < 1e-15:
            break
    return E


def elements_to_cartesian(a, e, inc, Omega, omega, M, mu):
    """Heliocentric position and velocity [..., 3] from Keplerian elements (elliptic)."""
    E = _solve_kepler(M, e)
    cE, sE = np.cos(E), np.sin(E)
    b = np.sqrt(1.0 - e * e)
    n = np.sqrt(mu / (a * a * a))
    xp, yp = a * (cE - e), a * b * sE
    den = 1.0 - e * cE
    vxp, vyp = -a * n * sE / den, a * n * b * cE / den
    cO, sO, co, so, ci, si = np.cos(Omega), np.sin(Omega), np.cos(omega), np.sin(omega), np.cos(inc), np.sin(inc)
    r11, r12 = cO * co - sO * so * ci, -cO * so - sO * co * ci
    r21, r22 = sO * co + cO * so * ci, -sO * so + cO * co * ci
    r31, r32 = so * si, co * si
    pos = np.stack([r11 * xp + r12 * yp, r21 * xp + r22 * yp, r31 * xp + r32 * yp], axis=-1)
    vel = np.stack([r11 * vxp + r12 * vyp, r21 * vxp + r22 * vyp, r31 * vxp + r32 * vyp], axis=-1)
    return pos, vel


@dataclass(frozen=True)
class Config:
    cfg: int
    integrator: int
    n_sys: int
    n_body: int
    dt: float
    steps: int
    r_close: float  # <= 0 disables
    r_eject: float  # inf disables
    seed: int
    name: str


CONFIGS = {
    0: Config(0, HERMITE, 1024, 3, 0.01, 2000, 0.0, math.inf, 0x5EED0000, "hermite_1024x3"),
    1: Config(1, HERMITE, 131072, 3, 0.01, 10000, 0.01, 100.0, 0x5EED0001, "hermite_131072x3"),
    2: Config(2, HERMITE, 32768, 6, 0.005, 10000, 0.01, 100.0, 0x5EED0002, "hermite_32768x6"),
    3: Config(3, HERMITE, 8192, 15, 0.002, 5000, 0.01, 100.0, 0x5EED0003, "hermite_8192x15"),
    4: Config(4, MVS, 131072, 4, 0.05, 10000, 0.0, math.inf, 0x5EED0004, "mvs_131072x4"),
}


def _planet_chain(seed, sysidx, n_pl, a1_lo, a1_hi, ratio_lo, ratio_hi, sig_e, sig_i, first_body=1):
    """n_pl planets: m log-U[1e-5,1e-3]; a_1 ~ U[a1_lo,a1_hi], a_{k+1} = a_k U[ratio_lo,ratio_hi]."""
    out = []
    a_prev = None
    for k in range(n_pl):
        body = first_body + k
        base = body * _DRAWS_PER_BODY
        m = 10.0 ** (-5.0 + 2.0 * uniform(seed, sysidx, base + 0))
        ua = uniform(seed, sysidx, base + 1)
        a = (a1_lo + (a1_hi - a1_lo) * ua) if a_prev is None else a_prev * (ratio_lo + (ratio_hi - ratio_lo) * ua)
        a_prev = a
        e = _rayleigh(seed, sysidx, body, sig_e)
        inc = sig_i * np.sqrt(-2.0 * np.log1p(-uniform(seed, sysidx, base + 3)))
        Om, om, M = (2.0 * math.pi * uniform(seed, sysidx, base + s) for s in (4, 5, 6))
        out.append((m, a, e, inc, Om, om, M))
    return out


def _planetesimals(seed, sysidx, n_p, first_body):
    out = []
    for k in range(n_p):
        body = first_body + k
        base = body * _DRAWS_PER_BODY
        m = 10.0 ** (-8.0 + 2.0 * uniform(seed, sysidx, base + 0))
        a = 0.5 + 4.5 * uniform(seed, sysidx, base + 1)
        e = _rayleigh(seed, sysidx, body, 0.05)
        inc = 0.05 * np.sqrt(-2.0 * np.log1p(-uniform(seed, sysidx, base + 3)))
        Om, om, M = (2.0 * math.pi * uniform(seed, sysidx, base + s) for s in (4, 5, 6))
        out.append((m, a, e, inc, Om, om, M))
    return out


def generate(cfg: int, n_sys: int | None = None, offset: int = 0, seed: int | None = None):
    """Initial conditions of systems [offset, offset + n_sys) of BASELINE.json config ``cfg``.

    Returns (pos [n_sys][n_body][3], vel, mass [n_sys][n_body]) as float64 C-order arrays, barycentric.
    """
    c = CONFIGS[cfg]
    n_sys = c.n_sys if n_sys is None else int(n_sys)
    seed = c.seed if seed is None else seed
    sysidx = np.arange(offset, offset + n_sys, dtype=np.uint64)
    if cfg in (0, 1):
        bodies = _planet_chain(seed, sysidx, 2, 0.8, 1.2, 1.6, 2.4, 0.02, 0.01)
    elif cfg == 2:
        bodies = _planet_chain(seed, sysidx, 5, 0.5, 1.0, 1.4, 1.8, 0.03, 0.02)
    elif cfg == 3:
        bodies = _planet_chain(seed, sysidx, 4, 0.5, 1.0, 1.4, 1.8, 0.03, 0.02) + _planetesimals(seed, sysidx, 10, 5)
    elif cfg == 4:
        bodies = _planet_chain(seed, sysidx, 3, 0.5, 1.0, 1.4, 1.8, 0.03, 0.02)
    else:
        raise KeyError(cfg)
    n_body = 1 + len(bodies)
    assert n_body == c.n_body
    pos = np.zeros((n_sys, n_body, 3))
    vel = np.zeros((n_sys, n_body, 3))
    mass = np.ones((n_sys, n_body))
    for b, (m, a, e, inc, Om, om, M) in enumerate(bodies, start=1):
        mass[:, b] = m
        pos[:, b], vel[:, b] = elements_to_cartesian(a, e, inc, Om, om, M, 1.0 + m)
    mt = mass.sum(axis=1)[:, None]
    pos -= ((mass[:, :, None] * pos).sum(axis=1) / mt)[:, None, :]
    vel -= ((mass[:, :, None] * vel).sum(axis=1) / mt)[:, None, :]
    return np.ascontiguousarray(pos), np.ascontiguousarray(vel), np.ascontiguousarray(mass)


def paper_ics(n_body: int, n_sys: int = 1, planet_mass: float = 1e-3, alpha: float = 0.4):
    """The paper's own test systems (§5.1): m0 = 1 at rest at the origin, equal-mass planets on
    circular coplanar orbits a_i = (1+alpha)^(i-1), speed sqrt(G m0 / a_i) (reading R15), all at phase 0."""
    pos = np.zeros((n_sys, n_body, 3))
    vel = np.zeros((n_sys, n_body, 3))
    mass = np.full((n_sys, n_body), planet_mass)
    mass[:, 0] = 1.0
    for i in range(1, n_body):
        a = (1.0 + alpha) ** (i - 1)
        pos[:, i, 0] = a
        vel[:, i, 1] = math.sqrt(1.0 / a)
    return pos, vel, mass
