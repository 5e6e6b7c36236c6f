"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is shared by the oracle tests, the GPU parity tests and ``bench.py``.  It holds NONE
of the method's arithmetic (no kick, no changeover, no drift, no r_crit): it only draws orbital
elements from a counter-based PRNG and converts them to heliocentric Cartesian states with the
textbook two-body formulae.  It imports neither ``oracle`` nor the CUDA binding.

The paper's own initial conditions (size-distributed planetesimal annuli, the
Nesvorny & Morbidelli five-planet set-up, the Woo et al. gas runs) are not in the container; these
configs take their shapes and sizes and stand in for them.

Recipe: SplitMix64 seeded ``0x2309082170 + cfg`` (sweep: ``+ 16*log2 N``); uniforms are
``(u64 >> 11) * 2**-53``; Rayleigh by inverse CDF ``sigma*sqrt(-2 ln(1-u))``; six uniforms per body
in the fixed order (a, e, i, Omega, omega, M), bodies in generation order.  Embryo masses (config 2)
come from a second stream seeded ``seed ^ 0x5EED``.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

K_GAUSS = 0.01720209895                 # Gaussian gravitational constant; G = k^2 [AU^3 Msun^-1 day^-2]
G_DEFAULT = K_GAUSS * K_GAUSS
M_EARTH = 1.0 / 332946.0487             # Msun
YEAR = 365.25                           # days
SEED0 = 0x2309082170

PAIR_MAX = 0
PAIR_MUTUAL_HILL = 1


def splitmix64(seed: int, n: int) -> np.ndarray:
    """First n outputs of SplitMix64 started at ``seed`` (vectorised: output k uses state seed + (k+1)*gamma)."""
    gamma = np.uint64(0x9E3779B97F4A7C15)
    with np.errstate(over="ignore"):
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + gamma * np.arange(1, n + 1, dtype=np.uint64)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def uniforms(seed: int, n: int) -> np.ndarray:
    """n doubles in [0, 1) with 53 random bits each."""
    return (splitmix64(seed, n) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def rayleigh(u: np.ndarray, sigma: float) -> np.ndarray:
    return sigma * np.sqrt(-2.0 * np.log1p(-u))


def solve_kepler_equation(M: np.ndarray, e: np.ndarray) -> np.ndarray:
    """Eccentric anomaly from E - e sin E = M (Newton, to 1e-15), elementwise."""
    E = M + e * np.sin(M)
    for _ in range(60):
        dE = (E - e * np.sin(E) - M) / (1.0 - e * np.cos(E))
        E = E - dE
        if np.max(np.abs(dE)) < 1e-15:
            break
    return E


def elements_to_cartesian(mu, a, e, inc, Omega, omega, M):
    """Heliocentric position and velocity from Keplerian elements (mu = G (M_star + m_i))."""
    mu, a, e, inc, Omega, omega, M = np.broadcast_arrays(*(np.asarray(q, dtype=np.float64)
                                                           for q in (mu, a, e, inc, Omega, omega, M)))
    E = solve_kepler_equation(M, e)
    cE, sE = np.cos(E), np.sin(E)
    b = np.sqrt(1.0 - e * e)
    n = np.sqrt(mu / a ** 3)
    xp = a * (cE - e)
    yp = a * b * sE
    d = 1.0 - e * cE
    vxp = -a * n * sE / d
    vyp = a * n * b * cE / d
    cO, sO = np.cos(Omega), np.sin(Omega)
    co, so = np.cos(omega), np.sin(omega)
    ci, si = np.cos(inc), np.sin(inc)
    # columns of Rz(Omega) Rx(i) Rz(omega)
    px = cO * co - sO * so * ci
    py = sO * co + cO * so * ci
    pz = so * si
    qx = -cO * so - sO * co * ci
    qy = -sO * so + cO * co * ci
    qz = co * si
    x = np.stack([px * xp + qx * yp, py * xp + qy * yp, pz * xp + qz * yp], axis=-1)
    v = np.stack([px * vxp + qx * vyp, py * vxp + qy * vyp, pz * vxp + qz * vyp], axis=-1)
    return np.ascontiguousarray(x), np.ascontiguousarray(v)


@dataclass
class Workload:
    """One synthetic problem.  ``v`` is HELIOCENTRIC (pass ``v_is_heliocentric=1`` to create)."""
    name: str
    cfg: int
    m: np.ndarray                  # [N]     Msun
    x: np.ndarray                  # [N, 3]  AU, heliocentric
    v: np.ndarray                  # [N, 3]  AU/day, heliocentric
    dt: float                      # days
    nsteps: int
    G: float = G_DEFAULT
    M_star: float = 1.0
    n1: float = 3.0
    n2: float = 0.0                # BASELINE.json configs: "r_crit = 3 mutual Hill radii"
    pair_rule: int = PAIR_MUTUAL_HILL
    seed: int = 0
    notes: dict = field(default_factory=dict)

    @property
    def N(self) -> int:
        return int(self.m.shape[0])


def _disc(seed, n, a_lo, a_hi, sig_e, sig_i, m, G=G_DEFAULT, M_star=1.0):
    u = uniforms(seed, 6 * n).reshape(n, 6)
    a = a_lo + (a_hi - a_lo) * u[:, 0]
    e = rayleigh(u[:, 1], sig_e)
    inc = rayleigh(u[:, 2], sig_i)
    two_pi = 2.0 * np.pi
    x, v = elements_to_cartesian(G * (M_star + m), a, e, inc, two_pi * u[:, 3], two_pi * u[:, 4], two_pi * u[:, 5])
    return x, v


def planetesimal_disc(n: int, total_mass_earth: float, seed: int, cfg: int, name: str,
                      dt: float = 6.0, nsteps: int = 10, a_lo: float = 0.5, a_hi: float = 4.0) -> Workload:
    m = np.full(n, total_mass_earth * M_EARTH / max(n, 1))
    x, v = _disc(seed, n, a_lo, a_hi, 0.01, 0.005, m)
    return Workload(name=name, cfg=cfg, m=m, x=x, v=v, dt=dt, nsteps=nsteps, seed=seed)


def config(cfg: int, n_override: int | None = None) -> Workload:
    """The BASELINE.json config ``cfg`` (0..4).  ``n_override`` rescales the planetesimal count
    (used by the config-4 N sweep and by reduced-size tests); the total disc mass is kept."""
    seed = SEED0 + cfg
    if cfg == 0:
        n = n_override or 2048
        return planetesimal_disc(n, 2.5, seed, 0, "c0_tiny_disc", 6.0, 10)
    if cfg == 1:
        n = n_override or 6600
        return planetesimal_disc(n, 5.0, seed, 1, "c1_statistical", 6.0, 2000)
    if cfg == 2:
        n_emb, n_pl = 100, (n_override or 8000)
        um = uniforms(seed ^ 0x5EED, n_emb)
        m_emb = 0.01 * M_EARTH * (10.0 ** um)                      # log-uniform 0.01..0.1 M_earth
        m_pl = np.full(n_pl, 2.0 * M_EARTH / n_pl)
        m = np.concatenate([m_emb, m_pl])
        x, v = _disc(seed, n_emb + n_pl, 0.7, 3.0, 0.01, 0.005, m)
        return Workload("c2_embryos", 2, m, x, v, 6.0, 1000, seed=seed)
    if cfg == 3:
        n_pl = n_override or 10000
        m_g = np.array([318.0, 95.0, 14.5, 17.0]) * M_EARTH
        a_g = np.array([5.5, 8.2, 11.5, 14.2])
        m_pl = np.full(n_pl, 35.0 * M_EARTH / n_pl)
        m = np.concatenate([m_g, m_pl])
        u = uniforms(seed, 6 * (4 + n_pl)).reshape(4 + n_pl, 6)
        two_pi = 2.0 * np.pi
        a = np.concatenate([a_g, 15.5 + (30.0 - 15.5) * u[4:, 0]])
        e = np.concatenate([np.zeros(4), rayleigh(u[4:, 1], 0.001)])
        inc = np.concatenate([np.zeros(4), rayleigh(u[4:, 2], 0.001)])
        Om = np.concatenate([np.zeros(4), two_pi * u[4:, 3]])
        om = np.concatenate([np.zeros(4), two_pi * u[4:, 4]])
        M = two_pi * u[:, 5]
        x, v = elements_to_cartesian(G_DEFAULT * (1.0 + m), a, e, inc, Om, om, M)
        return Workload("c3_giants_disc", 3, m, x, v, 0.5 * YEAR, 500, seed=seed)
    if cfg == 4:
        n = n_override or 40000
        if n_override is not None and n_override > 0 and (n_override & (n_override - 1)) == 0:
            seed = SEED0 + 4 + 16 * int(np.log2(n_override))          # sweep seeds
        return planetesimal_disc(n, 5.0, seed, 4, "c4_performance" if n_override is None else f"c4_sweep_N{n}",
                                 6.0, 200)
    raise ValueError(f"unknown config {cfg}")


SWEEP_N = [2 ** k for k in range(10, 18)]
