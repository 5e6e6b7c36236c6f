"""Pins for the oracle's Kepler drift (O9): closed forms, invariants, an independent
absolute-anomaly propagation and scipy's DOP853.  CPU only."""
import numpy as np
import pytest
from scipy.integrate import solve_ivp

import oracle
from paper_2309_08217_b200.workloads import elements_to_cartesian


def two_body_dop853(mu, x0, v0, t):
    f = lambda _, y: np.concatenate([y[3:], -mu * y[:3] / np.linalg.norm(y[:3]) ** 3])
    sol = solve_ivp(f, (0.0, t), np.concatenate([x0, v0]), method="DOP853", rtol=1e-13, atol=1e-15)
    return sol.y[:3, -1], sol.y[3:, -1]


def test_circular_orbit_turns_by_n_dt():
    mu, a = 0.8, 1.3
    n = np.sqrt(mu / a ** 3)
    x0, v0 = np.array([a, 0.0, 0.0]), np.array([0.0, a * n, 0.0])
    for dt in (0.01, 0.7, 3.3, -2.1, 40.0):
        x, v = oracle.kepler_drift_one(mu, dt, x0, v0)
        th = n * dt
        assert np.allclose(x, [a * np.cos(th), a * np.sin(th), 0], rtol=0, atol=4e-15 * a * max(1, abs(th)))
        assert np.allclose(v, [-a * n * np.sin(th), a * n * np.cos(th), 0], rtol=0, atol=4e-15 * a * n * max(1, abs(th)))


def test_two_body_circular_orbit_returns_after_one_period():
    # north_star: "a two-body circular orbit propagated by the Kepler drift"
    mu, a = 0.01720209895 ** 2, 1.0
    P = 2 * np.pi * np.sqrt(a ** 3 / mu)
    x0, v0 = np.array([a, 0.0, 0.0]), np.array([0.0, np.sqrt(mu / a), 0.0])
    x, v = x0, v0
    for _ in range(60):                                    # 60 drifts of P/60 (about 6.09 days each)
        x, v = oracle.kepler_drift_one(mu, P / 60, x, v)
    assert np.abs(x - x0).max() < 1e-13 and np.abs(v - v0).max() < 1e-13 * np.sqrt(mu)
    x, v = oracle.kepler_drift_one(mu, P, x0, v0)
    assert np.abs(x - x0).max() < 1e-14


@pytest.mark.parametrize("e", [0.0, 0.3, 0.9])
def test_against_absolute_kepler_equation(e):
    # independent route: elements at two mean anomalies through the textbook E - e sin E = M solution
    mu, a = 1.0, 1.7
    n = np.sqrt(mu / a ** 3)
    M0 = 0.4
    x0, v0 = elements_to_cartesian(mu, a, e, 0.3, 1.1, 2.2, M0)
    x, v = x0.copy(), v0.copy()
    steps, dt = (10000, 0.05) if e == 0.9 else (200, 0.37)
    for _ in range(steps):
        x, v = oracle.kepler_drift_one(mu, dt, x, v)
    xe, ve = elements_to_cartesian(mu, a, e, 0.3, 1.1, 2.2, M0 + n * steps * dt)
    tol = 2e-10 if e == 0.9 else 1e-12
    assert np.abs(x - xe).max() < tol * a and np.abs(v - ve).max() < tol * np.sqrt(mu / a) / (1 - e)
    # one big multi-revolution drift lands on the same point
    xb, vb = oracle.kepler_drift_one(mu, steps * dt, x0, v0)
    assert np.abs(xb - xe).max() < tol * a


def test_against_dop853_elliptic_and_hyperbolic():
    rng = np.random.default_rng(2)
    mu = 1.0
    for trial in range(6):
        x0 = rng.normal(size=3)
        vdir = rng.normal(size=3)
        vesc = np.sqrt(2 * mu / np.linalg.norm(x0))
        speed = vesc * (0.6 if trial < 3 else 1.4)          # bound, then unbound
        v0 = vdir / np.linalg.norm(vdir) * speed
        for dt in (0.8, -1.3):
            x, v = oracle.kepler_drift_one(mu, dt, x0, v0)
            xr, vr = two_body_dop853(mu, x0, v0, dt)
            assert np.abs(x - xr).max() < 2e-11 and np.abs(v - vr).max() < 2e-11


def test_parabolic_orbit():
    mu = 1.0
    x0 = np.array([2.0, 0.0, 0.0])
    v0 = np.array([0.0, 1.0, 0.0])                         # exactly escape speed: alpha = 2 mu/r - v^2 = 0
    assert 2 * mu / 2.0 - v0 @ v0 == 0.0
    x, v = oracle.kepler_drift_one(mu, 1.5, x0, v0)
    xr, vr = two_body_dop853(mu, x0, v0, 1.5)
    assert np.abs(x - xr).max() < 2e-11 and np.abs(v - vr).max() < 2e-11


def test_invariants_and_reversibility():
    rng = np.random.default_rng(5)
    mu = 0.01720209895 ** 2
    n = 500
    a = rng.uniform(0.5, 4, n); e = rng.uniform(0, 0.7, n)
    x0, v0 = elements_to_cartesian(mu, a, e, rng.uniform(0, 0.5, n), *(rng.uniform(0, 6.28, (3, n))))
    p = oracle.Params(G=mu, M_star=1.0)
    x1, v1 = oracle.drift(x0, v0, p, 6.0)
    en = lambda x, v: 0.5 * (v ** 2).sum(1) - mu / np.linalg.norm(x, axis=1)
    assert np.abs(en(x1, v1) / en(x0, v0) - 1).max() < 2e-14
    h0, h1 = np.cross(x0, v0), np.cross(x1, v1)
    assert np.abs(h1 - h0).max() < 4e-15 * np.abs(h0).max()
    xb, vb = oracle.drift(x1, v1, p, -6.0)
    assert np.abs(xb - x0).max() < 1e-13 and np.abs(vb - v0).max() < 1e-13 * np.abs(v0).max()
    # drift(dt1) o drift(dt2) = drift(dt1 + dt2)
    x2, v2 = oracle.drift(*oracle.drift(x0, v0, p, 2.5), p, 3.5)
    assert np.abs(x2 - x1).max() < 1e-13
