"""Pins of the oracle's hybrid step with the encounter complement (NEXT-1 of SURVEY.md 8(f); DESIGN.md
reading R11).  Not built on the GPU yet: these pin the oracle that the next round's kernels will be gated on."""
import numpy as np
import pytest
from scipy.integrate import solve_ivp

import oracle
from paper_2309_08217_b200 import workloads as W

G = W.G_DEFAULT


def encounter_system():
    """Star + two planets of 3e-5 Msun on nearly equal orbits, set up so that they pass each other inside
    0.5 r_crit within a few steps, plus two distant spectators."""
    m = np.array([3e-5, 3e-5, 1e-6, 1e-6])
    a = np.array([1.0, 1.012, 1.7, 2.6])
    lam = np.array([0.0, -0.035, 2.0, 4.0])
    x = np.stack([a * np.cos(lam), a * np.sin(lam), 0.002 * np.array([1, -1, 2, -2.0])], axis=1)
    vk = np.sqrt(G * (1 + m) / a)
    v = np.stack([-vk * np.sin(lam), vk * np.cos(lam), np.zeros(4)], axis=1)
    return m, x, oracle.to_democratic(m, v, 1.0)


def full_energy(m, x, v):
    return oracle.energy_angmom(m, x, v, oracle.Params(n1=0.0))[0]


def test_reduces_to_the_level0_step_without_encounters():
    n = 24
    u = W.uniforms(5, 3 * n).reshape(n, 3)
    m = np.full(n, 1e-7)
    a = 1.0 + 2.0 * (np.arange(n) + 0.5) / n
    x, v = W.elements_to_cartesian(G * (1 + m), a, 0.01 * u[:, 0], 0.005 * u[:, 1], 6.28 * u[:, 2], 0 * a,
                                   6.28 * ((np.arange(n) * 0.381966) % 1.0))
    v = oracle.to_democratic(m, v, 1.0)
    p = oracle.Params(n1=3.0, weight_mode=1)
    assert len(oracle.encounter_pairs(m, x, v, p)) == 0
    x1, v1 = oracle.step(m, x, v, p, 6.0)
    x2, v2 = oracle.step_hybrid(m, x, v, p, 6.0, nsub=400)          # RK4 of pure Kepler motion: converged to 1e-12
    assert np.abs(x1 - x2).max() <= 1e-11 and np.abs(v1 - v2).max() <= 1e-12
    with pytest.raises(ValueError):
        oracle.step_hybrid(m, x, v, oracle.Params(n1=3.0, weight_mode=0), 6.0)


def test_energy_is_kept_through_a_close_encounter():
    m, x, v = encounter_system()
    p = oracle.Params(n1=3.0, n2=0.4, dt_rcrit=2.0, pair_rule=oracle.PAIR_MAX, weight_mode=1)
    E0 = full_energy(m, x, v)
    dt, steps = 2.0, 40
    xh, vh = x.copy(), v.copy()
    xl, vl = x.copy(), v.copy()
    rmin, inside = 1e9, 0
    for _ in range(steps):
        rc, _, _ = oracle.rcrit(m, xh, vh, p)
        r01 = np.linalg.norm(xh[0] - xh[1])
        rmin = min(rmin, r01 / max(rc[0], rc[1]))
        inside += r01 < max(rc[0], rc[1])
        xh, vh = oracle.step_hybrid(m, xh, vh, p, dt, nsub=4000)
        xl, vl = oracle.step(m, xl, vl, p, dt)                       # level 0 only: the (1 - K) part is simply missing
    assert rmin < 0.6 and inside >= 3                                # the pair really went deep into its zone
    eh = abs(full_energy(m, xh, vh) / E0 - 1)
    el = abs(full_energy(m, xl, vl) / E0 - 1)
    assert eh < 1e-6, eh                                            # 2.5e-7 at dt = 2 d (level 0 only: 3.5e-4)
    assert el > 100 * eh, (el, eh)


def test_second_order_convergence_to_the_n_body_solution_through_an_encounter():
    m, x, v = encounter_system()
    M = 1.0
    T = 24.0
    # inertial-frame N-body ODE (star + planets), barycentre at rest
    vh = oracle.to_heliocentric(m, v, M)
    mt = M + m.sum()
    xs = -(m[:, None] * x).sum(0) / mt
    vs = -(m[:, None] * vh).sum(0) / mt
    X0 = np.vstack([xs, x + xs]); V0 = np.vstack([vs, vh + vs]); MM = np.concatenate([[M], m])

    def rhs(t, y):
        X = y[:15].reshape(5, 3); V = y[15:].reshape(5, 3)
        A = np.zeros_like(X)
        for i in range(5):
            d = X - X[i]
            r = np.linalg.norm(d, axis=1); r[i] = 1.0
            A[i] = (G * MM[:, None] * d / r[:, None] ** 3 * (np.arange(5) != i)[:, None]).sum(0)
        return np.concatenate([V.ravel(), A.ravel()])

    sol = solve_ivp(rhs, (0, T), np.concatenate([X0.ravel(), V0.ravel()]), method="DOP853", rtol=1e-13, atol=1e-16)
    Xf = sol.y[:15, -1].reshape(5, 3)
    x_true = Xf[1:] - Xf[0]
    p = oracle.Params(n1=3.0, n2=0.4, dt_rcrit=2.0, pair_rule=oracle.PAIR_MAX, weight_mode=1)
    errs = []
    for nst in (6, 12, 24):
        xx, vv = x.copy(), v.copy()
        for _ in range(nst):
            xx, vv = oracle.step_hybrid(m, xx, vv, p, T / nst, nsub=4000)
        errs.append(np.abs(xx - x_true).max())
    assert errs[2] < 2e-6
    assert 2.5 < errs[0] / errs[1] < 6.5 and 2.5 < errs[1] / errs[2] < 6.5, errs
