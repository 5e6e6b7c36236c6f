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


# ---- the A-flow with an error-controlled integrator (reading R15: Gragg-Bulirsch-Stoer extrapolation) ----------------
def _deep_state():
    """The encounter system advanced to the steps in which the two planets are deepest inside their zone."""
    m, x, v = encounter_system()
    p = oracle.Params(n1=3.0, n2=0.4, dt_rcrit=2.0, pair_rule=oracle.PAIR_MAX, weight_mode=1)
    for _ in range(14):
        x, v = oracle.step_hybrid(m, x, v, p, 2.0, nsub=2000)
    rc, _, _ = oracle.rcrit(m, x, v, p)
    assert np.linalg.norm(x[0] - x[1]) < 0.8 * max(rc[0], rc[1])
    return m, x, v, p


def test_bs_moves_a_single_body_on_its_kepler_orbit():
    # one body: no pair forces, so the hybrid step is Sun-kick, Kepler motion, Sun-kick; the closed-form drift of the
    # (pinned) level-0 step is the reference for the extrapolation integrator, through a fifth of an e = 0.4 orbit
    mm = np.array([3e-6])
    x, v = W.elements_to_cartesian(G * (1 + mm), np.array([1.0]), np.array([0.4]), np.array([0.1]), np.array([1.0]),
                                   np.array([2.0]), np.array([5.9]))
    v = oracle.to_democratic(mm, v, 1.0)
    p = oracle.Params(n1=3.0, weight_mode=1)
    for dt in (6.0, 73.0, -73.0):
        x1, v1 = oracle.step(mm, x, v, p, dt)
        x2, v2, st = oracle.step_hybrid_bs(mm, x, v, p, dt, tol=1e-13, stats=True)
        assert np.abs(x1 - x2).max() <= 2e-12 and np.abs(v1 - v2).max() <= 1e-13, (dt, np.abs(x1 - x2).max())
        assert st[0] >= 1 and st[2] > 20


def test_bs_step_equals_the_step_built_from_pinned_pieces_and_dop853():
    # B(dt/2) C(dt/2) A(dt) C(dt/2) B(dt/2) with B, C from the pinned oracle calls and A(dt) integrated by scipy's DOP853
    # on a right-hand side written here from the pinned weight function: an independent route to the same step
    m, x, v, p = _deep_state()
    dt = 2.0
    rc, sa, vk = oracle.rcrit(m, x, v, p)
    v1, _ = oracle.kick(m, x, v, p, 0.5 * dt)
    x1 = oracle.sunkick(m, x, v1, p, 0.5 * dt)
    n = len(m)

    def rhs(t, y):
        X = y[:3 * n].reshape(n, 3); V = y[3 * n:].reshape(n, 3)
        A = -G * X / np.linalg.norm(X, axis=1)[:, None] ** 3
        for i in range(n):
            for j in range(n):
                if i == j:
                    continue
                d = X[j] - X[i]; q = np.linalg.norm(d)
                rcij = oracle.pair_rcrit(p, m[i], m[j], rc[i], rc[j], sa[i], sa[j], vk[i], vk[j])
                A[i] += G * m[j] * (1.0 - oracle.weight(q, rcij, 1)) * d / q ** 3
        return np.concatenate([V.ravel(), A.ravel()])

    sol = solve_ivp(rhs, (0, dt), np.concatenate([x1.ravel(), v1.ravel()]), method="DOP853", rtol=1e-13, atol=1e-18)
    x2 = sol.y[:3 * n, -1].reshape(n, 3); v2 = sol.y[3 * n:, -1].reshape(n, 3)
    x3 = oracle.sunkick(m, x2, v2, p, 0.5 * dt)
    v3, _ = oracle.kick(m, x3, v2, p, 0.5 * dt)
    xb, vb = oracle.step_hybrid_bs(m, x, v, p, dt, tol=1e-13)
    assert np.abs(xb - x3).max() <= 2e-12 and np.abs(vb - v3).max() <= 1e-13, (np.abs(xb - x3).max(), np.abs(vb - v3).max())
    # ... and the converged fixed-step RK4 of oracle_step_hybrid (the route the first GPU integrator was gated on)
    xr, vr = oracle.step_hybrid(m, x, v, p, dt, nsub=20000)
    assert np.abs(xb - xr).max() <= 1e-11 and np.abs(vb - vr).max() <= 1e-12


def test_bs_error_follows_the_tolerance_and_the_step_reverses():
    m, x, v, p = _deep_state()
    ref = oracle.step_hybrid_bs(m, x, v, p, 2.0, tol=1e-14)
    prev_err, prev_rhs = None, None
    for tol in (1e-6, 1e-9, 1e-12):
        xb, vb, st = oracle.step_hybrid_bs(m, x, v, p, 2.0, tol=tol, stats=True)
        err = max(np.abs(xb - ref[0]).max(), np.abs(vb - ref[1]).max())
        assert err <= 20 * tol, (tol, err)
        if prev_err is not None:
            assert st[2] >= prev_rhs                                 # a tighter tolerance never costs fewer right-hand sides
        prev_err, prev_rhs = err, st[2]
    xf, vf = oracle.step_hybrid_bs(m, x, v, p, 2.0, tol=1e-13)
    xr, vr = oracle.step_hybrid_bs(m, xf, vf, p, -2.0, tol=1e-13)
    # r_crit is taken from the opening state of each call (a_i from vis-viva, which the encounter itself changes by
    # 1e-4 here), so the two planets return only to that order times the complement force; the spectators return exactly
    assert np.abs(xr - x)[:2].max() <= 1e-7 and np.abs(vr - v)[:2].max() <= 1e-7
    assert np.abs(xr - x)[2:].max() <= 1e-13 and np.abs(vr - v)[2:].max() <= 1e-14
    with pytest.raises(ValueError):
        oracle.step_hybrid_bs(m, x, v, oracle.Params(n1=3.0, weight_mode=0), 2.0)
