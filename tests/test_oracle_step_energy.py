"""Pins for the oracle's Sun-kick (O8), step (O10), merged run and diagnostics (O11): closed forms,
an inertial-frame re-derivation, convergence to a DOP853 solution of the full N-body problem,
symplectic invariants.  CPU only."""
import numpy as np
import pytest
from scipy.integrate import solve_ivp

import oracle
from paper_2309_08217_b200.workloads import elements_to_cartesian

NOZONE = dict(n1=0.0, n2=0.0, pair_rule=oracle.PAIR_MAX)


def inertial_energy_angmom(G, M, m, xh, vh):
    """E and L of star + bodies in the barycentric inertial frame, star treated as one more body."""
    mall = np.concatenate([[M], m])
    X = np.concatenate([[np.zeros(3)], xh])
    V = np.concatenate([[np.zeros(3)], vh])
    X = X - (mall[:, None] * X).sum(0) / mall.sum()
    V = V - (mall[:, None] * V).sum(0) / mall.sum()
    E = 0.5 * (mall * (V ** 2).sum(1)).sum()
    for i in range(len(mall)):
        for j in range(i + 1, len(mall)):
            E -= G * mall[i] * mall[j] / np.linalg.norm(X[i] - X[j])
    return E, (mall[:, None] * np.cross(X, V)).sum(0)


def small_system(seed=1, n=5, G=1.0, M=1.0, mass=3e-4):
    rng = np.random.default_rng(seed)
    m = mass * rng.uniform(0.5, 1.5, n)
    a = np.linspace(1.0, 1.0 + 0.9 * (n - 1), n)
    e = rng.uniform(0.0, 0.1, n)
    xh, vh = elements_to_cartesian(G * (M + m), a, e, rng.uniform(0, 0.05, n), *(rng.uniform(0, 6.28, (3, n))))
    return m, xh, vh


def test_two_body_closed_form():
    # one planet: E = -G M m/(2a), |L| = (M m/(M+m)) sqrt(G (M+m) a (1-e^2))
    G, M, m, a, e = 1.3, 1.0, 0.02, 1.4, 0.3
    xh, vh = elements_to_cartesian(G * (M + m), a, e, 0.2, 0.5, 1.0, 2.0)
    p = oracle.Params(G=G, M_star=M, **NOZONE)
    vd = oracle.to_democratic([m], vh, M)
    E, L = oracle.energy_angmom([m], xh, vd, p)
    assert E == pytest.approx(-G * M * m / (2 * a), rel=1e-14)
    assert np.linalg.norm(L) == pytest.approx(M * m / (M + m) * np.sqrt(G * (M + m) * a * (1 - e * e)), rel=1e-14)


def test_diagnostics_equal_inertial_frame_values():
    G, M = 0.9, 1.1
    m, xh, vh = small_system(3, 9, G, M, mass=2e-3)
    vd = oracle.to_democratic(m, vh, M)
    E, L = oracle.energy_angmom(m, xh, vd, oracle.Params(G=G, M_star=M, **NOZONE))
    Ei, Li = inertial_energy_angmom(G, M, m, xh, vh)
    assert E == pytest.approx(Ei, rel=1e-13)
    assert np.allclose(L, Li, rtol=1e-13, atol=1e-16)


def nbody_dop853(G, M, m, xh, vh, t):
    """Full (star + bodies) Newtonian problem in an inertial frame; returns heliocentric x, v at t."""
    mall = np.concatenate([[M], m]); nb = len(mall)
    y0 = np.concatenate([np.concatenate([[np.zeros(3)], xh]).ravel(), np.concatenate([[np.zeros(3)], vh]).ravel()])

    def f(_, y):
        X = y[:3 * nb].reshape(nb, 3)
        d = X[None] - X[:, None]
        r3 = (d ** 2).sum(-1) ** 1.5
        np.fill_diagonal(r3, np.inf)
        A = G * (mall[None, :, None] * d / r3[..., None]).sum(1)
        return np.concatenate([y[3 * nb:], A.ravel()])

    s = solve_ivp(f, (0, t), y0, method="DOP853", rtol=1e-13, atol=1e-16)
    X = s.y[:3 * nb, -1].reshape(nb, 3); V = s.y[3 * nb:, -1].reshape(nb, 3)
    return X[1:] - X[0], V[1:] - V[0]


def test_step_converges_to_true_dynamics_at_second_order():
    # With no changeover zone the level-0 map is a 2nd-order integrator of the real N-body problem:
    # halving dt must quarter the error against an independent high-accuracy ODE solution.
    G, M = 1.0, 1.0
    m, xh, vh = small_system(1, 4, G, M, mass=1e-3)
    T = 3.0
    xr, vr = nbody_dop853(G, M, m, xh, vh, T)
    p = oracle.Params(G=G, M_star=M, **NOZONE)
    errs = []
    for nsteps in (150, 300, 600):
        x, v = xh.copy(), oracle.to_democratic(m, vh, M)
        for _ in range(nsteps):
            x, v = oracle.step(m, x, v, p, T / nsteps)
        errs.append(max(np.abs(x - xr).max(), np.abs(oracle.to_heliocentric(m, v, M) - vr).max()))
    assert errs[0] < 1e-5
    assert 3.7 < errs[0] / errs[1] < 4.3 and 3.7 < errs[1] / errs[2] < 4.3


def test_sunkick_hand_value():
    p = oracle.Params(G=1.0, M_star=2.0, **NOZONE)
    m = np.array([0.5, 0.25]); v = np.array([[1.0, 0, 0], [0, 2.0, 0]]); x = np.zeros((2, 3))
    # s = (0.5*[1,0,0] + 0.25*[0,2,0]) / 2 = [0.25, 0.25, 0]; tau = 4 -> shift [1, 1, 0]
    assert np.array_equal(oracle.sunkick(m, x, v, p, 4.0), [[1, 1, 0], [1, 1, 0]])


def test_encounter_free_energy_error_bounded_and_second_order():
    # north_star: "bounded energy error for an encounter-free run"
    G, M = 0.01720209895 ** 2, 1.0
    m, xh, vh = small_system(4, 16, G, M, mass=3e-6)
    p = oracle.Params(G=G, M_star=M, n1=3.0, n2=0.0, pair_rule=oracle.PAIR_MUTUAL_HILL)
    v0 = oracle.to_democratic(m, vh, M)
    assert len(oracle.encounter_pairs(m, xh, v0, p)) == 0
    E0, L0 = oracle.energy_angmom(m, xh, v0, p)
    amp = []
    for dt in (8.0, 4.0):
        x, v = xh.copy(), v0.copy()
        dE, dL = [], []
        for _ in range(int(2400 / dt)):
            x, v = oracle.step(m, x, v, p, dt)
            E, L = oracle.energy_angmom(m, x, v, p)
            dE.append(E / E0 - 1); dL.append(np.linalg.norm(L) / np.linalg.norm(L0) - 1)
        dE = np.array(dE)
        assert np.abs(dL).max() < 1e-13                    # every sub-map conserves O11's L exactly
        half = len(dE) // 2                                 # bounded: no growth from first to second half
        assert np.abs(dE[half:]).max() < 1.5 * np.abs(dE[:half]).max()
        amp.append(np.abs(dE).max())
    assert amp[0] < 1e-7
    assert 3.0 < amp[0] / amp[1] < 5.0


def test_time_reversibility():
    G, M = 1.0, 1.0
    m, xh, vh = small_system(6, 6, G, M, mass=1e-4)
    p = oracle.Params(G=G, M_star=M, n1=3.0, n2=0.0, pair_rule=oracle.PAIR_MAX)
    x, v = xh.copy(), oracle.to_democratic(m, vh, M)
    v0 = v.copy()
    for _ in range(50):
        x, v = oracle.step(m, x, v, p, 0.02)
    for _ in range(50):
        x, v = oracle.step(m, x, v, p, -0.02)
    assert np.abs(x - xh).max() < 1e-11 and np.abs(v - v0).max() < 1e-11


def test_run_equals_step_sequence_when_rcrit_is_velocity_independent():
    # merged half-kicks: identical map up to rounding when W does not depend on v (no zone)
    G, M = 1.0, 1.0
    m, xh, vh = small_system(8, 7, G, M, mass=1e-4)
    p = oracle.Params(G=G, M_star=M, **NOZONE)
    x, v = xh.copy(), oracle.to_democratic(m, vh, M)
    xs, vs = x.copy(), v.copy()
    for _ in range(20):
        xs, vs = oracle.step(m, xs, vs, p, 0.03)
    xr, vr = oracle.run(m, x, v, p, 0.03, 20)
    assert np.abs(xr - xs).max() < 1e-13 and np.abs(vr - vs).max() < 1e-13
    x1, v1 = oracle.run(m, x, v, p, 0.03, 1)
    x2, v2 = oracle.step(m, x, v, p, 0.03)
    assert np.array_equal(x1, x2) and np.array_equal(v1, v2)
