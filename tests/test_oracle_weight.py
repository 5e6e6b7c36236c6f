"""Pins of the Hamiltonian-consistent pair weight W = K - r dK/dr (reading R10; NEXT-3 of
SURVEY.md 8(f)): the kick with this weight is minus the gradient of the pair potential -G m_i m_j K/r."""
import numpy as np

import oracle


def test_hand_value_and_limits():
    rc = 2.0
    # y = 1/2: K = 1/2, dK/dy = 2 (1/2)(1/2) / (1/2)^2 = 2, r = (0.1 + 0.45) rc, r dK/dr = 0.55 * 2 / 0.9 = 11/9
    assert abs(oracle.weight(0.55 * rc, rc, 1) - (0.5 - 11.0 / 9.0)) <= 4e-15
    assert abs(oracle.weight(0.55 * rc, rc, 0) - 0.5) <= 1e-15
    for mode in (0, 1):
        assert oracle.weight(0.1 * rc, rc, mode) == 0.0 and oracle.weight(0.05 * rc, rc, mode) == 0.0
        assert oracle.weight(rc, rc, mode) == 1.0 and oracle.weight(3.0 * rc, rc, mode) == 1.0
        assert oracle.weight(1.0, 0.0, mode) == 1.0                      # no zone: plain Newton
    # continuous at both ends of the zone (K' -> 0 there)
    assert abs(oracle.weight(0.1 * rc * (1 + 1e-9), rc, 1)) <= 1e-8
    assert abs(oracle.weight(rc * (1 - 1e-9), rc, 1) - 1.0) <= 1e-8


def test_weight_is_minus_r2_times_derivative_of_K_over_r():
    rc = 0.37
    for r in np.linspace(0.11, 0.99, 45) * rc:
        h = 1e-6 * rc
        f = lambda q: oracle.changeover(q, rc) / q            # the pinned K
        deriv = (f(r + h) - f(r - h)) / (2 * h)
        assert abs(oracle.weight(r, rc, 1) - (-r * r * deriv)) <= 2e-8 * max(1.0, abs(r * r * deriv))


def test_two_body_force_is_gradient_of_the_weighted_potential():
    # bodies a and b on the x axis inside each other's zone; PAIR_MAX with n2 term so that r_crit does not
    # depend on the masses' Hill radii only: fix r_crit through n2 * dt * v_K of circular orbits
    G, M = 1.0, 1.0
    m = np.array([1e-3, 2e-3])
    x = np.array([[1.0, 0.0, 0.0], [1.02, 0.0, 0.0]])
    v = np.array([[0.0, 1.0, 0.0], [0.0, 1.0 / np.sqrt(1.02), 0.0]])
    p1 = oracle.Params(G=G, M_star=M, n1=0.0, n2=0.05, dt_rcrit=1.0, pair_rule=oracle.PAIR_MAX, weight_mode=1)
    rc, _, _ = oracle.rcrit(m, x, v, p1)
    rcij = rc.max()
    r = 0.02
    assert 0.1 * rcij < r < rcij
    a = oracle.accel(m, x, v, p1)
    U = lambda q: -G * m[0] * m[1] * oracle.changeover(q, rcij) / q
    h = 1e-7
    dUdr = (U(r + h) - U(r - h)) / (2 * h)
    # force on body 0 along +x is +dU/dr (it sits at smaller x), on body 1 it is -dU/dr
    assert abs(m[0] * a[0, 0] - dUdr) <= 1e-6 * abs(dUdr)
    assert abs(m[1] * a[1, 0] + dUdr) <= 1e-6 * abs(dUdr)
    a0 = oracle.accel(m, x, v, oracle.Params(G=G, M_star=M, n1=0.0, n2=0.05, dt_rcrit=1.0, pair_rule=oracle.PAIR_MAX))
    assert abs(a0[0, 0] - G * m[1] * oracle.changeover(r, rcij) / r ** 2) <= 1e-12 * abs(a0[0, 0])
    assert abs(a0[0, 0] - a[0, 0]) > 0.1 * abs(a0[0, 0])              # the two weights really differ here
