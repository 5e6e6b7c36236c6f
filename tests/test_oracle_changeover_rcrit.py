"""Pins for the oracle's changeover function (O4), critical radius (O2, Eq. 1),
pair radius (O3) and velocity conventions (O1).  CPU only."""
import numpy as np
import pytest

import oracle
from conftest import read_golden

K_GAUSS = 0.01720209895


def test_changeover_hand_values():
    for q, K in read_golden("changeover_hand.txt"):
        for rc in (1.0, 0.037, 12.5):
            assert oracle.changeover(q * rc, rc) == pytest.approx(K, abs=1e-15)


def test_changeover_limits_exact():
    # north_star: K = 0 and K = 1 at the changeover limits
    rc = 0.3
    assert oracle.changeover(0.1 * rc, rc) == 0.0
    assert oracle.changeover(0.0, rc) == 0.0
    assert oracle.changeover(rc, rc) == 1.0
    assert oracle.changeover(np.nextafter(rc, 2.0), rc) == 1.0
    assert 0.0 < oracle.changeover(np.nextafter(rc, 0.0), rc) <= 1.0
    # no zone: K = 1 wherever the bodies are apart
    assert oracle.changeover(1e-9, 0.0) == 1.0
    assert oracle.changeover(0.0, 0.0) == 0.0


def test_changeover_symmetry_monotone_smooth():
    rc = 1.7
    y = np.linspace(0.0, 1.0, 10001)
    K = np.array([oracle.changeover(rc * (0.1 + 0.9 * t), rc) for t in y])
    assert np.all(np.diff(K) >= 0.0)
    assert np.max(np.abs(K + K[::-1] - 1.0)) < 1e-13        # K(y) + K(1-y) = 1
    assert np.max(np.abs(np.diff(K))) < 3e-4                  # no jump: max slope is 2
    assert K[0] == 0.0 and K[-1] == 1.0
    # slope vanishes at both ends (smooth switch)
    assert K[1] < 2e-8 and 1.0 - K[-2] < 2e-8


def test_rcrit_eq1_golden():
    for m, a, dt, n1, n2, expect in read_golden("rcrit_eq1.txt"):
        p = oracle.Params(G=K_GAUSS ** 2, M_star=1.0, n1=n1, n2=n2, dt_rcrit=dt, pair_rule=oracle.PAIR_MAX)
        x = np.array([[a, 0.0, 0.0]])
        v = np.array([[0.0, K_GAUSS / np.sqrt(a), 0.0]])
        rc, sa, vk = oracle.rcrit([m], x, v, p)
        assert sa[0] == pytest.approx(a, rel=1e-14)
        assert vk[0] == pytest.approx(K_GAUSS / np.sqrt(a), rel=1e-14)
        assert rc[0] == pytest.approx(expect, rel=2e-10)


def test_rcrit_uses_semi_major_axis_not_radius():
    # body at perihelion of an a = 2, e = 0.5 orbit: r = 1 but R_H = a (m/3M)^(1/3) = 0.02
    G, a, e = 1.0, 2.0, 0.5
    r = a * (1 - e)
    vp = np.sqrt(G * (1 + e) / (a * (1 - e)))
    p = oracle.Params(G=G, n1=3.0, n2=0.0, pair_rule=oracle.PAIR_MAX)
    rc, sa, vk = oracle.rcrit([3e-6], [[r, 0, 0]], [[0, vp, 0]], p)
    assert sa[0] == pytest.approx(2.0, rel=1e-14)
    assert rc[0] == pytest.approx(0.06, rel=1e-13)
    assert vk[0] == pytest.approx(np.sqrt(0.5), rel=1e-14)
    # unbound body: a falls back to r
    rc, sa, vk = oracle.rcrit([3e-6], [[r, 0, 0]], [[0, 10.0, 0]], p)
    assert sa[0] == pytest.approx(r)


def test_pair_rule_hand_values():
    # mutual Hill: m_i + m_j = 3e-6 -> cube root of 1e-6 = 0.01; mean a = 2 -> 3 * 0.01 * 2 = 0.06
    p = oracle.Params(G=1.0, n1=3.0, n2=0.0, pair_rule=oracle.PAIR_MUTUAL_HILL)
    assert oracle.pair_rcrit(p, 1.5e-6, 1.5e-6, 0.1, 0.2, 1.0, 3.0, 1.0, 0.5) == pytest.approx(0.06, rel=1e-14)
    # velocity term takes the faster body: 0.4 * 6 * 1.0 = 2.4
    p2 = oracle.Params(G=1.0, n1=3.0, n2=0.4, dt_rcrit=6.0, pair_rule=oracle.PAIR_MUTUAL_HILL)
    assert oracle.pair_rcrit(p2, 1.5e-6, 1.5e-6, 0.1, 0.2, 1.0, 3.0, 1.0, 0.5) == pytest.approx(2.4, rel=1e-14)
    # PAIR_MAX: the larger per-body radius
    p3 = oracle.Params(G=1.0, pair_rule=oracle.PAIR_MAX)
    assert oracle.pair_rcrit(p3, 1.0, 2.0, 0.1, 0.2, 1.0, 3.0, 1.0, 0.5) == 0.2
    # symmetric in (i, j)
    assert oracle.pair_rcrit(p2, 1e-6, 2e-6, 0.1, 0.2, 1.0, 3.0, 1.0, 0.5) == \
        oracle.pair_rcrit(p2, 2e-6, 1e-6, 0.2, 0.1, 3.0, 1.0, 0.5, 1.0)


def test_democratic_velocities_are_barycentric():
    rng = np.random.default_rng(7)
    n, M = 12, 1.3
    m = rng.uniform(1e-4, 1e-2, n)
    vh = rng.normal(size=(n, 3))
    vd = oracle.to_democratic(m, vh, M)
    # independent inertial-frame computation: star velocity V* = -sum m v_h/(M + sum m); v_bary = v_h + V*
    Vstar = -(m[:, None] * vh).sum(0) / (M + m.sum())
    assert np.allclose(vd, vh + Vstar, rtol=0, atol=1e-15)
    # total barycentric momentum including the star vanishes
    assert np.allclose((m[:, None] * vd).sum(0) + M * Vstar, 0.0, atol=1e-17)
    # round trip
    assert np.allclose(oracle.to_heliocentric(m, vd, M), vh, rtol=0, atol=2e-15)
