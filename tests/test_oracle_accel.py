"""Pins for the oracle's K-weighted all-pairs acceleration (O2-O5) and encounter set (O6):
hand values, closed forms, invariants, 50-digit brute force.  CPU only."""
import mpmath as mp
import numpy as np
import pytest

import oracle
from conftest import read_golden


def newton_numpy(m, x, G):
    """Textbook Newtonian accelerations, vectorised (library ops only)."""
    d = x[None, :, :] - x[:, None, :]
    r2 = (d ** 2).sum(-1)
    np.fill_diagonal(r2, np.inf)
    return G * (m[None, :, None] * d / r2[..., None] ** 1.5).sum(1)


NOZONE = dict(n1=0.0, n2=0.0, pair_rule=oracle.PAIR_MAX)


def test_collinear_three_body_hand_values():
    rows = read_golden("accel_collinear3.txt")
    x = np.array([[r[0], 0.0, 0.0] for r in rows])
    m = np.array([r[1] for r in rows])
    a = oracle.accel(m, x, np.zeros_like(x) + [0, 1, 0], oracle.Params(G=1.0, **NOZONE))
    assert np.allclose(a[:, 0], [r[2] for r in rows], rtol=1e-15)
    assert np.all(a[:, 1:] == 0.0)


def test_equilateral_triangle_and_square():
    G, mass, s = 2.5, 0.7, 1.3
    tri = s / np.sqrt(3) * np.array([[np.cos(t), np.sin(t), 0] for t in (0.3, 0.3 + 2 * np.pi / 3, 0.3 + 4 * np.pi / 3)])
    a = oracle.accel([mass] * 3, tri, np.ones_like(tri), oracle.Params(G=G, **NOZONE))
    assert np.allclose(np.linalg.norm(a, axis=1), np.sqrt(3) * G * mass / s ** 2, rtol=1e-14)
    assert np.allclose(a / np.linalg.norm(a, axis=1)[:, None], -tri / np.linalg.norm(tri, axis=1)[:, None], atol=1e-14)
    sq = 0.5 * s * np.array([[1, 1, 0], [-1, 1, 0], [-1, -1, 0], [1, -1, 0.0]])
    a = oracle.accel([mass] * 4, sq, np.ones_like(sq), oracle.Params(G=G, **NOZONE))
    assert np.allclose(np.linalg.norm(a, axis=1), (np.sqrt(2) + 0.5) * G * mass / s ** 2, rtol=1e-14)


def test_regular_polygon_closed_form():
    # n equal masses on a circle of radius R: |a| = (G m / 4 R^2) sum_{k=1}^{n-1} 1/sin(pi k/n), pointing inwards
    n, R, G, mass = 2048, 1.7, 0.9, 3e-7
    t = 2 * np.pi * np.arange(n) / n
    x = R * np.stack([np.cos(t), np.sin(t), np.zeros(n)], 1)
    a = oracle.accel(np.full(n, mass), x, np.ones_like(x), oracle.Params(G=G, **NOZONE))
    k = np.arange(1, n)
    expect = G * mass / (4 * R * R) * np.sum(1.0 / np.sin(np.pi * k / n))
    radial = -(a * x).sum(1) / R
    assert np.allclose(radial, expect, rtol=1e-12)
    tang = np.abs(a[:, 0] * (-np.sin(t)) + a[:, 1] * np.cos(t))
    # the two nearest neighbours pull 40x harder than the net force and cancel only as well as the
    # rounded vertex coordinates allow: bound the residual against that single-pair term
    nearest = G * mass / (2 * R * np.sin(np.pi / n)) ** 2
    assert tang.max() < 5e-12 * nearest


def clustered_system(seed, n, G=1.0):
    """Bodies on near-circular orbits in a narrow ring so that many pairs sit inside r_crit."""
    rng = np.random.default_rng(seed)
    m = 10.0 ** rng.uniform(-7, -4, n)
    a = rng.uniform(0.95, 1.05, n)
    th = rng.uniform(0, 2 * np.pi, n)
    x = np.stack([a * np.cos(th), a * np.sin(th), rng.normal(0, 2e-3, n)], 1)
    vc = np.sqrt(G / a)
    v = np.stack([-vc * np.sin(th), vc * np.cos(th), rng.normal(0, 1e-3, n)], 1)
    return m, x, v


@pytest.mark.parametrize("rule,n2", [(oracle.PAIR_MAX, 0.0), (oracle.PAIR_MUTUAL_HILL, 0.0),
                                     (oracle.PAIR_MAX, 0.4), (oracle.PAIR_MUTUAL_HILL, 0.4)])
def test_momentum_and_torque_vanish_with_changeover(rule, n2):
    # W_ij symmetric and the force central => sum m a = 0 and sum m x cross a = 0, for ANY r_crit
    m, x, v = clustered_system(3, 300)
    p = oracle.Params(G=1.0, n1=3.0, n2=n2, dt_rcrit=0.05, pair_rule=rule)
    assert len(oracle.encounter_pairs(m, x, v, p)) > 20            # the zone is actually exercised
    a = oracle.accel(m, x, v, p)
    scale = (m[:, None] * np.abs(a)).sum()
    assert np.abs((m[:, None] * a).sum(0)).max() < 2e-15 * scale
    assert np.abs((m[:, None] * np.cross(x, a)).sum(0)).max() < 4e-15 * scale * np.abs(x).max()


def test_no_zone_reduces_to_newton():
    m, x, v = clustered_system(5, 257)
    a = oracle.accel(m, x, v, oracle.Params(G=0.37, **NOZONE))
    ref = newton_numpy(m, x, 0.37)
    assert np.abs(a - ref).max() < 1e-12 * np.abs(ref).max()


def mp_accel(m, x, v, p):
    """The definition (O2-O5) in 50-digit arithmetic, plain double loop."""
    mp.mp.dps = 50
    n = len(m)
    M, G = mp.mpf(p.M_star), mp.mpf(p.G)
    mm = [mp.mpf(float(t)) for t in m]
    X = [[mp.mpf(float(t)) for t in row] for row in x]
    V = [[mp.mpf(float(t)) for t in row] for row in v]
    sa, rc, vk = [], [], []
    for i in range(n):
        r = mp.sqrt(sum(c * c for c in X[i]))
        v2 = sum(c * c for c in V[i])
        a = 1 / (2 / r - v2 / (G * M))
        if not a > 0:
            a = r
        sa.append(a)
        vk.append(mp.sqrt(G * M / a))
        rc.append(max(p.n1 * a * mp.cbrt(mm[i] / (3 * M)), p.n2 * p.dt_rcrit * vk[-1]))
    out = np.zeros((n, 3))
    enc = []
    for i in range(n):
        acc = [mp.mpf(0)] * 3
        for j in range(n):
            if j == i:
                continue
            d = [X[j][k] - X[i][k] for k in range(3)]
            r = mp.sqrt(sum(c * c for c in d))
            if p.pair_rule == oracle.PAIR_MUTUAL_HILL:
                rcij = max(p.n1 * mp.cbrt((mm[i] + mm[j]) / (3 * M)) * (sa[i] + sa[j]) / 2,
                           p.n2 * p.dt_rcrit * max(vk[i], vk[j]))
            else:
                rcij = max(rc[i], rc[j])
            if r < rcij and i < j:
                enc.append((i, j))
            if r == 0:
                continue
            if rcij > 0:
                y = (r - rcij / 10) / (9 * rcij / 10)
                K = 0 if y <= 0 else (1 if y >= 1 else y * y / (2 * y * y - 2 * y + 1))
            else:
                K = 1
            s = G * mm[j] * K / r ** 3
            acc = [acc[k] + s * d[k] for k in range(3)]
        out[i] = [float(c) for c in acc]
    return out, enc


@pytest.mark.parametrize("rule", [oracle.PAIR_MAX, oracle.PAIR_MUTUAL_HILL])
def test_brute_force_50_digits(rule):
    m, x, v = clustered_system(11, 40)
    m[:4] *= 300.0                                    # a few big bodies: wide zones, many K<1 pairs
    # force two coincident bodies and one pair exactly inside 0.1 r_crit
    x[7] = x[6]
    x[9] = x[8] + [1e-7, 0, 0]
    p = oracle.Params(G=1.0, n1=3.0, n2=0.4, dt_rcrit=0.02, pair_rule=rule)
    ref, enc = mp_accel(m, x, v, p)
    a = oracle.accel(m, x, v, p)
    assert np.all(np.isfinite(a))
    err = np.linalg.norm(a - ref, axis=1) / np.linalg.norm(ref, axis=1)
    assert err.max() < 5e-14
    got = oracle.encounter_pairs(m, x, v, p)
    assert len(enc) > 5
    assert [tuple(t) for t in got.tolist()] == sorted(enc)


def test_partial_weight_hand_value():
    # two bodies, r = 0.55 r_crit -> K = 1/2 (golden changeover_hand.txt): a = G m K / r^2
    G, rc = 1.0, 0.06                                  # m_i + m_j = 3e-6, mean a = 2 -> rc = 0.06 (mutual Hill)
    r = 0.55 * rc
    # circular-velocity states at a_1 = 2 - r/2, a_2 = 2 + r/2 so the mean semi-major axis is exactly 2
    x = np.array([[2 - r / 2, 0, 0], [2 + r / 2, 0, 0]])
    v = np.array([[0, np.sqrt(G / x[0, 0]), 0], [0, np.sqrt(G / x[1, 0]), 0]])
    m = np.array([1.5e-6, 1.5e-6])
    a = oracle.accel(m, x, v, oracle.Params(G=G, n1=3.0, n2=0.0, pair_rule=oracle.PAIR_MUTUAL_HILL))
    assert a[0, 0] == pytest.approx(+G * 1.5e-6 * 0.5 / r ** 2, rel=1e-9)
    assert a[1, 0] == pytest.approx(-G * 1.5e-6 * 0.5 / r ** 2, rel=1e-9)


def test_encounter_set_boundary_cases():
    # PAIR_MAX with one heavy body: r_crit,ij = 3 * 1 * (3e-6/3)^(1/3) = 0.03 for a circular orbit at a = 1
    p = oracle.Params(G=1.0, n1=3.0, n2=0.0, pair_rule=oracle.PAIR_MAX)
    for eps, inside in ((-1e-9, True), (+1e-9, False)):
        r = 0.03 * (1 + eps)
        x = np.array([[1.0, 0, 0], [1.0, r, 0]])
        v = np.array([[0, 1.0, 0], [0, 1.0, 0]])
        # second body massless so that only body 0 sets the radius; its a differs slightly but is unused
        pairs = oracle.encounter_pairs([3e-6, 0.0], x, v, p)
        assert (len(pairs) == 1) == inside
        if inside:
            assert pairs.tolist() == [[0, 1]]


def test_encounter_set_matches_numpy_brute_force():
    m, x, v = clustered_system(21, 400)
    p = oracle.Params(G=1.0, n1=3.0, n2=0.0, pair_rule=oracle.PAIR_MAX)
    rc, _, _ = oracle.rcrit(m, x, v, p)
    d = np.linalg.norm(x[None] - x[:, None], axis=-1)
    rcij = np.maximum(rc[None], rc[:, None])
    ii, jj = np.nonzero(np.triu(d < rcij, 1))
    got = oracle.encounter_pairs(m, x, v, p)
    assert len(got) > 30
    assert got.tolist() == np.stack([ii, jj], 1).tolist()


def test_subset_functions_equal_the_full_ones():
    # the sampled-output forms used at sizes where all N^2 pairs take too long on a CPU
    m, x, v = clustered_system(21, 300)
    p = oracle.Params(G=1.0, n1=3.0, n2=0.4, dt_rcrit=0.02, pair_rule=oracle.PAIR_MAX)
    a = oracle.accel(m, x, v, p)
    pf = set(map(tuple, oracle.encounter_pairs(m, x, v, p).tolist()))
    assert len(pf) > 10
    sel = np.array(sorted({i for q in list(pf)[:7] for i in q} | {0, 299, 150}))
    assert np.array_equal(oracle.accel_subset(m, x, v, p, sel), a[sel])
    ps = oracle.encounter_pairs_subset(m, x, v, p, sel)
    assert ps == {q for q in pf if q[0] in sel or q[1] in sel} and len(ps) >= 7
