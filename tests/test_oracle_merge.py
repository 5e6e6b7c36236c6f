"""Pins of the oracle's step-end perfect mergers (oracle_merge; NEXT-4, reading R13)
against what the mathematics fixes: textbook perfectly-inelastic-collision identities, hand values, a library
connected-components routine, conservation laws.  CPU only."""
import numpy as np
import pytest
from scipy.sparse import coo_matrix
from scipy.sparse.csgraph import connected_components

import oracle


def test_no_overlap_is_identity():
    rng = np.random.default_rng(1)
    m = rng.uniform(1, 2, 50); x = rng.uniform(-1, 1, (50, 3)) * 100; v = rng.normal(size=(50, 3))
    R = np.full(50, 1e-6)
    m2, x2, v2, R2, idx = oracle.merge(m, x, v, R)
    assert len(m2) == 50 and (idx == np.arange(50)).all()
    assert (m2 == m).all() and (x2 == x).all() and (v2 == v).all() and (R2 == R).all()
    # R = 0 everywhere: nothing can collide, not even coincident bodies (strict inequality)
    x[7] = x[3]
    assert len(oracle.merge(m, x, v, np.zeros(50))[0]) == 50


def test_touching_spheres_do_not_merge_overlapping_do():
    m = np.array([1.0, 1.0]); v = np.zeros((2, 3))
    x = np.array([[0.0, 0, 0], [3.0, 0, 0]])
    assert len(oracle.merge(m, x, v, np.array([1.0, 2.0]))[0]) == 2            # r == R_i + R_j exactly
    assert len(oracle.merge(m, x, v, np.array([1.0, 2.0 + 1e-12]))[0]) == 1


def test_two_body_hand_values():
    # m = 1 and 3 at x = 0 and 4: centre of mass at 3; v = (2,0,0) and (-2,4,0): momentum (-4,12,0)/4
    m = np.array([1.0, 3.0]); x = np.array([[0.0, 0, 0], [4.0, 0, 0]]); v = np.array([[2.0, 0, 0], [-2.0, 4, 0]])
    R = np.array([3.0, 2.0])
    m2, x2, v2, R2, idx = oracle.merge(m, x, v, R)
    assert m2.tolist() == [4.0]
    assert x2.tolist() == [[3.0, 0.0, 0.0]]
    assert v2.tolist() == [[-1.0, 3.0, 0.0]]
    assert R2[0] == pytest.approx(35.0 ** (1 / 3), rel=1e-15)
    assert idx.tolist() == [0, 0]


def test_perfectly_inelastic_collision_identities():
    """Textbook: the kinetic energy lost is mu |v_rel|^2 / 2 and the angular momentum about the origin lost is
    mu x_rel cross v_rel (the internal orbital part), mu = m_i m_j / (m_i + m_j); momentum is kept."""
    rng = np.random.default_rng(5)
    for _ in range(20):
        m = rng.uniform(0.1, 5, 2); x = rng.normal(size=(2, 3)); v = rng.normal(size=(2, 3))
        R = np.full(2, 10.0)
        m2, x2, v2, _, _ = oracle.merge(m, x, v, R)
        mu = m[0] * m[1] / m.sum()
        ke0 = 0.5 * (m[:, None] * v * v).sum(); ke1 = 0.5 * m2[0] * (v2[0] ** 2).sum()
        assert ke0 - ke1 == pytest.approx(0.5 * mu * ((v[1] - v[0]) ** 2).sum(), rel=1e-12)
        L0 = (m[:, None] * np.cross(x, v)).sum(0); L1 = m2[0] * np.cross(x2[0], v2[0])
        np.testing.assert_allclose(L0 - L1, mu * np.cross(x[1] - x[0], v[1] - v[0]), rtol=1e-11, atol=1e-14)
        np.testing.assert_allclose(m2[0] * v2[0], (m[:, None] * v).sum(0), rtol=1e-14)


def test_chain_merges_through_the_middle_body_and_arrays_close_up():
    # bodies 1 - 3 - 4 form a chain along x (1~3, 3~4, 1 and 4 apart); 0, 2, 5 are bystanders
    x = np.array([[100.0, 0, 0], [0.0, 0, 0], [0.0, 50, 0], [1.5, 0, 0], [3.0, 0, 0], [0.0, -50, 0]])
    m = np.array([7.0, 1.0, 8.0, 2.0, 1.0, 9.0])
    v = np.array([[0.0, 0, 1], [4.0, 0, 0], [0.0, 0, 2], [0.0, 2, 0], [0.0, 0, 8], [0.0, 0, 3]])
    R = np.array([1.0, 1.0, 1.0, 1.0, 1.0, 1.0])
    m2, x2, v2, R2, idx = oracle.merge(m, x, v, R)
    assert idx.tolist() == [0, 1, 2, 1, 1, 3]
    assert m2.tolist() == [7.0, 4.0, 8.0, 9.0]
    assert x2.tolist() == [[100.0, 0, 0], [1.5, 0, 0], [0.0, 50, 0], [0.0, -50, 0]]      # (0 + 3 + 3) / 4
    assert v2.tolist() == [[0.0, 0, 1], [1.0, 1.0, 2.0], [0.0, 0, 2], [0.0, 0, 3]]
    assert R2[1] == pytest.approx(3.0 ** (1 / 3), rel=1e-15) and R2[[0, 2, 3]].tolist() == [1.0, 1.0, 1.0]


def test_massless_component_keeps_the_state_of_its_smallest_index():
    m = np.zeros(3); x = np.array([[1.0, 0, 0], [1.1, 0, 0], [9.0, 0, 0]]); v = np.array([[0.0, 1, 0], [0.0, 2, 0], [0.0, 3, 0]])
    m2, x2, v2, R2, idx = oracle.merge(m, x, v, np.full(3, 0.2))
    assert idx.tolist() == [0, 0, 1] and m2.tolist() == [0.0, 0.0]
    assert x2.tolist() == [[1.0, 0, 0], [9.0, 0, 0]] and v2.tolist() == [[0.0, 1, 0], [0.0, 3, 0]]
    # a test particle swallowed by a massive body leaves that body's state untouched
    m = np.array([0.0, 2.0]); x = np.array([[1.0, 0, 0], [1.1, 0, 0]]); v = np.array([[5.0, 0, 0], [0.0, 1, 0]])
    m2, x2, v2, _, _ = oracle.merge(m, x, v, np.full(2, 0.2))
    assert m2.tolist() == [2.0] and x2.tolist() == [[1.1, 0, 0]] and v2.tolist() == [[0.0, 1, 0]]


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_components_equal_the_library_routine_and_extensive_sums_are_kept(seed):
    """Clumpy random input (pairs, chains, clusters).  The partition must be scipy's connected components of the
    overlap graph; mass, sum m x, sum m v and sum R^3 are conserved; survivors sit at the smallest member index."""
    rng = np.random.default_rng(seed)
    n = 400
    centres = rng.uniform(-10, 10, (120, 3))
    x = centres[rng.integers(0, 120, n)] + rng.normal(scale=0.05, size=(n, 3))
    m = rng.uniform(0.5, 2, n); v = rng.normal(size=(n, 3)); R = rng.uniform(0.01, 0.06, n)
    d = np.linalg.norm(x[:, None, :] - x[None, :, :], axis=2)
    adj = (d < R[:, None] + R[None, :]) & ~np.eye(n, dtype=bool)
    ncomp, lab = connected_components(coo_matrix(adj), directed=False)
    assert ncomp < n - 50                                     # the input does exercise merging
    assert np.bincount(lab).max() >= 3                        # ... including components of three or more
    m2, x2, v2, R2, idx = oracle.merge(m, x, v, R)
    assert len(m2) == ncomp
    # same partition: bodies share a new index iff they share a component
    assert ((idx[:, None] == idx[None, :]) == (lab[:, None] == lab[None, :])).all()
    # survivors in order of their smallest member
    first = np.array([np.flatnonzero(idx == k).min() for k in range(ncomp)])
    assert (np.diff(first) > 0).all()
    np.testing.assert_allclose(m2, np.bincount(idx, weights=m), rtol=1e-14)
    for dd in range(3):
        np.testing.assert_allclose(m2 * x2[:, dd], np.bincount(idx, weights=m * x[:, dd]), rtol=1e-12, atol=1e-13)
        np.testing.assert_allclose(m2 * v2[:, dd], np.bincount(idx, weights=m * v[:, dd]), rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(R2 ** 3, np.bincount(idx, weights=R ** 3), rtol=1e-13)
    # bodies that touched nobody are bit-identical
    alone = np.flatnonzero(np.bincount(lab)[lab] == 1)
    assert (x2[idx[alone]] == x[alone]).all() and (v2[idx[alone]] == v[alone]).all() and (m2[idx[alone]] == m[alone]).all()


def test_empty_and_single():
    z = np.zeros((0, 3))
    assert len(oracle.merge(np.zeros(0), z, z, np.zeros(0))[0]) == 0
    m2, x2, _, _, idx = oracle.merge(np.ones(1), np.ones((1, 3)), np.ones((1, 3)), np.ones(1))
    assert len(m2) == 1 and idx.tolist() == [0]


def test_tp2_rule_small_bodies_do_not_collide_with_each_other():
    """Reading R9 + R13: hand case on a line.  Bodies 0, 1 are big.  2 overlaps 0; 3 overlaps 2 only (a small-small
    contact: no edge, 3 stays); 4 and 5 overlap each other only (stay); 1 overlaps 0 (two bigs merge: one big left)."""
    x = np.zeros((6, 3)); x[:, 0] = [0.0, 1.5, -1.5, -3.0, 50.0, 51.0]
    m = np.array([10.0, 6.0, 1.0, 1.0, 1.0, 1.0]); v = np.zeros((6, 3)); v[:, 1] = [0.0, 1.0, 2.0, 3.0, 4.0, 5.0]
    R = np.ones(6)
    m2, x2, v2, R2, idx, nb = oracle.merge_tp2(m, x, v, R, 2)
    assert idx.tolist() == [0, 0, 0, 1, 2, 3] and nb == 1
    assert m2.tolist() == [17.0, 1.0, 1.0, 1.0]
    assert x2[:, 0].tolist() == [(6 * 1.5 - 1.5) / 17.0, -3.0, 50.0, 51.0]
    assert v2[:, 1].tolist() == [(6.0 + 2.0) / 17.0, 3.0, 4.0, 5.0]
    # the same bodies with every pair allowed: 0-1-2-3 is one chain, 4-5 a pair
    m3, _, _, _, idx3 = oracle.merge(m, x, v, R)
    assert idx3.tolist() == [0, 0, 0, 0, 1, 1] and m3.tolist() == [18.0, 2.0]
    # n_big = N is the all-pairs rule; n_big = 0 lets nothing collide
    assert oracle.merge_tp2(m, x, v, R, 6)[4].tolist() == idx3.tolist()
    assert len(oracle.merge_tp2(m, x, v, R, 0)[0]) == 6


def test_tp2_rule_equals_the_library_components_of_the_restricted_graph():
    rng = np.random.default_rng(3)
    n, nb = 300, 12
    x = rng.uniform(-1, 1, (n, 3)); R = rng.uniform(0.01, 0.05, n); R[:nb] = 0.25
    m = rng.uniform(0.5, 2, n); v = rng.normal(size=(n, 3))
    d = np.linalg.norm(x[:, None, :] - x[None, :, :], axis=2)
    big = np.arange(n) < nb
    adj = (d < R[:, None] + R[None, :]) & ~np.eye(n, dtype=bool) & (big[:, None] | big[None, :])
    ncomp, lab = connected_components(coo_matrix(adj), directed=False)
    m2, x2, v2, R2, idx, nb2 = oracle.merge_tp2(m, x, v, R, nb)
    assert len(m2) == ncomp < n - 10
    assert ((idx[:, None] == idx[None, :]) == (lab[:, None] == lab[None, :])).all()
    assert nb2 == len(set(idx[:nb].tolist()))
    np.testing.assert_allclose(m2, np.bincount(idx, weights=m), rtol=1e-14)
