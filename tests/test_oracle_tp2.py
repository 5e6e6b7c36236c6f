"""Pins of the oracle's TP2 mode (reading R9): pairs interact iff at least
one body is among the first n_big.  Pinned against hand values, against the already pinned
all-pairs path (full minus small-small subset), by symmetry, and by energy behaviour."""
import os

import numpy as np
import pytest

import oracle
from conftest import ROOT
from paper_2309_08217_b200 import workloads as W


def system(seed, n, n_big, spread=1.0):
    u = W.uniforms(seed, 7 * n).reshape(n, 7)
    m = 3e-7 * (0.5 + u[:, 0])
    m[:n_big] *= 3000.0
    a = 1.0 + spread * u[:, 1]
    x, v = W.elements_to_cartesian(W.G_DEFAULT * (1 + m), a, 0.02 * u[:, 2], 0.01 * u[:, 3],
                                   6.28 * u[:, 4], 6.28 * u[:, 5], 6.28 * u[:, 6])
    return m, x, oracle.to_democratic(m, v, 1.0)


def test_hand_values_three_bodies():
    rows = np.loadtxt(os.path.join(ROOT, "tests", "golden", "accel_tp2_collinear3.txt"))
    x = np.zeros((3, 3)); x[:, 0] = rows[:, 0]
    p = oracle.Params(G=1.0, n1=0.0, n2=0.0, n_big=1)
    a = oracle.accel(rows[:, 1].copy(), x, np.zeros((3, 3)), p)
    assert np.allclose(a[:, 0], rows[:, 2], rtol=1e-15, atol=0)
    assert np.all(a[:, 1:] == 0.0)


@pytest.mark.parametrize("rule", [oracle.PAIR_MAX, oracle.PAIR_MUTUAL_HILL])
def test_full_minus_small_subset_identity(rule):
    # forces on a small body: (all pairs) - (pairs among the small bodies only); on a big body: all pairs.
    # Both right-hand sides come from the all-pairs path, which has its own pins.  r_crit,i depends on
    # body i alone, so the subset system has the same zones.  A narrow ring puts many pairs inside zones.
    n, nb = 260, 5
    m, x, v = system(3, n, nb, spread=0.05)
    kw = dict(n1=3.0, n2=0.4, dt_rcrit=2.0, pair_rule=rule)
    full = oracle.accel(m, x, v, oracle.Params(**kw))
    sub = oracle.accel(m[nb:], x[nb:], v[nb:], oracle.Params(**kw))
    tp2 = oracle.accel(m, x, v, oracle.Params(n_big=nb, **kw))
    expect = full.copy()
    expect[nb:] -= sub
    scale = np.linalg.norm(full, axis=1)
    assert (np.linalg.norm(tp2 - expect, axis=1) / scale).max() <= 1e-13
    assert np.linalg.norm(sub, axis=1).max() > 0.0
    # encounter pairs: the full set without the small-small pairs
    pf = set(map(tuple, oracle.encounter_pairs(m, x, v, oracle.Params(**kw)).tolist()))
    pt = set(map(tuple, oracle.encounter_pairs(m, x, v, oracle.Params(n_big=nb, **kw)).tolist()))
    assert len(pf) > len(pt) > 0
    assert pt == {(i, j) for (i, j) in pf if i < nb or j < nb}


def test_limits_and_symmetry():
    n, nb = 150, 4
    m, x, v = system(5, n, nb, spread=0.3)
    base = dict(n1=3.0, n2=0.0)
    a_all = oracle.accel(m, x, v, oracle.Params(**base))
    assert np.array_equal(oracle.accel(m, x, v, oracle.Params(n_big=n, **base)), a_all)      # everybody big
    assert np.array_equal(oracle.accel(m, x, v, oracle.Params(n_big=-1, **base)), a_all)
    assert np.all(oracle.accel(m, x, v, oracle.Params(n_big=0, **base)) == 0.0)              # nobody big
    assert len(oracle.encounter_pairs(m, x, v, oracle.Params(n_big=0, n1=50.0))) == 0
    a = oracle.accel(m, x, v, oracle.Params(n_big=nb, **base))
    # the interaction is still pairwise and symmetric: total momentum and torque vanish
    f = m[:, None] * a
    assert np.abs(f.sum(0)).max() <= 1e-14 * np.abs(f).sum()
    assert np.abs(np.cross(x, f).sum(0)).max() <= 1e-14 * np.abs(np.cross(x, f)).sum()
    # a small body feels exactly the big ones (no zones: n1 = 0, so W = 1 and plain Newton)
    a0 = oracle.accel(m, x, v, oracle.Params(n1=0.0, n_big=nb))
    i = n - 1
    d = x[:nb] - x[i]
    r = np.linalg.norm(d, axis=1)
    direct = (W.G_DEFAULT * m[:nb, None] * d / r[:, None] ** 3).sum(0)
    assert np.allclose(a0[i], direct, rtol=1e-13, atol=0)


def spaced_system(n, n_big):
    """Well separated, nearly circular orbits (no close approaches over the short test runs)."""
    u = W.uniforms(77, 3 * n).reshape(n, 3)
    m = np.full(n, 3e-7)
    m[:n_big] = 3e-5
    a = 1.0 + 2.0 * (np.arange(n) + 0.5) / n
    x, v = W.elements_to_cartesian(W.G_DEFAULT * (1 + m), a, 0.005 * u[:, 0], 0.002 * u[:, 1],
                                   6.28 * u[:, 2], 0 * a, 6.28 * ((np.arange(n) * 0.381966) % 1.0))
    return m, x, oracle.to_democratic(m, v, 1.0)


def test_energy_counts_interacting_pairs_only_and_is_conserved():
    n, nb = 60, 3
    m, x, v = spaced_system(n, nb)
    p_all = oracle.Params(n1=0.0)
    p_tp2 = oracle.Params(n1=0.0, n_big=nb)
    E_all, L_all = oracle.energy_angmom(m, x, v, p_all)
    E_tp2, L_tp2 = oracle.energy_angmom(m, x, v, p_tp2)
    small = 0.0
    for i in range(nb, n):
        for j in range(i + 1, n):
            small += W.G_DEFAULT * m[i] * m[j] / np.linalg.norm(x[i] - x[j])
    assert abs((E_tp2 - E_all) - small) <= 4e-16 * abs(E_all)      # E_tp2 - E_all is a difference of rounded sums
    assert small > 1e6 * 4e-16 * abs(E_all)                         # ... that resolves the small-small potential well
    assert np.array_equal(L_all, L_tp2)
    # the TP2 forces are the gradient of the TP2 energy: bounded error that falls as dt^2
    errs = []
    for dt, steps in ((8.0, 20), (4.0, 40), (2.0, 80)):
        xx, vv = oracle.run(m, x, v, p_tp2, dt, steps)
        E1, L1 = oracle.energy_angmom(m, xx, vv, p_tp2)
        errs.append(abs(E1 / E_tp2 - 1))
        assert abs(np.linalg.norm(L1) / np.linalg.norm(L_tp2) - 1) <= 1e-13
    assert errs[0] < 1e-7, errs
    assert 2.5 < errs[0] / errs[1] < 6.0 and 2.5 < errs[1] / errs[2] < 6.0, errs
