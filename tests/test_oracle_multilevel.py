"""Pins of the oracle's multi-level hybrid step (NEXT-3 of SURVEY.md 8(f), second half; reading R16:
PAPER.md:45-47 "multiple changeover functions ... another symplectic integration step with a reduced time step can be
applied in between", PAPER.md:55 levels and sub-steps).  The level structure itself is a reading (Grimm et al. 2022 is
not in the container); what is pinned here is that the oracle computes that reading correctly."""
import os

import numpy as np
import pytest
from scipy.integrate import solve_ivp

import oracle
from paper_2309_08217_b200 import workloads as W

from test_oracle_hybrid import encounter_system, full_energy

G = W.G_DEFAULT
GOLD = os.path.join(os.path.dirname(__file__), "golden", "level_weight_hand.txt")


def params():
    return oracle.Params(n1=3.0, n2=0.4, dt_rcrit=2.0, pair_rule=oracle.PAIR_MAX, weight_mode=1)


def test_shell_weights_hand_values_and_partition_of_unity():
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        r, rc, l, L, F, wgt = line.split()
        assert oracle.level_weight(float(r), float(rc), int(l), int(L), float(F)) == pytest.approx(float(wgt), abs=1e-15)
    for L, F in ((1, 2.0), (2, 2.0), (3, 2.08), (4, 1.5)):
        for r in np.linspace(0.01, 1.3, 200):
            tot = sum(oracle.level_weight(r, 1.0, l, L, F) for l in range(L + 1))
            assert tot == pytest.approx(1.0, abs=1e-13)
        # outside the outermost zone only shell 0 acts; inside the innermost core (0.1 r_crit / F^(L-1)) only Bulirsch-Stoer
        assert [oracle.level_weight(1.0001, 1.0, l, L, F) for l in range(L + 1)] == [1.0] + [0.0] * L
        core = 0.0999 / F ** (L - 1)
        assert [oracle.level_weight(core, 1.0, l, L, F) for l in range(L + 1)] == [0.0] * L + [1.0]
        # shell l only acts between 0.1 r_crit / F^l and r_crit / F^(l-1)
        for l in range(1, L):
            assert oracle.level_weight(1.0001 / F ** (l - 1), 1.0, l, L, F) == 0.0
            assert oracle.level_weight(0.0999 / F ** l, 1.0, l, L, F) == 0.0


def test_one_level_is_the_two_level_hybrid_step_bit_for_bit():
    m, x, v = encounter_system()
    p = params()
    for _ in range(16):
        x, v = oracle.step_hybrid_bs(m, x, v, p, 2.0, tol=1e-12)
    a = oracle.step_hybrid_bs(m, x, v, p, 2.0, tol=1e-13)
    b = oracle.step_multilevel(m, x, v, p, 2.0, 1, 3, 2.0, tol=1e-13)
    assert (a[0] == b[0]).all() and (a[1] == b[1]).all()
    for bad in ((0, 3, 2.0), (2, 0, 2.0), (2, 3, 1.0)):
        with pytest.raises(ValueError):
            oracle.step_multilevel(m, x, v, p, 2.0, *bad)


def test_without_encounters_it_is_the_level0_step():
    n = 24
    u = W.uniforms(5, 3 * n).reshape(n, 3)
    m = np.full(n, 1e-7)
    a = 1.0 + 2.0 * (np.arange(n) + 0.5) / n
    x, v = W.elements_to_cartesian(G * (1 + m), a, 0.01 * u[:, 0], 0.005 * u[:, 1], 6.28 * u[:, 2], 0 * a,
                                   6.28 * ((np.arange(n) * 0.381966) % 1.0))
    v = oracle.to_democratic(m, v, 1.0)
    p = oracle.Params(n1=3.0, weight_mode=1)
    x1, v1 = oracle.step(m, x, v, p, 6.0)
    x2, v2 = oracle.step_multilevel(m, x, v, p, 6.0, 3, 3, 2.08, tol=1e-13)      # 9 Kepler sub-flows by extrapolation
    assert np.abs(x1 - x2).max() <= 2e-12 and np.abs(v1 - v2).max() <= 1e-13


def test_two_levels_equal_the_composition_written_out_with_pinned_pieces():
    # A state in which the two planets are inside the level-0 zone but OUTSIDE the level-1 zone (r > r_crit / F) for
    # the whole step: the Bulirsch-Stoer remainder vanishes and flow_1(dt) = [kick_1(h/2) Kepler(h) kick_1(h/2)]^S with
    # h = dt / S.  The same composition is written here from the closed-form drift and a shell kick built from the
    # pinned weight function: an independent route through the recursion, the step sizes and the shell weights.
    m, x, v = encounter_system()
    p = params()
    for _ in range(11):
        x, v = oracle.step_hybrid_bs(m, x, v, p, 2.0, tol=1e-12)
    rc, sa, vk = oracle.rcrit(m, x, v, p)
    rc01 = oracle.pair_rcrit(p, m[0], m[1], rc[0], rc[1], sa[0], sa[1], vk[0], vk[1])
    F, S, dt = 4.0, 3, 1.0
    r01 = np.linalg.norm(x[0] - x[1])
    assert rc01 / F < 0.9 * r01 < r01 < 0.95 * rc01                          # inside zone 0, well outside zone 1
    got = oracle.step_multilevel(m, x, v, p, dt, 2, S, F, tol=1e-13)

    def shell_kick(xx, vv, tau):
        out = vv.copy()
        for i in range(len(m)):
            for j in range(len(m)):
                if i == j:
                    continue
                d = xx[j] - xx[i]; q = np.linalg.norm(d)
                rcij = oracle.pair_rcrit(p, m[i], m[j], rc[i], rc[j], sa[i], sa[j], vk[i], vk[j])
                out[i] += tau * G * m[j] * (oracle.weight(q, rcij / F, 1) - oracle.weight(q, rcij, 1)) * d / q ** 3
        return out

    v1, _ = oracle.kick(m, x, v, p, 0.5 * dt)
    x1 = oracle.sunkick(m, x, v1, p, 0.5 * dt)
    h = dt / S
    for _ in range(S):
        v1 = shell_kick(x1, v1, 0.5 * h)
        x1, v1 = oracle.drift(x1, v1, p, h)
        v1 = shell_kick(x1, v1, 0.5 * h)
    x2 = oracle.sunkick(m, x1, v1, p, 0.5 * dt)
    v2, _ = oracle.kick(m, x2, v1, p, 0.5 * dt)
    assert np.linalg.norm(x2[0] - x2[1]) > rc01 / F                         # still outside zone 1 at the end
    assert np.abs(got[0] - x2).max() <= 5e-13 and np.abs(got[1] - v2).max() <= 5e-14


def test_second_order_convergence_to_the_n_body_solution_with_three_levels():
    m, x, v = encounter_system()
    M, T = 1.0, 24.0
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
    p = params()
    errs = []
    for nst in (6, 12, 24):
        xx, vv = x.copy(), v.copy()
        for _ in range(nst):
            xx, vv = oracle.step_multilevel(m, xx, vv, p, T / nst, 3, 3, 2.08, tol=1e-12)
        errs.append(np.abs(xx - x_true).max())
    assert errs[2] < 2e-6
    assert 2.5 < errs[0] / errs[1] < 6.5 and 2.5 < errs[1] / errs[2] < 6.5, errs


def test_energy_through_the_encounter_and_the_work_left_to_bulirsch_stoer():
    m, x0, v0 = encounter_system()
    p = params()
    E0 = full_energy(m, x0, v0)
    out = {}
    for L in (1, 2, 3):
        x, v = x0.copy(), v0.copy()
        rhs = 0
        for _ in range(40):
            x, v, st = oracle.step_multilevel(m, x, v, p, 2.0, L, 3, 2.08, tol=1e-12, stats=True)
            rhs += st[2]
        out[L] = (abs(full_energy(m, x, v) / E0 - 1), rhs)
    assert all(e < 1e-6 for e, _ in out.values()), out                 # level 0 alone loses 3.5e-4 here
    # the sub-levels are symplectic maps of their own: the energy error stays of the size of the two-level step's
    assert out[2][0] < 5 * out[1][0] + 1e-8 and out[3][0] < 5 * out[1][0] + 1e-8, out
