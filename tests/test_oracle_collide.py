"""Pins of oracle_step_hybrid_collide (reading R14: collision pass after every substep of the hybrid step's
A-flow; NOT built on the GPU yet): reduction to the pinned hybrid step, closed forms for two free bodies (the Sun and
their own gravity made negligible), the difference from a step-end pass.  CPU only."""
import numpy as np
import pytest

import oracle
from paper_2309_08217_b200 import workloads as W


def free_params():
    # G = 1e-60 with a 1e30 star: G M = 1e-30 and the Sun-kick sum(m v) / M_star vanish against positions of order
    # 100, no force matters over the step: the bodies move on straight lines
    return oracle.Params(G=1e-60, M_star=1e30, n1=3.0, n2=0.0, dt_rcrit=1.0, pair_rule=1, weight_mode=1)


def test_without_radii_it_is_the_hybrid_step_bit_for_bit():
    w = W.config(0, 300)
    p = oracle.Params(G=w.G, M_star=w.M_star, n1=w.n1, n2=w.n2, dt_rcrit=w.dt, pair_rule=w.pair_rule, weight_mode=1)
    vd = oracle.to_democratic(w.m, w.v, w.M_star)
    xh, vh = oracle.step_hybrid(w.m, w.x, vd, p, w.dt, nsub=16)
    m2, x2, v2, R2, idx = oracle.step_hybrid_collide(w.m, w.x, vd, np.zeros(w.N), p, w.dt, 16)
    assert len(m2) == w.N and (idx == np.arange(w.N)).all()
    assert (x2 == xh).all() and (v2 == vh).all() and (m2 == w.m).all()


def test_two_free_bodies_merge_and_follow_their_centre_of_mass():
    """Straight-line motion: the merged body ends at x_cm(0) + v_cm dt whenever the merger happens, carries the total
    momentum, and has lost mu u^2 / 2 of kinetic energy (perfectly inelastic collision)."""
    p = free_params()
    m = np.array([2.0, 1.0]); R = np.array([0.3, 0.2])
    x = np.array([[100.0, 0.0, 0.0], [104.0, 0.2, 0.0]]); v = np.array([[1.0, 0.0, 0.5], [-1.0, 0.0, 0.5]])
    m2, x2, v2, R2, idx = oracle.step_hybrid_collide(m, x, v, R, p, 3.0, 300)
    assert idx.tolist() == [0, 0] and m2.tolist() == [3.0]
    xcm = (m[:, None] * x).sum(0) / 3.0; vcm = (m[:, None] * v).sum(0) / 3.0
    np.testing.assert_allclose(x2[0], xcm + 3.0 * vcm, rtol=1e-13)
    np.testing.assert_allclose(v2[0], vcm, rtol=1e-13, atol=1e-15)
    ke0 = 0.5 * (m[:, None] * v * v).sum(); ke1 = 0.5 * 3.0 * (v2[0] ** 2).sum()
    assert ke0 - ke1 == pytest.approx(0.5 * (2.0 / 3.0) * 4.0, rel=1e-12)
    assert R2[0] == pytest.approx((0.027 + 0.008) ** (1 / 3), rel=1e-14)


def test_impact_parameter_decides():
    # closest approach = impact parameter b (reached in mid-step, sampled finely): b < R_1 + R_2 merges, b > does not
    p = free_params()
    m = np.array([1.0, 1.0]); R = np.array([0.25, 0.25]); v = np.array([[1.0, 0, 0], [-1.0, 0, 0]])
    for b, n_expected in ((0.49, 1), (0.51, 2)):
        x = np.array([[100.0, 0.0, 0.0], [104.0, b, 0.0]])
        assert len(oracle.step_hybrid_collide(m, x, v, R, p, 4.0, 4000)[0]) == n_expected


def test_a_pair_that_passes_through_within_the_step_is_caught_here_but_not_by_a_step_end_pass():
    p = free_params()
    m = np.array([1.0, 1.0]); R = np.array([0.25, 0.25])
    x = np.array([[100.0, 0.0, 0.0], [104.0, 0.1, 0.0]]); v = np.array([[1.0, 0, 0], [-1.0, 0, 0]])
    # closest approach after 2 of the 4 time units; apart again (4 units) at the end of the step
    xe, ve = oracle.step_hybrid(m, x, v, p, 4.0, nsub=400)
    assert len(oracle.merge(m, xe, ve, R)[0]) == 2                     # reading R13 alone misses it
    assert len(oracle.step_hybrid_collide(m, x, v, R, p, 4.0, 400)[0]) == 1
    # detection happens at substep ENDS only: 2 substeps sample t = 2 (closest approach: caught), 3 substeps sample
    # t = 4/3, 8/3 (separation 4/3 > 0.5: missed) -- the stated limitation of fixed substeps
    assert len(oracle.step_hybrid_collide(m, x, v, R, p, 4.0, 2)[0]) == 1
    assert len(oracle.step_hybrid_collide(m, x, v, R, p, 4.0, 3)[0]) == 2


def test_disc_with_one_planted_collision_keeps_mass_and_the_other_bodies():
    """In a real disc step: one pair on a collision course merges, every other body ends within rounding-level
    perturbation distance of the plain hybrid step (the merged pair's field is that of its centre of mass)."""
    w = W.config(0, 200)
    p = oracle.Params(G=w.G, M_star=w.M_star, n1=w.n1, n2=w.n2, dt_rcrit=w.dt, pair_rule=w.pair_rule, weight_mode=1)
    x = w.x.copy(); v = w.v.copy()
    x[7] = x[5] + [3.0e-4, 0.0, 0.0]; v[7] = v[5] + [-1.0e-4, 0.0, 0.0]     # closes 6e-4 AU in the 6-day step
    vd = oracle.to_democratic(w.m, v, w.M_star)
    R = np.full(w.N, 5.0e-5)
    m2, x2, v2, R2, idx = oracle.step_hybrid_collide(w.m, x, vd, R, p, w.dt, 64)
    assert len(m2) == w.N - 1 and idx[7] == idx[5] == 5
    assert m2.sum() == pytest.approx(w.m.sum(), rel=1e-15)
    xh, vh = oracle.step_hybrid(w.m, x, vd, p, w.dt, nsub=64)
    others = np.array([i for i in range(w.N) if i not in (5, 7)])
    assert np.abs(x2[idx[others]] - xh[others]).max() < 1e-9                # AU: the pair's quadrupole is all that changed
    xcm = (w.m[5] * xh[5] + w.m[7] * xh[7]) / (w.m[5] + w.m[7])
    assert np.abs(x2[5] - xcm).max() < 1e-7                                  # the merged body rides the pair's centre of mass
