"""GPU parity of the opt-in encounter mode (NEXT-1 of SURVEY.md 8(f); reading R11) against the
oracle's hybrid step: the oracle integrates the flow of H_A for ALL bodies with no lists and no groups, the
library moves only the bodies of an encounter group that way and every other body on its Kepler orbit."""
import numpy as np
import pytest

import oracle
from paper_2309_08217_b200 import binding as B
from paper_2309_08217_b200 import workloads as W

pytestmark = pytest.mark.gpu

G = W.G_DEFAULT


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    import torch
    assert torch.cuda.is_available(), "the gpu-marked tests need a CUDA device"
    B.load()


def workload(name, m, x, v_helio, dt, n2, pair_rule):
    return W.Workload(name, 0, np.ascontiguousarray(m), np.ascontiguousarray(x), np.ascontiguousarray(v_helio), dt, 1,
                      n2=n2, pair_rule=pair_rule)


def oparams(w):
    return oracle.Params(G=w.G, M_star=w.M_star, n1=w.n1, n2=w.n2, dt_rcrit=w.dt, pair_rule=w.pair_rule, weight_mode=1)


def encounter_system(lam1=-0.035, dt=2.0):
    """Two planets of 3e-5 Msun on nearly equal orbits that pass each other deep inside r_crit within a few
    steps, and two distant spectators (the system of tests/test_oracle_hybrid.py, heliocentric velocities)."""
    m = np.array([3e-5, 3e-5, 1e-6, 1e-6])
    a = np.array([1.0, 1.012, 1.7, 2.6])
    lam = np.array([0.0, lam1, 2.0, 4.0])
    x = np.stack([a * np.cos(lam), a * np.sin(lam), 0.002 * np.array([1, -1, 2, -2.0])], axis=1)
    vk = np.sqrt(G * (1 + m) / a)
    v = np.stack([-vk * np.sin(lam), vk * np.cos(lam), np.zeros(4)], axis=1)
    return workload("enc4", m, x, v, dt, 0.4, B.PAIR_MAX)


def disc_with_planted_groups(n, seed):
    """A disc of n small bodies in which a handful of pairs and one triple sit inside their changeover zones."""
    u = W.uniforms(seed, 6 * n).reshape(n, 6)
    m = 1e-7 * (0.5 + u[:, 0])
    a = 0.6 + 2.4 * (np.arange(n) + u[:, 1]) / n
    x, v = W.elements_to_cartesian(G * (1 + m), a, 0.01 * u[:, 2], 0.005 * u[:, 3], 6.28 * u[:, 4], 6.28 * u[:, 5],
                                   6.28 * ((np.arange(n) * 0.381966) % 1.0))
    # plant: body k+1 (and k+2 for the triple) next to body k, a fraction of body k's r_crit away
    for k, members in ((10, 1), (200, 1), (333, 2), (600, 1), (n - 40, 1)):
        r = np.linalg.norm(x[k])
        rc = 3.0 * np.cbrt(2 * m[k] / 3.0) * r
        for q in range(1, members + 1):
            x[k + q] = x[k] + rc * np.array([0.35 * q, 0.3 * (-1) ** q, 0.05])
            v[k + q] = v[k] * (1.0 + 2e-4 * q)
    return workload("disc+groups", m, x, v, 6.0, 0.0, B.PAIR_MUTUAL_HILL)


def hybrid(w, **kw):
    args = dict(weight_mode=1, encounter_mode=1, mega_nmax=-1)
    args.update(kw)
    return B.from_workload(w, **args)


def state_err(x, v, xo, vo):
    ex = np.linalg.norm(x - xo, axis=1) / np.linalg.norm(xo, axis=1)
    ev = np.linalg.norm(v - vo, axis=1) / np.linalg.norm(vo, axis=1)
    return max(ex.max(), ev.max())


def test_hybrid_steps_through_a_close_encounter_match_the_oracle():
    w = encounter_system()
    p = oparams(w)
    nsub = 512
    xo, vo = w.x.copy(), oracle.to_democratic(w.m, w.v, w.M_star)
    E0 = oracle.energy_angmom(w.m, xo, vo, oracle.Params(n1=0.0))[0]
    g = hybrid(w, enc_nsub=nsub)                                 # default listing: 8 r_crit, velocity test 1.25
    grouped_steps, worst = 0, 0.0
    for _ in range(30):
        xo, vo = oracle.step_hybrid(w.m, xo, vo, p, w.dt, nsub=nsub)
        g.step(w.dt, B.FP64)
        x, v = (t.cpu().numpy() for t in g.get_state())
        groups, bodies, largest, missed, status = g.encounter_stats()
        assert status == 0 and missed == 0
        grouped_steps += groups
        worst = max(worst, state_err(x, v, xo, vo))
    E, _ = g.energy_angmom()
    g.close()
    assert grouped_steps >= 5                                   # the pair was integrated as a group for several steps
    assert worst <= 1e-10, worst
    assert abs(E / E0 - 1) < 1e-6                                # level 0 alone loses 3.5e-4 here (test_oracle_hybrid.py)


def test_a_pair_that_enters_its_zone_ungrouped_is_reported():
    # listing only r < r_crit (enc_list_scale = 1): the step in which the two planets cross into their zone moves
    # them on Kepler orbits, and the next force evaluation says so
    w = encounter_system(lam1=0.09, dt=6.0)                      # starts at 1.4 r_crit, closing by 0.03 r_crit per step
    g = hybrid(w, enc_nsub=64, enc_list_scale=1.0)
    seen, flagged = 0, 0
    for _ in range(40):
        g.step(w.dt, B.FP64)
        groups, bodies, largest, missed, status = g.encounter_stats()
        seen += missed
        flagged += bool(status & 4)
        assert (missed > 0) == bool(status & 4)
    g.close()
    assert seen >= 1 and flagged >= 1


def test_hybrid_step_fp32_forces():
    # the kick in FP32 (policy P32), the encounter integration always in FP64
    w = encounter_system()
    p = oparams(w)
    xo, vo = oracle.step_hybrid(w.m, w.x, oracle.to_democratic(w.m, w.v, w.M_star), p, w.dt, nsub=256)
    g = hybrid(w, enc_nsub=256)
    g.step(w.dt, B.FP32)
    x, v = (t.cpu().numpy() for t in g.get_state())
    groups, bodies, largest, missed, status = g.encounter_stats()
    g.close()
    assert (groups, bodies, largest, missed, status) == (1, 2, 2, 0, 0)
    assert state_err(x, v, xo, vo) <= 1e-7


def test_disc_with_pairs_and_a_triple_one_step():
    n = 1000
    w = disc_with_planted_groups(n, 4)
    p = oparams(w)
    vd = oracle.to_democratic(w.m, w.v, w.M_star)
    po = oracle.encounter_pairs(w.m, w.x, vd, p)
    assert len(po) >= 6
    xo, vo = oracle.step_hybrid(w.m, w.x, vd, p, w.dt, nsub=128)
    xl, vl = oracle.step(w.m, w.x, vd, p, w.dt)
    assert state_err(xl, vl, xo, vo) > 1e-6                     # the complement matters for the planted bodies
    for prec, tol in ((B.FP64, 1e-10), (B.FP32, 1e-7)):
        g = hybrid(w, enc_nsub=128)
        g.step(w.dt, prec)
        x, v = (t.cpu().numpy() for t in g.get_state())
        groups, bodies, largest, missed, status = g.encounter_stats()
        g.close()
        assert missed == 0
        assert status == 0 and 3 <= largest <= 8 and groups >= 5 and bodies >= 11, (groups, bodies, largest, status)
        assert state_err(x, v, xo, vo) <= tol, (prec, state_err(x, v, xo, vo))


def test_hot_disc_pairs_entering_their_zones_are_grouped_in_time():
    # the performance shape at N = 4000: bodies cross a good part of a zone per step (velocity dispersion x dt is
    # 0.2 r_crit and more), so pairs ENTER their zones during a step.  The oracle has no lists; agreement over
    # consecutive steps says the velocity-aware listing grouped them before they got there.
    w = W.config(4, 4000)
    p = oparams(w)
    xo, vo = w.x.copy(), oracle.to_democratic(w.m, w.v, w.M_star)
    g = hybrid(w, enc_nsub=64)
    g1 = hybrid(w, enc_nsub=64, enc_list_scale=1.0)              # lists r < r_crit only: entering pairs are missed
    worst, missed, missed1, grouped = 0.0, 0, 0, 0
    for _ in range(6):
        xo, vo = oracle.step_hybrid(w.m, xo, vo, p, w.dt, nsub=64)
        g.step(w.dt, B.FP64)
        g1.step(w.dt, B.FP64)
        x, v = (t.cpu().numpy() for t in g.get_state())
        st = g.encounter_stats()
        assert st[4] == 0
        grouped += st[0]; missed += st[3]; missed1 += g1.encounter_stats()[3]
        worst = max(worst, state_err(x, v, xo, vo))
    g.close(); g1.close()
    assert grouped >= 3 and missed == 0 and worst <= 1e-10, (grouped, missed, worst)
    assert missed1 >= 1, missed1                                 # the check itself sees what the plain listing misses


def test_without_encounters_the_hybrid_step_is_the_level0_step():
    w = W.config(0)
    vd = oracle.to_democratic(w.m, w.v, w.M_star)
    w.n1 = 0.3                                                   # small zones: no pair within 1.5 r_crit in 5 steps
    assert len(oracle.encounter_pairs(w.m, w.x, vd, oracle.Params(G=w.G, n1=0.6, pair_rule=w.pair_rule))) == 0
    out = []
    for mode in (0, 1):
        g = B.from_workload(w, weight_mode=1, encounter_mode=mode, mega_nmax=-1)
        g.run(w.dt, 5, B.FP64)
        out.append([t.cpu().numpy() for t in g.get_state()])
        if mode:
            assert g.encounter_stats() == (0, 0, 0, 0, 0)
        g.close()
    # same arithmetic in two separately compiled kernels (and grids): equal up to the rounding of the momentum sums
    assert state_err(out[1][0], out[1][1], out[0][0], out[0][1]) <= 4e-15


def test_oversized_groups_are_reported_and_parameters_checked():
    u = W.uniforms(13, 6 * 800).reshape(800, 6)
    m = 3e-6 * (0.5 + u[:, 0])
    x, v = W.elements_to_cartesian(G * (1 + m), 1.0 + 0.02 * u[:, 1], 0.01 * u[:, 2], 0.005 * u[:, 3],
                                   0.3 * u[:, 4], 0.3 * u[:, 5], 0.2 * u[:, 0])
    w = workload("ring", m, x, v, 6.0, 0.0, B.PAIR_MUTUAL_HILL)      # a narrow ring: one percolating group
    g = hybrid(w, pair_capacity=200000)
    g.step(w.dt, B.FP64)
    groups, bodies, largest, missed, status = g.encounter_stats()
    x, v = (t.cpu().numpy() for t in g.get_state())
    g.close()
    assert status & 2 and largest <= 256 and np.isfinite(x).all() and np.isfinite(v).all()
    for bad in (dict(weight_mode=0), dict(n_big=3), dict(enc_list_scale=0.5), dict(enc_list_scale=9.0), dict(no_fused_step=True)):
        with pytest.raises(Exception):
            hybrid(w, **bad).close()


def deep_flyby_system():
    """Two 10 M_earth planets that pass each other within 1e-4 AU (1e-3 r_crit) in the middle of a 2-day step: the
    approach lasts a few thousandths of a day, below dt / 256."""
    m = np.array([3e-5, 3e-5, 1e-6])
    xa = np.array([1.0, 0.0, 0.0])
    va = np.array([0.0, np.sqrt(G * (1 + m[0])), 0.0])
    x = np.stack([xa, xa + np.array([0.004, 3.0e-4, 0.0]), [0.0, 1.9, 0.0]])
    v = np.stack([va, va + np.array([-0.004, 0.0, 0.0]), [-np.sqrt(G / 1.9), 0.0, 0.0]])
    return workload("flyby", m, x, v, 2.0, 0.0, B.PAIR_MUTUAL_HILL)


def test_bulirsch_stoer_resolves_a_deep_flyby():
    # default integrator of the groups (enc_nsub = 0): Bulirsch-Stoer extrapolation to enc_tol (reading R15).  Reference:
    # the oracle's extrapolation integrator over ALL bodies (no groups), itself pinned against DOP853 and the converged RK4.
    w = deep_flyby_system()
    p = oparams(w)
    vd = oracle.to_democratic(w.m, w.v, w.M_star)
    xo, vo = oracle.step_hybrid_bs(w.m, w.x, vd, p, w.dt, tol=1e-13)
    xh, vh = oracle.step_hybrid(w.m, w.x, vd, p, w.dt, nsub=100000)
    assert state_err(xh, vh, xo, vo) <= 1e-8                     # the two oracles agree where RK4 has converged that far
    x256, v256 = oracle.step_hybrid(w.m, w.x, vd, p, w.dt, nsub=256)
    err = {}
    for kw in (dict(enc_nsub=256), dict(), dict(enc_tol=1e-9)):
        g = hybrid(w, **kw)
        g.step(w.dt, B.FP64)
        x, v = (t.cpu().numpy() for t in g.get_state())
        st = g.encounter_stats()
        g.close()
        assert st == (1, 2, 2, 0, 0), st
        err[tuple(kw.items())] = state_err(x, v, xo, vo)
        if "enc_nsub" in kw:                                   # the fixed scheme is the first oracle's, resolved or not
            assert state_err(x, v, x256, v256) <= 1e-8
    assert err[(("enc_nsub", 256),)] > 1e-3, err                # 256 fixed substeps step over the approach
    # the flyby amplifies an error made before the closest approach about a thousandfold (the outgoing direction
    # depends on the impact parameter of 1e-4 AU), so the state error is ~1e3 x the tolerance of the integration
    assert err[()] <= 5e-9, err                                 # tolerance 1e-12 (default): 9e-10 measured
    assert err[(("enc_tol", 1e-9),)] <= 1e-6, err


def chain_cluster_disc(n, seed, sizes):
    """A disc of n small bodies with planted chains: `sizes[j]` bodies in a row, each 0.35 r_crit from the next, so
    that every chain is ONE encounter group of that size."""
    u = W.uniforms(seed, 6 * n).reshape(n, 6)
    m = 1e-7 * (0.5 + u[:, 0])
    a = 0.6 + 2.4 * (np.arange(n) + u[:, 1]) / n
    x, v = W.elements_to_cartesian(G * (1 + m), a, 0.01 * u[:, 2], 0.005 * u[:, 3], 6.28 * u[:, 4], 6.28 * u[:, 5],
                                   6.28 * ((np.arange(n) * 0.381966) % 1.0))
    k = 20
    for size in sizes:
        r = np.linalg.norm(x[k])
        rc = 3.0 * np.cbrt(2 * m[k] / 3.0) * r
        t = np.cross([0.0, 0.0, 1.0], x[k] / r)                    # along the orbit
        for q in range(1, size):
            x[k + q] = x[k] + rc * (0.35 * q * t + 0.05 * (-1) ** q * x[k] / r + [0.0, 0.0, 0.02 * (q % 3)])
            v[k + q] = v[k] * (1.0 + 1e-4 * (q % 5))
        k += size + 37
    return workload("disc+chains", m, x, v, 6.0, 0.0, B.PAIR_MUTUAL_HILL)


def test_large_groups_are_integrated_by_a_warp_or_a_cta():
    # groups of 14 (one warp, pair table in shared memory) and of 23 and 60 bodies (the whole CTA): one hybrid step
    # against the oracle, which knows nothing about groups
    w = chain_cluster_disc(900, 9, (14, 23, 60, 3))
    p = oparams(w)
    vd = oracle.to_democratic(w.m, w.v, w.M_star)
    po = oracle.encounter_pairs(w.m, w.x, vd, p)
    import scipy.sparse as sp
    from scipy.sparse.csgraph import connected_components
    adj = sp.coo_matrix((np.ones(len(po)), (po[:, 0], po[:, 1])), shape=(w.N, w.N))
    _, lab = connected_components(adj, directed=False)
    sizes = np.bincount(lab)
    assert sorted(sizes[sizes > 2].tolist())[-3:] == [14, 23, 60] or max(sizes) >= 60, sorted(sizes[sizes > 1].tolist())
    xo, vo = oracle.step_hybrid_bs(w.m, w.x, vd, p, w.dt, tol=1e-13)
    xl, vl = oracle.step(w.m, w.x, vd, p, w.dt)
    assert state_err(xl, vl, xo, vo) > 1e-6                     # the complement matters for the chains
    for prec, kw, tol in ((B.FP64, dict(), 1e-10), (B.FP32, dict(), 1e-7), (B.FP64, dict(enc_tol=1e-13), 1e-10)):
        g = hybrid(w, **kw)
        g.step(w.dt, prec)
        x, v = (t.cpu().numpy() for t in g.get_state())
        groups, bodies, largest, missed, status = g.encounter_stats()
        g.close()
        assert status == 0 and missed == 0 and largest >= 60 and bodies >= 100, (groups, bodies, largest, missed, status)
        assert state_err(x, v, xo, vo) <= tol, (prec, kw, state_err(x, v, xo, vo))
    # the RK4 scheme through the same teams: the first oracle with the same substeps
    xr, vr = oracle.step_hybrid(w.m, w.x, vd, p, w.dt, nsub=64)
    g = hybrid(w, enc_nsub=64)
    g.step(w.dt, B.FP64)
    x, v = (t.cpu().numpy() for t in g.get_state())
    g.close()
    assert state_err(x, v, xr, vr) <= 1e-10


def test_bs_steps_through_a_close_encounter_match_the_oracle():
    w = encounter_system()
    p = oparams(w)
    xo, vo = w.x.copy(), oracle.to_democratic(w.m, w.v, w.M_star)
    E0 = oracle.energy_angmom(w.m, xo, vo, oracle.Params(n1=0.0))[0]
    g = hybrid(w)                                                # Bulirsch-Stoer, tolerance 1e-12
    worst, grouped = 0.0, 0
    for _ in range(30):
        xo, vo = oracle.step_hybrid_bs(w.m, xo, vo, p, w.dt, tol=1e-13)
        g.step(w.dt, B.FP64)
        x, v = (t.cpu().numpy() for t in g.get_state())
        st = g.encounter_stats()
        assert st[3] == 0 and st[4] == 0
        grouped += st[0]
        worst = max(worst, state_err(x, v, xo, vo))
    E, _ = g.energy_angmom()
    g.close()
    assert grouped >= 5 and worst <= 1e-10, (grouped, worst)
    assert abs(E / E0 - 1) < 1e-6


def test_leapfrog_as_the_first_call_builds_its_own_pair_list():
    # genga_leapfrog has no leading kick: called right after genga_create (or after set_state(x), genga_drift,
    # genga_sunkick) there is no pair list of the current positions.  The library must make one before it forms the
    # groups; otherwise the planted pairs and the triple drift on Kepler orbits and their complement forces are lost.
    w = disc_with_planted_groups(1000, 4)
    res = []
    for prime in (False, True):
        g = hybrid(w, enc_nsub=128)
        if prime:
            g.accel(B.FP64)                                      # list and r_crit of the initial state, explicitly
        g.leapfrog(w.dt, 1, B.FP64)
        x, v = (t.cpu().numpy() for t in g.get_state())
        st = g.encounter_stats()
        g.close()
        assert st[3] == 0 and st[4] == 0 and st[0] >= 5 and st[1] >= 11, (prime, st)
        res.append((x, v))
    assert state_err(res[0][0], res[0][1], res[1][0], res[1][1]) <= 1e-13
    g = B.from_workload(w, weight_mode=1, mega_nmax=-1)          # level 0 only: the planted bodies end elsewhere
    g.leapfrog(w.dt, 1, B.FP64)
    x0, v0 = (t.cpu().numpy() for t in g.get_state())
    g.close()
    assert state_err(res[0][0], res[0][1], x0, v0) > 1e-6
    # and after a plain drift (which invalidates the list) the same holds
    g = hybrid(w, enc_nsub=128)
    g.accel(B.FP64); g.drift(0.0); g.leapfrog(w.dt, 1, B.FP64)
    x, v = (t.cpu().numpy() for t in g.get_state())
    st = g.encounter_stats()
    g.close()
    assert st[0] >= 5 and state_err(x, v, res[1][0], res[1][1]) <= 1e-13


def test_multilevel_changeover_matches_the_oracle():
    # NEXT-3, reading R16: L changeover levels with S sub-steps each and radius ratio F between
    # level 0 and the Bulirsch-Stoer integration.  The oracle recurses over ALL bodies; the library over each group.
    w = encounter_system()
    p = oparams(w)
    for L, S, F in ((2, 3, 2.08), (3, 2, 1.7), (2, 4, 0.0)):
        Fo = F if F > 0 else float(np.cbrt(S * S))                # the default ratio: S^(2/3)
        xo, vo = w.x.copy(), oracle.to_democratic(w.m, w.v, w.M_star)
        E0 = oracle.energy_angmom(w.m, xo, vo, oracle.Params(n1=0.0))[0]
        g = hybrid(w, enc_levels=L, enc_substeps=S, enc_level_ratio=F)
        worst, grouped = 0.0, 0
        for _ in range(30):
            xo, vo = oracle.step_multilevel(w.m, xo, vo, p, w.dt, L, S, Fo, tol=1e-13)
            g.step(w.dt, B.FP64)
            x, v = (t.cpu().numpy() for t in g.get_state())
            st = g.encounter_stats()
            assert st[3] == 0 and st[4] == 0
            grouped += st[0]
            worst = max(worst, state_err(x, v, xo, vo))
        E, _ = g.energy_angmom()
        g.close()
        assert grouped >= 5 and worst <= 1e-10, (L, S, F, grouped, worst)
        assert abs(E / E0 - 1) < 1e-6
    # a disc with planted pairs, a triple and chains of 14 and 23 bodies (warp and CTA teams), three levels
    w = chain_cluster_disc(700, 5, (14, 23, 3, 2))
    p = oparams(w)
    vd = oracle.to_democratic(w.m, w.v, w.M_star)
    xo, vo = oracle.step_multilevel(w.m, w.x, vd, p, w.dt, 3, 3, 2.08, tol=1e-13)
    x2, v2 = oracle.step_hybrid_bs(w.m, w.x, vd, p, w.dt, tol=1e-13)
    assert state_err(x2, v2, xo, vo) > 1e-9                      # the levels are a different splitting, not a relabelling
    g = hybrid(w, enc_levels=3, enc_substeps=3, enc_level_ratio=2.08)
    g.step(w.dt, B.FP64)
    x, v = (t.cpu().numpy() for t in g.get_state())
    st = g.encounter_stats()
    g.close()
    assert st[3] == 0 and st[4] == 0 and st[2] >= 23
    assert state_err(x, v, xo, vo) <= 1e-10, state_err(x, v, xo, vo)
    for bad in (dict(enc_levels=2, enc_nsub=16), dict(enc_levels=5), dict(enc_levels=2, enc_level_ratio=0.9)):
        with pytest.raises(Exception):
            hybrid(w, **bad).close()
