"""GPU parity of the step-end perfect mergers (genga_set_radii / genga_merge; NEXT-4, R13)
against oracle.merge on the same seeded state: the partition (newidx) bit-exact, merged m, x, v, R to rounding
(the member sums are atomic adds: <= 1e-14), untouched bodies bit-exact; then the SHRUNK system against the oracle
on the merged state (accelerations, encounter sets, steps, E and L) in both force precisions."""
import dataclasses

import numpy as np
import pytest

import oracle
from paper_2309_08217_b200 import binding as B
from paper_2309_08217_b200 import workloads as W

pytestmark = pytest.mark.gpu

R_BODY = 1.0e-4          # AU: inflated planetesimals, still far inside r_crit (a few 1e-3 AU)


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    import torch
    assert torch.cuda.is_available(), "the gpu-marked tests need a CUDA device"
    B.load()


def oparams(w, **kw):
    d = dict(G=w.G, M_star=w.M_star, n1=w.n1, n2=w.n2, dt_rcrit=w.dt, pair_rule=w.pair_rule)
    d.update(kw)
    return oracle.Params(**d)


def planted(cfg, n, seed, n_pairs, n_chains, n_clusters):
    """A config disc in which some bodies were moved onto others: overlapping pairs, chains of three whose ends do
    not touch (1.5 R apart each, ends 3 R apart), tight clusters of four.  Radii differ from body to body."""
    w = W.config(cfg, n)
    n = w.N                                  # config 2 adds its 100 embryos to n planetesimals
    rng = np.random.default_rng(seed)
    x = w.x.copy(); v = w.v.copy()
    R = R_BODY * (0.8 + 0.4 * W.uniforms(seed + 1, n))
    ids = rng.permutation(n)[: 2 * n_pairs + 3 * n_chains + 4 * n_clusters]
    k = 0
    for _ in range(n_pairs):
        i, j = ids[k], ids[k + 1]; k += 2
        x[j] = x[i] + 0.9 * (R[i] + R[j]) * np.array([0.6, 0.0, 0.8]); v[j] = v[i] * (1 + 1e-4)
    for _ in range(n_chains):
        a, b, c = ids[k], ids[k + 1], ids[k + 2]; k += 3
        x[b] = x[a] + np.array([0.95 * (R[a] + R[b]), 0, 0])
        x[c] = x[b] + np.array([0.95 * (R[b] + R[c]), 0, 0])
        assert np.linalg.norm(x[c] - x[a]) > R[a] + R[c]
        v[b] = v[a] * (1 - 2e-4); v[c] = v[a] * (1 + 3e-4)
    for _ in range(n_clusters):
        q = ids[k:k + 4]; k += 4
        for t in q[1:]:
            x[t] = x[q[0]] + 0.3 * R_BODY * rng.normal(size=3); v[t] = v[q[0]] * (1 + 1e-4 * rng.normal())
    return dataclasses.replace(w, x=x, v=v), R


def merged_pair(w, R, precision, prepare=None, **kw):
    """(GPU handle after genga_merge, its results, the oracle's results from the GPU's own pre-merge state)."""
    import torch
    g = B.from_workload(w, **kw)
    g.set_radii(torch.from_numpy(R).to(g.device))
    if prepare:
        prepare(g)
    else:
        g.accel(precision)
    x0, v0 = (t.cpu().numpy() for t in g.get_state())           # stored (democratic) velocities
    n_merged, status, newidx = g.merge(precision)
    mo, xo, vo, Ro, idxo = oracle.merge(w.m, x0, v0, R)
    return g, (n_merged, status, newidx.cpu().numpy()), (x0, v0), (mo, xo, vo, Ro, idxo)


def check_merge(g, res, pre, orc, w, R):
    n_merged, status, newidx = res
    x0, v0 = pre
    mo, xo, vo, Ro, idxo = orc
    assert status == 0
    assert n_merged == len(w.m) - len(mo) and g.N == len(mo)
    assert (newidx == idxo).all()                                    # the partition and the order: exact
    x, v = (t.cpu().numpy() for t in g.get_state())
    Rg = g.get_radii().cpu().numpy()
    mg = g.get_mass().cpu().numpy()
    assert x.shape == xo.shape
    assert np.abs(mg / np.where(mo > 0, mo, 1.0) - (mo > 0)).max() <= 1e-13      # atomic sums of up to 700 members
    scale_x = np.linalg.norm(xo, axis=1, keepdims=True); scale_v = np.linalg.norm(vo, axis=1, keepdims=True)
    assert (np.abs(x - xo) / scale_x).max() <= 1e-14
    assert (np.abs(v - vo) / scale_v).max() <= 1e-14
    assert np.abs(Rg / Ro - 1).max() <= 1e-14
    alone = np.flatnonzero(np.bincount(idxo)[idxo] == 1)             # bodies nothing happened to: bit-exact
    assert (x[idxo[alone]] == x0[alone]).all() and (v[idxo[alone]] == v0[alone]).all() and (Rg[idxo[alone]] == R[alone]).all() and (mg[idxo[alone]] == w.m[alone]).all()


@pytest.mark.parametrize("cfg,n,seed,plant", [
    (0, 2048, 3, (6, 3, 2)),          # one-kernel step path (N <= 3000); 20 bodies removed: NP stays 2048
    (0, 2050, 4, (2, 1, 1)),          # 7 removed: N' = 2043 falls below a padding boundary (NP 2560 -> 2048)
    (2, 5000, 5, (10, 4, 3)),         # unequal masses (embryos + planetesimals), the three-launch step path
    (4, 40000, 6, (30, 10, 5)),       # the performance shape at full size
])
@pytest.mark.parametrize("precision", [B.FP64, B.FP32])
def test_merge_parity_and_the_shrunk_system(cfg, n, seed, plant, precision):
    w, R = planted(cfg, n, seed, *plant)
    g, res, pre, orc = merged_pair(w, R, precision)
    check_merge(g, res, pre, orc, w, R)
    assert res[0] == plant[0] + 2 * plant[1] + 3 * plant[2]
    mo, xo, vo, Ro, _ = orc
    p = oparams(w)
    # the force evaluation genga_merge ran on the new body set
    big = len(mo) > 20000
    sel = np.arange(0, len(mo), 97 if big else 1)
    ao = oracle.accel_subset(mo, xo, vo, p, sel) if big else oracle.accel(mo, xo, vo, p)
    a = g.get_accel().cpu().numpy()[sel]
    err = np.linalg.norm(a - ao, axis=1) / np.linalg.norm(ao, axis=1)
    assert err.max() <= (1e-12 if precision == B.FP64 else 1e-4), err.max()
    if not big:
        assert set(map(tuple, g.encounter_pairs().tolist())) == set(map(tuple, oracle.encounter_pairs(mo, xo, vo, p).tolist()))
        # E and L of the merged state, then three steps of the smaller system
        E, L = g.energy_angmom(); Eo, Lo = oracle.energy_angmom(mo, xo, vo, p)
        assert abs(E / Eo - 1) <= 1e-12 and np.abs(L - Lo).max() <= 1e-12 * np.linalg.norm(Lo)
        g.run(w.dt, 3, precision)
        xr, vr = oracle.run(mo, xo, vo, p, w.dt, 3)
        x, v = (t.cpu().numpy() for t in g.get_state())
        tol = 1e-10 if precision == B.FP64 else 1e-6
        assert (np.linalg.norm(x - xr, axis=1) / np.linalg.norm(xr, axis=1)).max() <= tol
        assert (np.linalg.norm(v - vr, axis=1) / np.linalg.norm(vr, axis=1)).max() <= tol
    # nothing overlaps any more: a second pass merges nothing and changes nothing
    xb, vb = (t.clone() for t in g.get_state())
    n2, s2, idx2 = g.merge(precision)
    assert n2 == 0 and s2 == 0 and (idx2.cpu().numpy() == np.arange(g.N)).all()
    xa, va = g.get_state()
    assert (xa == xb).all() and (va == vb).all()
    g.close()


def test_total_momentum_mass_and_centre_of_mass_are_kept():
    w, R = planted(0, 2048, 11, 8, 4, 3)
    import torch
    g = B.from_workload(w)
    g.set_radii(torch.from_numpy(R).to(g.device))
    g.accel(B.FP64)
    m0 = w.m; x0, v0 = (t.cpu().numpy() for t in g.get_state())
    n_merged, status, newidx = g.merge()
    assert n_merged == 8 + 8 + 9 and status == 0
    idx = newidx.cpu().numpy()
    x1, v1 = (t.cpu().numpy() for t in g.get_state())
    m1 = np.bincount(idx, weights=m0)                                  # exact: what the masses must be
    for d in range(3):
        assert np.allclose(m1 * x1[:, d], np.bincount(idx, weights=m0 * x0[:, d]), rtol=1e-13, atol=1e-22)
        assert np.allclose(m1 * v1[:, d], np.bincount(idx, weights=m0 * v0[:, d]), rtol=1e-13, atol=1e-24)
    assert np.allclose(g.get_radii().cpu().numpy() ** 3, np.bincount(idx, weights=R ** 3), rtol=1e-13)
    g.close()


def test_without_radii_nothing_merges_even_coincident_bodies():
    w, R = planted(0, 1000, 7, 5, 2, 1)
    g = B.from_workload(w)
    g.accel(B.FP64)
    xb, vb = (t.clone() for t in g.get_state())
    n_merged, status, newidx = g.merge()
    assert n_merged == 0 and status == 0 and g.N == 1000
    xa, va = g.get_state()
    assert (xa == xb).all() and (va == vb).all()
    g.close()


def test_merge_after_a_drift_refreshes_the_pair_list_first():
    # the list of the last force evaluation is stale after genga_drift: genga_merge must not use it
    w, R = planted(0, 1500, 8, 0, 0, 0)
    x = w.x.copy(); v = w.v.copy()
    # bodies 10 and 11 on the same orbit a little apart, closing at 6.5e-5 AU/day: they overlap after the drift only
    x[11] = x[10] + np.array([0.0, 0.0, 5.0e-4]); v[11] = v[10] + np.array([0.0, 0.0, -6.5e-5])
    w = dataclasses.replace(w, x=x, v=v)

    def prepare(g):
        g.accel(B.FP64)
        g.drift(6.0)

    g, res, pre, orc = merged_pair(w, R, B.FP64, prepare=prepare)
    assert np.linalg.norm(pre[0][11] - pre[0][10]) < R[10] + R[11] < np.linalg.norm(w.x[11] - w.x[10])
    check_merge(g, res, pre, orc, w, R)
    assert res[0] == 1
    g.close()


def test_oversized_radius_is_reported():
    import torch
    w, R = planted(0, 1000, 9, 2, 0, 0)
    g = B.from_workload(w)
    Rb = R.copy(); Rb[5] = 0.1                                        # 0.1 AU: far beyond half its critical radius
    g.set_radii(torch.from_numpy(Rb).to(g.device))
    g.accel(B.FP64)
    _, status, _ = g.merge()
    assert status & 2
    g.close()


@pytest.mark.parametrize("n_pl", [3000, 30000])                          # 30 000: the size of the paper's runs
def test_tp2_mode_giants_accrete_planetesimals_which_do_not_collide_with_each_other(n_pl):
    """Config 3 in TP2 mode (the paper's planetesimal-driven migration runs): planetesimals moved
    into giants are accreted; overlapping planetesimals are left alone (readings R9 + R13); two giants moved onto
    each other leave one big body, and the handle's n_big follows."""
    import torch
    w = W.config(3, n_pl)
    n = w.N
    rng = np.random.default_rng(12)
    x = w.x.copy(); v = w.v.copy()
    R = np.full(n, 2.0e-5); R[:4] = [4.7e-4, 3.9e-4, 1.7e-4, 1.6e-4]          # roughly the giants' radii in AU
    ids = 4 + rng.permutation(n - 4)[:16]
    for k, i in enumerate(ids[:9]):                                     # three planetesimals into each of giants 0, 1, 2
        gidx = k % 3
        x[i] = x[gidx] + 0.5 * R[gidx] * rng.normal(size=3) / np.sqrt(3); v[i] = v[gidx] * (1 + 1e-3 * rng.normal())
    for i, j in zip(ids[9:15:2], ids[10:16:2]):                          # three overlapping small-small pairs
        x[j] = x[i] + [1.0e-5, 0.0, 0.0]
    for case_big_merge in (False, True):
        xx = x.copy()
        if case_big_merge:
            xx[3] = xx[2] + [2.0e-4, 0.0, 0.0]                          # giant 3 into giant 2
        ww = dataclasses.replace(w, x=xx, v=v)
        g = B.from_workload(ww, n_big=4)
        g.set_radii(torch.from_numpy(R).to(g.device))
        g.accel(B.FP64)
        x0, v0 = (t.cpu().numpy() for t in g.get_state())
        n_merged, status, newidx = g.merge()
        mo, xo, vo, Ro, idxo, nbo = oracle.merge_tp2(ww.m, x0, v0, R, 4)
        assert status == 0 and n_merged == 9 + case_big_merge and g.N == len(mo)
        assert nbo == 4 - case_big_merge and g.n_big == nbo
        assert (newidx.cpu().numpy() == idxo).all()
        x1, v1 = (t.cpu().numpy() for t in g.get_state())
        assert (np.abs(x1 - xo) / np.linalg.norm(xo, axis=1, keepdims=True)).max() <= 1e-14
        assert (np.abs(v1 - vo) / np.linalg.norm(vo, axis=1, keepdims=True)).max() <= 1e-14
        # the shrunk TP2 system against the oracle: forces, pairs, two steps
        p = oparams(ww, n_big=nbo)
        ao = oracle.accel(mo, xo, vo, p)
        a = g.get_accel().cpu().numpy()
        assert (np.linalg.norm(a - ao, axis=1) / np.linalg.norm(ao, axis=1)).max() <= 1e-12
        assert set(map(tuple, g.encounter_pairs().tolist())) == set(map(tuple, oracle.encounter_pairs(mo, xo, vo, p).tolist()))
        g.run(ww.dt, 2, B.FP64)
        xr, vr = oracle.run(mo, xo, vo, p, ww.dt, 2)
        x2, _ = (t.cpu().numpy() for t in g.get_state())
        assert (np.linalg.norm(x2 - xr, axis=1) / np.linalg.norm(xr, axis=1)).max() <= 1e-10
        g.close()


def test_merge_inside_the_hybrid_step():
    """Encounter mode: the pair list also holds pairs listed ahead of their zone, and the group labels share the
    scratch arrays with the merger pass; a merge between hybrid steps must leave a consistent handle."""
    w, R = planted(0, 1500, 10, 4, 1, 1)
    import torch
    kw = dict(weight_mode=1, encounter_mode=1, enc_nsub=64)
    g = B.from_workload(w, **kw)
    g.set_radii(torch.from_numpy(R).to(g.device))
    g.accel(B.FP64)
    x0, v0 = (t.cpu().numpy() for t in g.get_state())
    n_merged, status, newidx = g.merge()
    mo, xo, vo, Ro, idxo = oracle.merge(w.m, x0, v0, R)
    assert n_merged == 4 + 2 + 3 and (newidx.cpu().numpy() == idxo).all()
    g.step(w.dt, B.FP64)
    p = oparams(w, weight_mode=1)
    xr, vr = oracle.step_hybrid(mo, xo, vo, p, w.dt, 64)
    x, v = (t.cpu().numpy() for t in g.get_state())
    assert (np.linalg.norm(x - xr, axis=1) / np.linalg.norm(xr, axis=1)).max() <= 1e-10
    groups, bodies, largest, missed, st = g.encounter_stats()
    assert missed == 0 and st == 0
    g.close()


def test_degenerate_sizes_and_everything_merging_into_one_body():
    import torch
    dev = "cuda:0"
    for n in (0, 1):                                                   # empty and single-body handles
        m = torch.full((n,), 1e-7, dtype=torch.float64, device=dev)
        x = torch.ones((n, 3), dtype=torch.float64, device=dev); v = torch.zeros((n, 3), dtype=torch.float64, device=dev)
        g = B.Genga(m, x, v, device=dev)
        g.set_radii(torch.ones((n,), dtype=torch.float64, device=dev))
        n_merged, status, newidx = g.merge()
        assert n_merged == 0 and g.N == n and newidx.cpu().tolist() == list(range(n))
        g.close()
    # 700 bodies (two 512-blocks, ragged) inside one radius: a single component whatever the order of the relabelling
    w = W.config(0, 700)
    rng = np.random.default_rng(2)
    x = w.x[0] + 1.0e-5 * rng.normal(size=(700, 3)); v = w.v[0] * (1 + 1e-4 * rng.normal(size=(700, 1)))
    ww = dataclasses.replace(w, x=x, v=v)
    R = np.full(700, 2.0e-4)
    g, res, pre, orc = merged_pair(ww, R, B.FP64, n1=300.0, pair_capacity=300000)   # r_crit wide enough to list all pairs
    assert res[0] == 699 and g.N == 1 and len(orc[0]) == 1
    check_merge(g, res, pre, orc, ww, R)
    g.step(w.dt, B.FP64)                                                # a one-body system still steps (pure Kepler)
    xr, vr = oracle.step(orc[0], orc[1], orc[2], oparams(ww, n1=300.0), w.dt)
    x1, _ = (t.cpu().numpy() for t in g.get_state())
    assert np.abs(x1 - xr).max() <= 1e-12 * np.linalg.norm(xr)
    g.close()


def test_an_overflowed_pair_list_is_reported():
    w, R = planted(0, 1000, 13, 12, 0, 0)
    import torch
    g = B.from_workload(w, pair_capacity=4)
    g.set_radii(torch.from_numpy(R).to(g.device))
    g.accel(B.FP64)
    _, status, _ = g.merge()
    assert status & 1                                                  # pairs may have been missed, and the call says so
    g.close()


# ---- reading R14: collisions INSIDE the encounter integration (oracle_step_hybrid_collide) ----------------
def _collide_disc(n=400):
    """Config-0 shaped disc with: a pair on a collision course that passes THROUGH within the step (closest approach in
    mid-step, apart again at its end), a chain of three that overlaps pairwise during the step, a close pair that does
    not touch, and radii far inside the critical radii."""
    w = W.config(0, n)
    x = w.x.copy(); v = w.v.copy()
    x[7] = x[5] + [3.0e-4, 0.0, 0.0]; v[7] = v[5] + [-1.0e-4, 0.0, 0.0]            # closes 6e-4 AU in the 6-day step
    x[41] = x[40] + [2.0e-4, 1.0e-5, 0.0]; v[41] = v[40] + [-2.5e-5, 0.0, 0.0]      # 40-41 touch after ~4 days ...
    x[42] = x[40] + [-2.2e-4, 0.0, 1.0e-5]; v[42] = v[40] + [3.0e-5, 0.0, 0.0]      # ... 42 joins from the other side
    x[90] = x[88] + [1.2e-3, 6.0e-4, 0.0]; v[90] = v[88]                            # inside the zone, never touches
    R = np.full(w.N, 5.0e-5)
    return W.Workload("collide", 0, w.m.copy(), x, v, w.dt, 1), R


def test_collisions_inside_the_encounter_integration_match_the_oracle():
    import torch
    w, R = _collide_disc()
    p = oracle.Params(G=w.G, M_star=w.M_star, n1=w.n1, n2=w.n2, dt_rcrit=w.dt, pair_rule=w.pair_rule, weight_mode=1)
    vd = oracle.to_democratic(w.m, w.v, w.M_star)
    nsub = 64
    mo, xo, vo, Ro, idxo = oracle.step_hybrid_collide(w.m, w.x, vd, R, p, w.dt, nsub)
    assert len(mo) == w.N - 3 and idxo[7] == idxo[5] and idxo[40] == idxo[41] == idxo[42] and idxo[90] != idxo[88]
    # the step-end pass alone (reading R13) misses the pair that passed through
    xe, ve = oracle.step_hybrid(w.m, w.x, vd, p, w.dt, nsub=nsub)
    assert oracle.merge(w.m, xe, ve, R)[4][7] != oracle.merge(w.m, xe, ve, R)[4][5]
    # state: the merger arithmetic itself agrees to 1e-15; what is left (1.1e-12 measured on the bodies of the groups) is
    # the rounding of 256 force evaluations with refined MUFU reciprocal roots against the oracle's sqrt and divide
    for prec, tol in ((B.FP64, 5e-12), (B.FP32, 1e-7)):
        g = B.from_workload(w, weight_mode=1, encounter_mode=1, enc_nsub=nsub, enc_collide=1, mega_nmax=-1)
        g.set_radii(torch.from_numpy(R).to(g.device))
        g.step(w.dt, prec)
        assert g.encounter_stats()[3:] == (0, 0)
        n_merged, status, newidx = g.merge(prec)
        assert n_merged == 3 and status == 0 and g.N == len(mo)
        assert (newidx.cpu().numpy() == idxo).all()                       # the partition, exactly
        x, v = (t.cpu().numpy() for t in g.get_state())
        m = g.get_mass().cpu().numpy(); Rg = g.get_radii().cpu().numpy()
        assert np.abs(m / mo - 1).max() <= 1e-15 and np.abs(Rg / Ro - 1).max() <= 1e-14
        ex = np.linalg.norm(x - xo, axis=1) / np.linalg.norm(xo, axis=1)
        ev = np.linalg.norm(v - vo, axis=1) / np.linalg.norm(vo, axis=1)
        assert ex.max() <= tol and ev.max() <= tol, (prec, ex.max(), ev.max())
        # the shrunk system goes on: one more hybrid step against the oracle from its own merged state
        mo2, xo2, vo2, Ro2, idx2 = oracle.step_hybrid_collide(mo, xo, vo, Ro, p, w.dt, nsub)
        g.step(w.dt, prec)
        n2, st2, _ = g.merge(prec)
        x, v = (t.cpu().numpy() for t in g.get_state())
        assert n2 == len(mo) - len(mo2) and g.N == len(mo2)
        assert (np.linalg.norm(x - xo2, axis=1) / np.linalg.norm(xo2, axis=1)).max() <= 10 * tol
        g.close()
    # without enc_collide the same step + step-end pass leaves the pass-through pair alone (reading R13's limitation)
    g = B.from_workload(w, weight_mode=1, encounter_mode=1, enc_nsub=nsub, mega_nmax=-1)
    g.set_radii(torch.from_numpy(R).to(g.device))
    g.step(w.dt, B.FP64)
    n_merged, status, newidx = g.merge(B.FP64)
    idx = newidx.cpu().numpy()
    g.close()
    assert idx[7] != idx[5] and n_merged < 3
    # parameter checks: collisions need the RK4 substeps of an encounter-mode handle
    for bad in (dict(encounter_mode=1, enc_collide=1), dict(enc_collide=1, enc_nsub=8), dict(encounter_mode=1, enc_nsub=8, enc_collide=2)):
        with pytest.raises(Exception):
            B.from_workload(w, weight_mode=1, mega_nmax=-1, **bad).close()
