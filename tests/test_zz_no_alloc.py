"""genga_energy_angmom_static (include/genga.h, csrc/noalloc.cu): the one entry point that allocates nothing -- its
scratch is a file-scope __device__ array of the library.  Checked against the existing path (genga_energy_angmom of a
handle) within the tolerance of the energy parity tests (1e-13), on calls in a row that share the array, and against
the oracle.  This file is collected last on purpose (the suite runs with pytest -x); it must pass alone as well."""
import numpy as np
import pytest

import oracle
from paper_2309_08217_b200 import binding as B
from paper_2309_08217_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-13          # tests/test_gpu_parity.py: test_energy_angmom_parity


def _state_on_device(w):
    """(m, x, v democratic) as device tensors, and (E, L) of the existing path, for one workload."""
    g = B.from_workload(w)
    x, v = g.get_state(heliocentric_v=False)
    m = g.get_mass()
    E, L = g.energy_angmom()
    g.synchronize()
    x, v, m = x.clone(), v.clone(), m.clone()
    g.close()
    return m, x, v, E, L


def _static(torch, w, m, x, v, out4):
    s = torch.cuda.current_stream()
    B.energy_angmom_static(w.N, m.data_ptr(), x.data_ptr(), v.data_ptr(), w.G, w.M_star, s.cuda_stream, out4.data_ptr())
    s.synchronize()
    r = out4.cpu().numpy()
    return float(r[0]), r[1:4].copy()


def test_static_entry_point_matches_the_handle_path_on_calls_in_a_row():
    import torch
    B.load()
    # sizes: a multiple of 128, ragged ones, one smaller than its predecessor (the shared array then still holds
    # records and partials of the larger call), tiny ones
    cases = [W.config(0), W.config(3, 2500), W.config(0, 333), W.config(2, 1500), W.config(0, 1), W.config(0, 2), W.config(4, 9000)]
    ref = [_state_on_device(w) for w in cases]
    out4 = torch.full((4,), float("nan"), dtype=torch.float64, device="cuda:0")
    first = []
    for w, (m, x, v, E, L) in zip(cases, ref):
        Es, Ls = _static(torch, w, m, x, v, out4)
        first.append((Es, Ls))
        assert abs(Es / E - 1) <= TOL, (w.name, w.N, Es, E)
        assert np.linalg.norm(Ls - L) <= TOL * np.linalg.norm(L), (w.name, w.N)
        vd = oracle.to_democratic(w.m, w.v, w.M_star)
        Eo, Lo = oracle.energy_angmom(w.m, w.x, vd, oracle.Params(G=w.G, M_star=w.M_star, n1=w.n1, n2=w.n2, dt_rcrit=w.dt, pair_rule=w.pair_rule))
        assert abs(Es / Eo - 1) <= TOL and np.linalg.norm(Ls - Lo) <= TOL * np.linalg.norm(Lo), (w.name, w.N)
    # the same calls again, back to back on one stream without a synchronisation in between, in reverse order: every call
    # must give what it gave before, bit for bit (fixed summation order; nothing of a neighbour's scratch may leak in),
    # and no device memory may have been taken meanwhile
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    outs = [torch.empty(4, dtype=torch.float64, device="cuda:0") for _ in cases]
    free0, _ = torch.cuda.mem_get_info()
    s = torch.cuda.current_stream()
    for k in reversed(range(len(cases))):
        w, (m, x, v, _, _) = cases[k], ref[k]
        B.energy_angmom_static(w.N, m.data_ptr(), x.data_ptr(), v.data_ptr(), w.G, w.M_star, s.cuda_stream, outs[k].data_ptr())
    s.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, (free0, free1)
    for k, o in enumerate(outs):
        r = o.cpu().numpy()
        assert r[0] == first[k][0] and np.array_equal(r[1:4], first[k][1]), (cases[k].name, cases[k].N)


def test_static_entry_point_rejects_what_it_cannot_hold():
    import torch
    B.load()
    out4 = torch.zeros(4, dtype=torch.float64, device="cuda:0")
    buf = torch.zeros(8, dtype=torch.float64, device="cuda:0")
    s = torch.cuda.current_stream().cuda_stream
    with pytest.raises(B.GengaError) as ei:                    # beyond the fixed size: refused before anything is launched
        B.energy_angmom_static(B.STATIC_NMAX + 1, buf.data_ptr(), buf.data_ptr(), buf.data_ptr(), 1.0, 1.0, s, out4.data_ptr())
    assert ei.value.code == B.ELIMIT and "GENGA_STATIC_NMAX" in str(ei.value) and str(B.STATIC_NMAX) in str(ei.value)
    for bad in (dict(N=-1), dict(M_star=0.0), dict(m=0), dict(out=0)):
        with pytest.raises(B.GengaError) as ei:
            B.energy_angmom_static(bad.get("N", 2), bad.get("m", buf.data_ptr()), buf.data_ptr(), buf.data_ptr(), 1.0,
                                   bad.get("M_star", 1.0), s, bad.get("out", out4.data_ptr()))
        assert ei.value.code == B.EINVAL
    B.energy_angmom_static(0, 0, 0, 0, 1.0, 1.0, s, out4.data_ptr())       # no bodies: E = 0, L = 0
    torch.cuda.synchronize()
    assert np.array_equal(out4.cpu().numpy(), np.zeros(4))
    # the largest size it takes runs (and uses every record of the array): two bodies' worth of physics, the rest massless
    n = B.STATIC_NMAX
    w = W.config(0, 2)
    m = torch.zeros(n, dtype=torch.float64, device="cuda:0"); m[:2] = torch.from_numpy(w.m).cuda()
    x = torch.ones(n, 3, dtype=torch.float64, device="cuda:0") * torch.arange(1, n + 1, dtype=torch.float64, device="cuda:0")[:, None]
    v = torch.zeros(n, 3, dtype=torch.float64, device="cuda:0")
    vd = oracle.to_democratic(w.m, w.v, w.M_star)
    x[:2] = torch.from_numpy(w.x).cuda(); v[:2] = torch.from_numpy(vd).cuda()
    B.energy_angmom_static(n, m.data_ptr(), x.data_ptr(), v.data_ptr(), w.G, w.M_star, s, out4.data_ptr())
    torch.cuda.synchronize()
    Eo, Lo = oracle.energy_angmom(w.m, w.x, vd, oracle.Params(G=w.G, M_star=w.M_star))
    r = out4.cpu().numpy()
    assert abs(r[0] / Eo - 1) <= TOL and np.linalg.norm(r[1:4] - Lo) <= TOL * np.linalg.norm(Lo)
