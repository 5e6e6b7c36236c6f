"""ctypes binding of the CPU FP64 oracle (``oracle/genga_oracle.c``).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package.  It imports
nothing from ``paper_2309_08217_b200`` and shares no code with the CUDA path.

Every function takes and returns numpy float64 arrays (``m[N]``, ``x[N,3]``, ``v[N,3]``) and
cites the oracle step (O1..O11, SURVEY.md section 8(c) / DESIGN.md section 3) it wraps.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "genga_oracle.c")
_HDR = os.path.join(_HERE, "genga_oracle.h")
_LIB = os.path.join(_HERE, "libgenga_oracle.so")

PAIR_MAX = 0
PAIR_MUTUAL_HILL = 1


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (C99, -O2, no fast-math, no FMA contraction, OpenMP)."""
    stale = (not os.path.exists(_LIB)
             or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR)))
    if force or stale:
        cmd = ["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
               "-Wall", "-Wextra", _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


class _Params(ctypes.Structure):
    _fields_ = [("G", ctypes.c_double), ("M_star", ctypes.c_double),
                ("n1", ctypes.c_double), ("n2", ctypes.c_double),
                ("dt_rcrit", ctypes.c_double), ("pair_rule", ctypes.c_int), ("n_big", ctypes.c_int), ("weight_mode", ctypes.c_int)]


@dataclass
class Params:
    """Mirror of ``oracle_params``.  Defaults: Gaussian units, the configs' r_crit rule."""
    G: float = 0.01720209895 ** 2          # O0: k^2, AU^3 Msun^-1 day^-2
    M_star: float = 1.0
    n1: float = 3.0
    n2: float = 0.0                        # BASELINE.json configs: "3 mutual Hill radii"
    dt_rcrit: float = 0.0
    pair_rule: int = PAIR_MUTUAL_HILL
    n_big: int = -1                        # TP2 mode: pairs interact iff i < n_big or j < n_big
    weight_mode: int = 0                   # 0: W = K; 1: W = K - r dK/dr (reading R10)

    def c(self) -> _Params:
        return _Params(self.G, self.M_star, self.n1, self.n2, self.dt_rcrit, int(self.pair_rule), int(self.n_big),
                       int(self.weight_mode))


_lib = None
_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int)
_pp = ctypes.POINTER(_Params)


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        L.oracle_changeover.restype = ctypes.c_double
        L.oracle_changeover.argtypes = [ctypes.c_double, ctypes.c_double]
        L.oracle_step_hybrid.restype = ctypes.c_int
        L.oracle_step_hybrid.argtypes = [ctypes.c_int, _dp, _dp, _dp, _pp, ctypes.c_double, ctypes.c_int]
        L.oracle_step_hybrid_bs.restype = ctypes.c_int
        L.oracle_step_hybrid_bs.argtypes = [ctypes.c_int, _dp, _dp, _dp, _pp, ctypes.c_double, ctypes.c_double,
                                            ctypes.POINTER(ctypes.c_longlong)]
        L.oracle_level_weight.restype = ctypes.c_double
        L.oracle_level_weight.argtypes = [ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_int, ctypes.c_double]
        L.oracle_step_multilevel.restype = ctypes.c_int
        L.oracle_step_multilevel.argtypes = [ctypes.c_int, _dp, _dp, _dp, _pp, ctypes.c_double, ctypes.c_int, ctypes.c_int,
                                             ctypes.c_double, ctypes.c_double, ctypes.POINTER(ctypes.c_longlong)]
        L.oracle_weight.restype = ctypes.c_double
        L.oracle_weight.argtypes = [ctypes.c_double, ctypes.c_double, ctypes.c_int]
        L.oracle_pair_rcrit.restype = ctypes.c_double
        L.oracle_pair_rcrit.argtypes = [_pp] + [ctypes.c_double] * 8
        L.oracle_to_democratic.argtypes = [ctypes.c_int, _dp, _dp, ctypes.c_double]
        L.oracle_to_heliocentric.argtypes = [ctypes.c_int, _dp, _dp, ctypes.c_double]
        L.oracle_rcrit.argtypes = [ctypes.c_int, _dp, _dp, _dp, _pp, _dp, _dp, _dp]
        L.oracle_accel.argtypes = [ctypes.c_int, _dp, _dp, _dp, _pp, _dp]
        L.oracle_encounter_pairs.argtypes = [ctypes.c_int, _dp, _dp, _dp, _pp, _ip, ctypes.c_int, _ip]
        L.oracle_kick.argtypes = [ctypes.c_int, _dp, _dp, _dp, _pp, ctypes.c_double, _dp]
        L.oracle_sunkick.argtypes = [ctypes.c_int, _dp, _dp, _dp, _pp, ctypes.c_double]
        L.oracle_kepler_drift_one.restype = ctypes.c_int
        L.oracle_kepler_drift_one.argtypes = [ctypes.c_double, ctypes.c_double, _dp, _dp]
        L.oracle_drift.restype = ctypes.c_int
        L.oracle_drift.argtypes = [ctypes.c_int, _dp, _dp, _pp, ctypes.c_double]
        L.oracle_step.restype = ctypes.c_int
        L.oracle_step.argtypes = [ctypes.c_int, _dp, _dp, _dp, _pp, ctypes.c_double]
        L.oracle_run.restype = ctypes.c_int
        L.oracle_run.argtypes = [ctypes.c_int, _dp, _dp, _dp, _pp, ctypes.c_double, ctypes.c_int]
        L.oracle_energy_angmom.argtypes = [ctypes.c_int, _dp, _dp, _dp, _pp, _dp, _dp]
        L.oracle_merge.restype = ctypes.c_int
        L.oracle_merge.argtypes = [ctypes.c_int, _dp, _dp, _dp, _dp, _ip]
        L.oracle_step_hybrid_collide.restype = ctypes.c_int
        L.oracle_step_hybrid_collide.argtypes = [ctypes.c_int, _dp, _dp, _dp, _dp, _pp, ctypes.c_double, ctypes.c_int, _ip]
        L.oracle_merge_tp2.restype = ctypes.c_int
        L.oracle_merge_tp2.argtypes = [ctypes.c_int, _dp, _dp, _dp, _dp, _ip, ctypes.c_int, _ip]
        L.oracle_num_threads.restype = ctypes.c_int
        _lib = L
    return _lib


def _a(arr, shape=None) -> np.ndarray:
    out = np.ascontiguousarray(arr, dtype=np.float64)
    if shape is not None:
        out = out.reshape(shape)
    return out


def _p(arr: np.ndarray):
    return arr.ctypes.data_as(_dp)


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def changeover(r: float, rcrit: float) -> float:
    """O4 (reading G1)."""
    return float(lib().oracle_changeover(float(r), float(rcrit)))


def weight(r: float, rcrit: float, mode: int) -> float:
    """Pair weight W: mode 0 = K, mode 1 = K - r dK/dr (reading R10)."""
    return float(lib().oracle_weight(float(r), float(rcrit), int(mode)))


def to_democratic(m, v, M_star: float = 1.0) -> np.ndarray:
    """O1: heliocentric -> stored barycentric velocities (returns a new array)."""
    m = _a(m); v = _a(v).copy()
    lib().oracle_to_democratic(len(m), _p(m), _p(v), float(M_star))
    return v


def to_heliocentric(m, v, M_star: float = 1.0) -> np.ndarray:
    """O1 inverse."""
    m = _a(m); v = _a(v).copy()
    lib().oracle_to_heliocentric(len(m), _p(m), _p(v), float(M_star))
    return v


def rcrit(m, x, v, p: Params):
    """O2 (Eq. 1): returns (r_crit, a, v_K) per body."""
    m = _a(m); x = _a(x); v = _a(v)
    n = len(m)
    rc = np.empty(n); sa = np.empty(n); vk = np.empty(n)
    c = p.c()
    lib().oracle_rcrit(n, _p(m), _p(x), _p(v), ctypes.byref(c), _p(rc), _p(sa), _p(vk))
    return rc, sa, vk


def pair_rcrit(p: Params, mi, mj, rci, rcj, ai, aj, vki, vkj) -> float:
    """O3 (reading G2)."""
    c = p.c()
    return float(lib().oracle_pair_rcrit(ctypes.byref(c), mi, mj, rci, rcj, ai, aj, vki, vkj))


def accel(m, x, v, p: Params) -> np.ndarray:
    """O2-O5: the K-weighted all-pairs acceleration, shape (N, 3)."""
    m = _a(m); x = _a(x); v = _a(v)
    a = np.zeros((len(m), 3))
    c = p.c()
    lib().oracle_accel(len(m), _p(m), _p(x), _p(v), ctypes.byref(c), _p(a))
    return a


def encounter_pairs(m, x, v, p: Params) -> np.ndarray:
    """O6: int array (count, 2) of pairs i<j with r_ij < r_crit,ij."""
    m = _a(m); x = _a(x); v = _a(v)
    c = p.c()
    cnt = ctypes.c_int(0)
    cap = 1024
    while True:
        buf = np.zeros((cap, 2), dtype=np.int32)
        lib().oracle_encounter_pairs(len(m), _p(m), _p(x), _p(v), ctypes.byref(c),
                                     buf.ctypes.data_as(_ip), cap, ctypes.byref(cnt))
        if cnt.value <= cap:
            return buf[:cnt.value].copy()
        cap = cnt.value


def accel_subset(m, x, v, p: Params, sel) -> np.ndarray:
    """O5 for the bodies ``sel`` only (sampled outputs at large N), shape (len(sel), 3)."""
    m = _a(m); x = _a(x); v = _a(v)
    sel = np.ascontiguousarray(sel, dtype=np.int32)
    a = np.zeros((len(sel), 3))
    c = p.c()
    lib().oracle_accel_subset(len(m), _p(m), _p(x), _p(v), ctypes.byref(c), len(sel),
                              sel.ctypes.data_as(_ip), _p(a))
    return a


def encounter_pairs_subset(m, x, v, p: Params, sel) -> set:
    """O6 restricted to pairs touching a body of ``sel``: a set of (i, j), i < j."""
    m = _a(m); x = _a(x); v = _a(v)
    sel = np.ascontiguousarray(sel, dtype=np.int32)
    c = p.c()
    cnt = ctypes.c_int(0)
    cap = 4096
    while True:
        buf = np.zeros((cap, 2), dtype=np.int32)
        lib().oracle_encounter_pairs_subset(len(m), _p(m), _p(x), _p(v), ctypes.byref(c), len(sel),
                                            sel.ctypes.data_as(_ip), buf.ctypes.data_as(_ip), cap, ctypes.byref(cnt))
        if cnt.value <= cap:
            return set(map(tuple, buf[:cnt.value].tolist()))
        cap = cnt.value


def kick(m, x, v, p: Params, tau: float):
    """O7: returns (v + tau a, a)."""
    m = _a(m); x = _a(x); v = _a(v).copy()
    a = np.zeros((len(m), 3))
    c = p.c()
    lib().oracle_kick(len(m), _p(m), _p(x), _p(v), ctypes.byref(c), float(tau), _p(a))
    return v, a


def sunkick(m, x, v, p: Params, tau: float) -> np.ndarray:
    """O8: returns x + tau (sum m v)/M_star."""
    m = _a(m); x = _a(x).copy(); v = _a(v)
    c = p.c()
    lib().oracle_sunkick(len(m), _p(m), _p(x), _p(v), ctypes.byref(c), float(tau))
    return x


def kepler_drift_one(mu: float, dt: float, x, v):
    """O9 for one body: returns (x', v')."""
    x = _a(x).copy(); v = _a(v).copy()
    rc = lib().oracle_kepler_drift_one(float(mu), float(dt), _p(x), _p(v))
    if rc != 0:
        raise RuntimeError("oracle Kepler solve did not converge")
    return x, v


def drift(x, v, p: Params, dt: float):
    """O9 for all bodies: returns (x', v')."""
    x = _a(x).copy(); v = _a(v).copy()
    c = p.c()
    rc = lib().oracle_drift(x.shape[0], _p(x), _p(v), ctypes.byref(c), float(dt))
    if rc != 0:
        raise RuntimeError("oracle Kepler solve did not converge")
    return x, v


def step(m, x, v, p: Params, dt: float):
    """O10: one K(dt/2) S(dt/2) D(dt) S(dt/2) K(dt/2) step; returns (x', v')."""
    m = _a(m); x = _a(x).copy(); v = _a(v).copy()
    c = p.c()
    if lib().oracle_step(len(m), _p(m), _p(x), _p(v), ctypes.byref(c), float(dt)) != 0:
        raise RuntimeError("oracle Kepler solve did not converge")
    return x, v


def step_hybrid(m, x, v, p: Params, dt: float, nsub: int = 2000):
    """NEXT-1 (reading R11): one hybrid step with the encounter complement; returns (x', v')."""
    m = _a(m); x = _a(x).copy(); v = _a(v).copy()
    c = p.c()
    rc = lib().oracle_step_hybrid(len(m), _p(m), _p(x), _p(v), ctypes.byref(c), float(dt), int(nsub))
    if rc != 0:
        raise ValueError("oracle_step_hybrid needs weight_mode = 1 and nsub >= 1")
    return x, v


def step_hybrid_bs(m, x, v, p: Params, dt: float, tol: float = 1.0e-13, stats: bool = False):
    """NEXT-1 (readings R11, R15): the hybrid step with the A-flow integrated by Gragg-Bulirsch-Stoer extrapolation to the
    relative tolerance tol (all bodies as one system); returns (x', v') [, (accepted, rejected, right-hand sides)]."""
    m = _a(m); x = _a(x).copy(); v = _a(v).copy()
    c = p.c()
    st = (ctypes.c_longlong * 3)()
    rc = lib().oracle_step_hybrid_bs(len(m), _p(m), _p(x), _p(v), ctypes.byref(c), float(dt), float(tol), st)
    if rc != 0:
        raise ValueError("oracle_step_hybrid_bs: needs weight_mode = 1 and tol > 0, or the step size collapsed")
    return (x, v, tuple(int(q) for q in st)) if stats else (x, v)


def level_weight(r: float, rcrit: float, l: int, L: int, F: float) -> float:
    """Reading R16: shell weight of level l (l < L: W_l - W_{l-1}; l == L: the Bulirsch-Stoer remainder 1 - W_{L-1})."""
    return float(lib().oracle_level_weight(float(r), float(rcrit), int(l), int(L), float(F)))


def step_multilevel(m, x, v, p: Params, dt: float, L: int, S: int, F: float, tol: float = 1.0e-13, stats: bool = False):
    """NEXT-3 (reading R16): the hybrid step with L changeover levels, S sub-steps per level and radius ratio F."""
    m = _a(m); x = _a(x).copy(); v = _a(v).copy()
    c = p.c()
    st = (ctypes.c_longlong * 3)()
    rc = lib().oracle_step_multilevel(len(m), _p(m), _p(x), _p(v), ctypes.byref(c), float(dt), int(L), int(S), float(F), float(tol), st)
    if rc != 0:
        raise ValueError("oracle_step_multilevel: needs weight_mode = 1, tol > 0, L >= 1, S >= 1, F > 1 (or the step size collapsed)")
    return (x, v, tuple(int(q) for q in st)) if stats else (x, v)


def run(m, x, v, p: Params, dt: float, nsteps: int):
    """nsteps steps with merged half-kicks (reading R7); returns (x', v')."""
    m = _a(m); x = _a(x).copy(); v = _a(v).copy()
    c = p.c()
    if lib().oracle_run(len(m), _p(m), _p(x), _p(v), ctypes.byref(c), float(dt), int(nsteps)) != 0:
        raise RuntimeError("oracle Kepler solve did not converge")
    return x, v


def energy_angmom(m, x, v, p: Params):
    """O11: returns (E, L[3])."""
    m = _a(m); x = _a(x); v = _a(v)
    c = p.c()
    E = ctypes.c_double(0.0)
    L = np.zeros(3)
    lib().oracle_energy_angmom(len(m), _p(m), _p(x), _p(v), ctypes.byref(c), ctypes.byref(E), _p(L))
    return float(E.value), L


def merge(m, x, v, R):
    """NEXT-4, reading R13: step-end perfect mergers.  Returns (m', x', v', R', newidx):
    the closed-up arrays and, per old body, the new index of the body it is now part of."""
    m = _a(m).copy(); x = _a(x).copy(); v = _a(v).copy(); R = _a(R).copy()
    newidx = np.zeros(len(m), dtype=np.int32)
    n = lib().oracle_merge(len(m), _p(m), _p(x), _p(v), _p(R), newidx.ctypes.data_as(_ip))
    return m[:n].copy(), x[:n].copy(), v[:n].copy(), R[:n].copy(), newidx


def merge_tp2(m, x, v, R, n_big: int):
    """oracle.merge under TP2 mode's pair rule (readings R9, R13): only pairs that involve one of the first n_big bodies
    can collide.  Returns (m', x', v', R', newidx, n_big')."""
    m = _a(m).copy(); x = _a(x).copy(); v = _a(v).copy(); R = _a(R).copy()
    newidx = np.zeros(len(m), dtype=np.int32)
    nb = ctypes.c_int(0)
    n = lib().oracle_merge_tp2(len(m), _p(m), _p(x), _p(v), _p(R), newidx.ctypes.data_as(_ip), int(n_big), ctypes.byref(nb))
    return m[:n].copy(), x[:n].copy(), v[:n].copy(), R[:n].copy(), newidx, int(nb.value)


def step_hybrid_collide(m, x, v, R, p: Params, dt: float, nsub: int):
    """Reading R14 (oracle only so far): hybrid step with the collision pass after every substep of the A-flow.
    Returns (m', x', v', R', newidx)."""
    m = _a(m).copy(); x = _a(x).copy(); v = _a(v).copy(); R = _a(R).copy()
    newidx = np.zeros(len(m), dtype=np.int32)
    c = p.c()
    n = lib().oracle_step_hybrid_collide(len(m), _p(m), _p(x), _p(v), _p(R), ctypes.byref(c), float(dt), int(nsub),
                                         newidx.ctypes.data_as(_ip))
    if n < 0:
        raise ValueError("step_hybrid_collide needs weight_mode = 1 and nsub >= 1")
    return m[:n].copy(), x[:n].copy(), v[:n].copy(), R[:n].copy(), newidx
