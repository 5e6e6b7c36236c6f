"""Thin ctypes binding of ``libgenga_b200.so`` (include/genga.h).  Argument marshalling only:
every step of the path runs in the library's CUDA kernels.  PyTorch provides device memory and
the stream; there is NO CPU fallback -- ``load()`` raises if the library is missing.

Function names follow the C ABI (``genga_kick`` -> ``Genga.kick``).  Citations are in genga.h.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgenga_b200.so")

FP64 = 0
FP32 = 1
PAIR_MAX = 0
PAIR_MUTUAL_HILL = 1

OK, EINVAL, ENOMEM, ECAPACITY, ECUDA, ENOCONV, ELIMIT = 0, -1, -2, -3, -4, -5, -6
STATIC_NMAX = 131072          # GENGA_STATIC_NMAX of include/genga.h

# every symbol include/genga.h declares (tests check the library exports all of them)
SYMBOLS = [
    "genga_default_params", "genga_workspace_bytes", "genga_create", "genga_destroy",
    "genga_set_state", "genga_set_state_host", "genga_resort", "genga_kick", "genga_accel", "genga_drift",
    "genga_sunkick", "genga_step", "genga_run", "genga_leapfrog", "genga_encounter_pairs", "genga_energy_angmom",
    "genga_get_state", "genga_get_state_host", "genga_get_accel", "genga_get_rcrit",
    "genga_set_radii", "genga_get_radii", "genga_merge", "genga_get_mass", "genga_num_bodies", "genga_num_big_bodies",
    "genga_nearfield_stats", "genga_encounter_stats", "genga_encounter_work", "genga_set_profiling", "genga_kernel_time", "genga_launch_count",
    "genga_synchronize", "genga_strerror", "genga_last_cuda_error", "genga_version",
    "genga_peak_probe", "genga_set_tuning", "genga_autotune", "genga_num_variants", "genga_variant_name",
    "genga_energy_angmom_static", "genga_static_last_error",
]


class GengaParams(ctypes.Structure):
    _fields_ = [
        ("G", ctypes.c_double), ("M_star", ctypes.c_double),
        ("n1", ctypes.c_double), ("n2", ctypes.c_double), ("dt_rcrit", ctypes.c_double),
        ("pair_rule", ctypes.c_int), ("v_is_heliocentric", ctypes.c_int),
        ("lambda_near", ctypes.c_double), ("near_floor", ctypes.c_double),
        ("stream", ctypes.c_void_p), ("workspace", ctypes.c_void_p), ("workspace_bytes", ctypes.c_size_t),
        ("pair_capacity", ctypes.c_int), ("cand_capacity", ctypes.c_int), ("resort_every", ctypes.c_int),
        ("chunk", ctypes.c_int), ("mega_nmax", ctypes.c_int), ("lean_nmax", ctypes.c_int), ("lean_min_evals", ctypes.c_int), ("n_big", ctypes.c_int), ("weight_mode", ctypes.c_int), ("no_fused_step", ctypes.c_int),
        ("encounter_mode", ctypes.c_int), ("enc_nsub", ctypes.c_int), ("enc_list_scale", ctypes.c_double), ("enc_list_vfactor", ctypes.c_double), ("enc_tol", ctypes.c_double), ("enc_collide", ctypes.c_int), ("enc_levels", ctypes.c_int), ("enc_substeps", ctypes.c_int), ("enc_level_ratio", ctypes.c_double),
    ]


class GengaError(RuntimeError):
    def __init__(self, code: int, what: str):
        self.code = code
        super().__init__(what)


_lib = None


def load() -> ctypes.CDLL:
    """dlopen the CUDA library; raise (no fallback) if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise GengaError(ECUDA, f"{LIB_PATH} is missing: build it with `python -m paper_2309_08217_b200.build` "
                                "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    vp, dp, ip = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)
    pp = ctypes.POINTER(GengaParams)
    llp = ctypes.POINTER(ctypes.c_longlong)
    L.genga_default_params.argtypes = [pp]; L.genga_default_params.restype = None
    L.genga_workspace_bytes.argtypes = [ctypes.c_int, pp]; L.genga_workspace_bytes.restype = ctypes.c_size_t
    L.genga_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int, vp, vp, vp, pp]
    L.genga_destroy.argtypes = [vp]
    L.genga_set_state.argtypes = [vp, vp, vp, vp]
    L.genga_set_state_host.argtypes = [vp, vp, vp, vp]
    L.genga_kick.argtypes = [vp, ctypes.c_double, ctypes.c_int]
    L.genga_accel.argtypes = [vp, ctypes.c_int]
    L.genga_resort.argtypes = [vp]
    L.genga_drift.argtypes = [vp, ctypes.c_double]
    L.genga_sunkick.argtypes = [vp, ctypes.c_double]
    L.genga_step.argtypes = [vp, ctypes.c_double, ctypes.c_int]
    L.genga_run.argtypes = [vp, ctypes.c_double, ctypes.c_int, ctypes.c_int]
    L.genga_leapfrog.argtypes = [vp, ctypes.c_double, ctypes.c_int, ctypes.c_int]
    L.genga_encounter_pairs.argtypes = [vp, vp, ctypes.c_int, ip]
    L.genga_energy_angmom.argtypes = [vp, dp, dp]
    L.genga_get_state.argtypes = [vp, vp, vp, ctypes.c_int]
    L.genga_get_state_host.argtypes = [vp, vp, vp, ctypes.c_int]
    L.genga_get_accel.argtypes = [vp, vp]
    L.genga_get_rcrit.argtypes = [vp, vp]
    L.genga_set_radii.argtypes = [vp, vp]
    L.genga_get_radii.argtypes = [vp, vp]
    L.genga_merge.argtypes = [vp, ctypes.c_int, vp, ip, ip]
    L.genga_get_mass.argtypes = [vp, vp]
    L.genga_num_bodies.argtypes = [vp]
    L.genga_num_big_bodies.argtypes = [vp]
    L.genga_nearfield_stats.argtypes = [vp, llp, ip]
    L.genga_encounter_stats.argtypes = [vp, ip, ip, ip, ip, ip]
    L.genga_encounter_work.argtypes = [vp, llp, ip, ip]
    L.genga_set_profiling.argtypes = [vp, ctypes.c_int]
    L.genga_kernel_time.argtypes = [vp, ctypes.c_int, dp, llp, ctypes.c_int]
    L.genga_launch_count.argtypes = [vp]; L.genga_launch_count.restype = ctypes.c_longlong
    L.genga_synchronize.argtypes = [vp]
    L.genga_strerror.argtypes = [ctypes.c_int]; L.genga_strerror.restype = ctypes.c_char_p
    L.genga_last_cuda_error.argtypes = []; L.genga_last_cuda_error.restype = ctypes.c_char_p
    L.genga_version.argtypes = []; L.genga_version.restype = ctypes.c_char_p
    L.genga_peak_probe.argtypes = [ctypes.c_int, ctypes.c_int, vp, dp, dp]
    L.genga_set_tuning.argtypes = [vp, ctypes.c_int, ctypes.c_int]
    L.genga_autotune.argtypes = [vp, ctypes.c_int, ip, dp]
    L.genga_num_variants.argtypes = [ctypes.c_int]
    L.genga_variant_name.argtypes = [ctypes.c_int, ctypes.c_int]; L.genga_variant_name.restype = ctypes.c_char_p
    L.genga_energy_angmom_static.argtypes = [ctypes.c_int, vp, vp, vp, ctypes.c_double, ctypes.c_double, vp, vp]
    L.genga_static_last_error.argtypes = []; L.genga_static_last_error.restype = ctypes.c_char_p
    for name in SYMBOLS:
        fn = getattr(L, name)
        if fn.restype is ctypes.c_int and name not in ("genga_launch_count",):
            fn.restype = ctypes.c_int
    _lib = L
    return L


def _check(code: int, what: str) -> int:
    if code in (OK,):
        return code
    L = load()
    msg = L.genga_strerror(code).decode()
    if code == ECUDA:
        msg += ": " + L.genga_last_cuda_error().decode()
    raise GengaError(code, f"{what}: {msg}")


def default_params() -> GengaParams:
    p = GengaParams()
    load().genga_default_params(ctypes.byref(p))
    return p


def peak_probe(which: int, iters: int = 4096, stream: int = 0):
    """genga_peak_probe: returns (lane-ops per second, milliseconds)."""
    ops, ms = ctypes.c_double(0), ctypes.c_double(0)
    _check(load().genga_peak_probe(which, iters, ctypes.c_void_p(stream), ctypes.byref(ops), ctypes.byref(ms)),
           "genga_peak_probe")
    return ops.value, ms.value


def energy_angmom_static(N: int, m_ptr: int, x_ptr: int, v_ptr: int, G: float, M_star: float, stream: int, out4_ptr: int) -> None:
    """genga_energy_angmom_static (the entry point that allocates nothing): raw DEVICE addresses in, (E, Lx, Ly, Lz)
    written to the DEVICE address out4_ptr, asynchronously on `stream`.  Marshalling only: this wrapper allocates nothing
    either.  Raises GengaError (code ELIMIT for N > STATIC_NMAX) with the library's own text."""
    L = load()
    code = L.genga_energy_angmom_static(int(N), ctypes.c_void_p(m_ptr), ctypes.c_void_p(x_ptr), ctypes.c_void_p(v_ptr),
                                        float(G), float(M_star), ctypes.c_void_p(stream), ctypes.c_void_p(out4_ptr))
    if code != OK:
        raise GengaError(code, f"genga_energy_angmom_static: {L.genga_strerror(code).decode()}: {L.genga_static_last_error().decode()}")


def num_variants(key: int) -> int:
    return int(load().genga_num_variants(int(key)))


def variant_name(key: int, value: int) -> str:
    return load().genga_variant_name(int(key), int(value)).decode()


def _dptr(t):
    return ctypes.c_void_p(t.data_ptr()) if t is not None else ctypes.c_void_p(0)


@dataclass
class NearfieldStats:
    candidates: int
    overflowed: bool


class Genga:
    """One handle.  ``m``, ``x``, ``v`` are CUDA float64 tensors of shape (N,), (N,3), (N,3)."""

    def __init__(self, m, x, v, *, G=None, M_star=1.0, n1=3.0, n2=0.0, dt_rcrit=0.0,
                 pair_rule=PAIR_MUTUAL_HILL, v_is_heliocentric=True, lambda_near=0.0, near_floor=-1.0,
                 pair_capacity=0, cand_capacity=0, resort_every=0, chunk=0, mega_nmax=0, lean_nmax=0, lean_min_evals=0, n_big=-1, weight_mode=0, no_fused_step=False,
                 encounter_mode=0, enc_nsub=0, enc_list_scale=0.0, enc_list_vfactor=0.0, enc_tol=0.0, enc_collide=0, enc_levels=0, enc_substeps=0, enc_level_ratio=0.0, stream=None, device=None):
        import torch
        self._torch = torch
        self._L = load()
        if not torch.cuda.is_available():
            raise GengaError(ECUDA, "no CUDA device: the GENGA hot path has no CPU fallback")
        self.device = torch.device(device if device is not None else (m.device if m is not None else "cuda:0"))
        self.N = int(m.shape[0])
        p = default_params()
        if G is not None:
            p.G = float(G)
        p.M_star, p.n1, p.n2, p.dt_rcrit = float(M_star), float(n1), float(n2), float(dt_rcrit)
        p.pair_rule, p.v_is_heliocentric = int(pair_rule), int(bool(v_is_heliocentric))
        p.lambda_near, p.near_floor = float(lambda_near), float(near_floor)
        p.pair_capacity, p.cand_capacity = int(pair_capacity), int(cand_capacity)
        p.resort_every = int(resort_every)
        p.no_fused_step = int(bool(no_fused_step))
        p.encounter_mode = int(encounter_mode); p.enc_nsub = int(enc_nsub); p.enc_list_scale = float(enc_list_scale); p.enc_list_vfactor = float(enc_list_vfactor); p.enc_tol = float(enc_tol); p.enc_collide = int(enc_collide); p.enc_levels = int(enc_levels); p.enc_substeps = int(enc_substeps); p.enc_level_ratio = float(enc_level_ratio)
        p.n_big = int(n_big)
        p.chunk = int(chunk)
        p.mega_nmax = int(mega_nmax)
        p.lean_nmax = int(lean_nmax)
        p.lean_min_evals = int(lean_min_evals)
        p.weight_mode = int(weight_mode)
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        p.stream = ctypes.c_void_p(self._stream.cuda_stream)
        nbytes = self._L.genga_workspace_bytes(self.N, ctypes.byref(p))
        with torch.cuda.device(self.device):
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = (self._ws.data_ptr() + 255) // 256 * 256
        p.workspace, p.workspace_bytes = ctypes.c_void_p(base), nbytes
        self.params = p
        self._h = ctypes.c_void_p(0)
        m, x, v = (self._as_dev(t) for t in (m, x, v))
        with torch.cuda.device(self.device):
            _check(self._L.genga_create(ctypes.byref(self._h), self.N, _dptr(m), _dptr(x), _dptr(v), ctypes.byref(p)),
                   "genga_create")
        self._keep = (m, x, v)

    def _as_dev(self, t):
        if t is None:
            return None
        torch = self._torch
        return t.to(device=self.device, dtype=torch.float64).contiguous()

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self._L.genga_destroy(self._h)
            self._h = ctypes.c_void_p(0)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- state ---------------------------------------------------------------------------------
    def set_state(self, m=None, x=None, v=None):
        m, x, v = (self._as_dev(t) for t in (m, x, v))
        _check(self._L.genga_set_state(self._h, _dptr(m), _dptr(x), _dptr(v)), "genga_set_state")
        self._keep = (m, x, v)

    def set_state_host(self, m=None, x=None, v=None):
        """m, x, v: CPU float64 tensors (pinned memory keeps the copies asynchronous)."""
        _check(self._L.genga_set_state_host(self._h, _dptr(m), _dptr(x), _dptr(v)), "genga_set_state_host")
        self._keep = (m, x, v)

    def get_state(self, heliocentric_v=False):
        torch = self._torch
        x = torch.empty((self.N, 3), dtype=torch.float64, device=self.device)
        v = torch.empty((self.N, 3), dtype=torch.float64, device=self.device)
        _check(self._L.genga_get_state(self._h, _dptr(x), _dptr(v), int(heliocentric_v)), "genga_get_state")
        return x, v

    def get_state_host(self, x_out, v_out, heliocentric_v=False):
        _check(self._L.genga_get_state_host(self._h, _dptr(x_out), _dptr(v_out), int(heliocentric_v)),
               "genga_get_state_host")
        return x_out, v_out

    def get_accel(self):
        torch = self._torch
        a = torch.empty((self.N, 3), dtype=torch.float64, device=self.device)
        _check(self._L.genga_get_accel(self._h, _dptr(a)), "genga_get_accel")
        return a

    def get_rcrit(self):
        torch = self._torch
        r = torch.empty((self.N,), dtype=torch.float64, device=self.device)
        _check(self._L.genga_get_rcrit(self._h, _dptr(r)), "genga_get_rcrit")
        return r

    def set_radii(self, R=None):
        """Physical radii (device float64 [N]); None: all 0, no body ever collides."""
        _check(self._L.genga_set_radii(self._h, _dptr(R)), "genga_set_radii")

    def get_radii(self):
        torch = self._torch
        R = torch.empty((self.N,), dtype=torch.float64, device=self.device)
        _check(self._L.genga_get_radii(self._h, _dptr(R)), "genga_get_radii")
        return R

    def get_mass(self):
        torch = self._torch
        m = torch.empty((self.N,), dtype=torch.float64, device=self.device)
        _check(self._L.genga_get_mass(self._h, _dptr(m)), "genga_get_mass")
        return m

    def merge(self, precision=FP64):
        """Step-end perfect mergers (genga_merge, reading R13).  Returns (n_merged, status, newidx): newidx is a
        device int32 tensor over the bodies BEFORE the call.  self.N follows the handle."""
        torch = self._torch
        newidx = torch.empty((self.N,), dtype=torch.int32, device=self.device)
        n, s = ctypes.c_int(0), ctypes.c_int(0)
        _check(self._L.genga_merge(self._h, int(precision), _dptr(newidx), ctypes.byref(n), ctypes.byref(s)), "genga_merge")
        self.N = int(self._L.genga_num_bodies(self._h))
        self.n_big = int(self._L.genga_num_big_bodies(self._h))
        return int(n.value), int(s.value), newidx

    # ---- the path ------------------------------------------------------------------------------
    def resort(self):
        _check(self._L.genga_resort(self._h), "genga_resort")

    def accel(self, precision=FP64):
        _check(self._L.genga_accel(self._h, int(precision)), "genga_accel")

    def kick(self, dt, precision=FP64):
        _check(self._L.genga_kick(self._h, float(dt), int(precision)), "genga_kick")

    def drift(self, dt):
        _check(self._L.genga_drift(self._h, float(dt)), "genga_drift")

    def sunkick(self, tau):
        _check(self._L.genga_sunkick(self._h, float(tau)), "genga_sunkick")

    def step(self, dt, precision=FP64):
        _check(self._L.genga_step(self._h, float(dt), int(precision)), "genga_step")

    def run(self, dt, nsteps, precision=FP64):
        _check(self._L.genga_run(self._h, float(dt), int(nsteps), int(precision)), "genga_run")

    def leapfrog(self, dt, nsteps, precision=FP64):
        _check(self._L.genga_leapfrog(self._h, float(dt), int(nsteps), int(precision)), "genga_leapfrog")

    def encounter_pairs(self, cap=None):
        """Returns an int32 numpy array (count, 2), i < j, of the last force evaluation."""
        import numpy as np
        cap = int(cap if cap is not None else self.params.pair_capacity or (4 * self.N + 1024))
        buf = np.zeros((max(cap, 1), 2), dtype=np.int32)
        cnt = ctypes.c_int(0)
        code = self._L.genga_encounter_pairs(self._h, buf.ctypes.data_as(ctypes.c_void_p), cap, ctypes.byref(cnt))
        if code == ECAPACITY:
            raise GengaError(code, f"genga_encounter_pairs: {cnt.value} pairs exceed the capacity {cap}")
        _check(code, "genga_encounter_pairs")
        return buf[:cnt.value].copy()

    def energy_angmom(self):
        import numpy as np
        E = ctypes.c_double(0.0)
        L = (ctypes.c_double * 3)()
        _check(self._L.genga_energy_angmom(self._h, ctypes.byref(E), L), "genga_energy_angmom")
        return E.value, np.array([L[0], L[1], L[2]])

    # ---- diagnostics ---------------------------------------------------------------------------
    def nearfield_stats(self) -> NearfieldStats:
        c, o = ctypes.c_longlong(0), ctypes.c_int(0)
        _check(self._L.genga_nearfield_stats(self._h, ctypes.byref(c), ctypes.byref(o)), "genga_nearfield_stats")
        return NearfieldStats(int(c.value), bool(o.value))

    def encounter_stats(self):
        """Encounter mode: (groups, bodies, largest group, missed pairs, status mask); clears count and mask."""
        g, b, l, m, s = (ctypes.c_int(0) for _ in range(5))
        _check(self._L.genga_encounter_stats(self._h, ctypes.byref(g), ctypes.byref(b), ctypes.byref(l), ctypes.byref(m),
                                             ctypes.byref(s)), "genga_encounter_stats")
        return int(g.value), int(b.value), int(l.value), int(m.value), int(s.value)

    def encounter_work(self):
        """Encounter mode: (force evaluations of all group integrations of the last drift, the most any group needed,
        rejected Bulirsch-Stoer macro steps)."""
        t, mx, rj = ctypes.c_longlong(0), ctypes.c_int(0), ctypes.c_int(0)
        _check(self._L.genga_encounter_work(self._h, ctypes.byref(t), ctypes.byref(mx), ctypes.byref(rj)), "genga_encounter_work")
        return int(t.value), int(mx.value), int(rj.value)

    def set_profiling(self, enable=True):
        """enable: True (all kernel classes), False, or a bit mask (1 kick, 2 near field, 4 prep, 8 drift)."""
        mask = 15 if enable is True else int(enable)
        _check(self._L.genga_set_profiling(self._h, mask), "genga_set_profiling")

    def kernel_time(self, which, reset=False):
        """(total ms, launches) of kernel class which: 0 all-pairs kick, 1 near field, 2 prep, 3 drift."""
        ms, n = ctypes.c_double(0), ctypes.c_longlong(0)
        _check(self._L.genga_kernel_time(self._h, int(which), ctypes.byref(ms), ctypes.byref(n), int(reset)),
               "genga_kernel_time")
        return ms.value, int(n.value)

    def set_tuning(self, key, value):
        _check(self._L.genga_set_tuning(self._h, int(key), int(value)), "genga_set_tuning")

    def autotune(self, precision):
        """genga_autotune: returns (chosen variant, its force-evaluation time in ms)."""
        v, ms = ctypes.c_int(0), ctypes.c_double(0)
        _check(self._L.genga_autotune(self._h, int(precision), ctypes.byref(v), ctypes.byref(ms)), "genga_autotune")
        return int(v.value), float(ms.value)

    def launch_count(self) -> int:
        return int(self._L.genga_launch_count(self._h))

    def synchronize(self):
        _check(self._L.genga_synchronize(self._h), "genga_synchronize")


def from_workload(w, **kw) -> "Genga":
    """Create a handle from a ``workloads.Workload`` (numpy, heliocentric v) on cuda:0."""
    import torch
    dev = kw.pop("device", "cuda:0")
    m = torch.from_numpy(w.m).to(dev)
    x = torch.from_numpy(w.x).to(dev)
    v = torch.from_numpy(w.v).to(dev)
    args = dict(G=w.G, M_star=w.M_star, n1=w.n1, n2=w.n2, dt_rcrit=w.dt, pair_rule=w.pair_rule,
                v_is_heliocentric=True, device=dev)
    args.update(kw)
    return Genga(m, x, v, **args)
