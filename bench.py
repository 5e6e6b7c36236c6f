#!/usr/bin/env python
"""bench.py -- the headline benchmark of the GENGA level-0 hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--n N_BODIES] [--sweep]
    python bench.py --impl reference ...        # the CPU oracle, as it stands, on the host cores

One "step" is one pass of the whole hot path over the workload: S(dt/2) D(dt) S(dt/2) K(dt), the
body of the merged-leapfrog loop of genga_run (one force evaluation per step: r_crit, packing,
all-pairs kick, FP64 near field + encounter list, velocity update, Sun-kick, Kepler drift).
The default workload is BASELINE.json configs[4]: 40 000 self-gravitating planetesimals.
Metric: ordered pair interactions per second, N (N - 1) per force evaluation;
steps/s and N x steps/s ("steps per second per particle") are reported beside it
for FP32 (headline; the paper's contribution) and FP64 force precision.

Prints ONE JSON line on rank 0.  Under torchrun every rank integrates its own, independently
seeded, system of the same shape (the path shards over independent problems: weak scaling, no
data-path collective); time is the max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "pair interactions/s & steps/s per body at N=40k, FP32 vs FP64 forces"
UNIT = "pair interactions/s"
# flops per ordered pair interaction, the stated convention
FLOP_FP32, FLOP_FP64 = 18.0, 25.0
SMS, SM_MAX_HZ = 148, 1.965e9
PEAK_FP32_TFLOPS = SMS * 128 * 2 * SM_MAX_HZ / 1e12      # 74.45: 128 FP32 lanes/SM, FMA = 2 flop
PEAK_FP64_TFLOPS = SMS * 64 * 2 * SM_MAX_HZ / 1e12       # 37.22: 64 FP64 lanes/SM (DFMA probe confirms)


def capture_traffic(variant_name, precision):
    """DRAM bytes per launch of the all-pairs kernel from the committed ncu capture (profiles/kick_traffic.json, written
    from `ncu --set full`: dram__bytes_read.sum + dram__bytes_write.sum).  None unless the capture is of the very
    variant this run times."""
    try:
        with open(os.path.join(ROOT, "profiles", "kick_traffic.json")) as f:
            rec = json.load(f)
        for e in rec["captures"]:
            if e["precision"] == precision and e["variant"] == variant_name:
                return e["dram_bytes_per_launch"], f"{e['capture']} (git {e['git']}, N = {e['N']})", e.get("pipe_busy_pct")
    except Exception:
        pass
    return None, "no ncu capture of this kernel variant is committed (profiles/kick_traffic.json)", None


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--n", type=int, default=None, help="override the body count of the config")
    ap.add_argument("--sweep", action="store_true", help="also run the N = 2^10..2^17 sweep (extra JSON key)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-flush", action="store_true", help="do not flush L2 between timed steps")
    ap.add_argument("--report", action="store_true",
                    help="run every BASELINE.json config (0-4) for its full step count in both precisions and print one "
                         "JSON line per (config, precision): rates, fractions of peak, dE/E, dL/L, encounter counts")
    ap.add_argument("--variant32", type=int, default=None, help="with --no-autotune: FP32 kernel variant (genga_set_tuning key 0)")
    ap.add_argument("--variant64", type=int, default=None, help="with --no-autotune: FP64 kernel variant (genga_set_tuning key 1)")
    ap.add_argument("--mergers", action="store_true",
                    help="NEXT-4: the performance shape with inflated radii and a merger pass (genga_merge) after every step; "
                         "one JSON line: ms per step with and without the pass, bodies merged, what is conserved")
    ap.add_argument("--hybrid", action="store_true",
                    help="time the hybrid step instead (NEXT-1: weight_mode = 1, encounter_mode = 1, default listing and substeps)")
    ap.add_argument("--no-autotune", action="store_true", help="keep the default kernel variants (no start-up self-tuning)")
    ap.add_argument("--no-tables", action="store_true",
                    help="skip the per-config table (configs 0-3, full step counts) and the N sweep that a default run adds "
                         "to its JSON line under 'configs' and 'sweep' (each row with its own clock record)")
    return ap.parse_args()


def dist_env():
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


class ClockSampler:
    """Samples SM clock and throttle reasons of one GPU through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.02):
        self.index, self.period = index, period_s
        self.sm, self.reasons, self.power = [], set(), []
        self.sm_max = None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self._nv = None

    def _loop(self):
        nv = self._nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4),
        }
        while not self._stop.is_set():
            try:
                self.sm.append(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self._h) / 1000.0)
                mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
                for k, bit in names.items():
                    if mask & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self._nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        out = {"sm_mhz": statistics.median(self.sm) if self.sm else None,
               "sm_max_mhz": self.sm_max, "reasons": sorted(self.reasons),
               "power_w_max": max(self.power) if self.power else None, "samples": len(self.sm)}
        # a row measured under a slowdown, or with the SM clock stuck well below max for no stated reason, does not count
        bad = {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"} & self.reasons
        stuck = bool(self.sm) and self.sm_max and not self.reasons and out["sm_mhz"] < 0.85 * self.sm_max
        out["rejected"] = bool(bad or stuck)
        return out


def make_workload(args, rank):
    from paper_2309_08217_b200 import workloads as W
    w = W.config(args.config, args.n)
    if rank > 0 and args.config in (0, 1, 4):          # every rank its own independently seeded system
        tot = {0: 2.5, 1: 5.0, 4: 5.0}[args.config]
        w = W.planetesimal_disc(w.N, tot, w.seed + 7919 * rank, args.config, w.name, w.dt, w.nsteps)
    return w


def max_over_ranks(torch, dist, values, device):
    """Every rank times its own system; the job's time is the slowest rank's (one all-reduce(MAX) of
    the timed totals, after the timed region -- the data path itself has no collective)."""
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.tolist()]


def whole_job_rate(world, units_per_rank_step, steps, total_ms):
    """Units all ranks processed / the max-over-ranks time (weak scaling: fixed work per rank)."""
    return world * units_per_rank_step * steps / (total_ms * 1e-3)


def time_steps(torch, g, w, prec, steps, warmup, flush_buf, dist, profile_timed=True):
    """K timed steps, each bracketed by CUDA events on the handle's stream; L2 flushed between."""
    stream = torch.cuda.current_stream()
    # profile_timed: CUDA events around every all-pairs launch inside the timed region (the headline's roofline
    # figure).  For small N (sweep) the event records themselves cost ~8 us per step, so there the steps are
    # timed without them and the kernel is timed in the extra pass below.
    g.set_profiling(1 if profile_timed else 0)
    g.kick(0.5 * w.dt, prec)                           # opening half kick of the merged leapfrog
    for _ in range(warmup):
        g.leapfrog(w.dt, 1, prec)
    g.synchronize()
    for k in range(4):
        g.kernel_time(k, reset=True)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    l0 = g.launch_count()
    t0 = time.perf_counter()
    for s in range(steps):
        if flush_buf is not None:
            flush_buf.zero_()                          # > L2 capacity, untimed
        ev[s][0].record(stream)
        g.leapfrog(w.dt, 1, prec)
        ev[s][1].record(stream)
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    if dist is not None:
        dist.barrier()
    ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = float(sum(ms))
    launches = g.launch_count() - l0
    kick_ms, kick_n = g.kernel_time(0, reset=True)        # the dominant kernel, timed live in the timed region
    # per-kernel breakdown of the other classes: a short extra pass, not part of the timed region
    g.set_profiling(15)
    for _ in range(5):
        g.leapfrog(w.dt, 1, prec)
    g.synchronize()
    kt = [g.kernel_time(k, reset=True) for k in range(4)]
    g.set_profiling(1 if profile_timed else 0)
    kms = [(t / max(n, 1)) for t, n in kt]
    if profile_timed:
        kms[0] = kick_ms / max(kick_n, 1)
    else:
        kick_n = kt[0][1]
    return {"total_ms": total_ms, "ms_median": statistics.median(ms), "wall_s": wall,
            "launches": launches, "kernel_ms": kms, "kernel_n": [kick_n] + [n for _, n in kt[1:]]}


def time_e2e(torch, g, w, prec, steps, warmup, flush_buf):
    """The same step through the C ABI with HOST buffers: pinned host -> device copy of (m, x, v),
    one step, device -> host read of (x, v); every step, inside the timed region."""
    import numpy as np
    stream = torch.cuda.current_stream()
    m = torch.from_numpy(w.m).pin_memory()
    x = torch.from_numpy(np.ascontiguousarray(w.x)).pin_memory()
    v = torch.from_numpy(np.ascontiguousarray(w.v)).pin_memory()
    xo, vo = torch.empty_like(x).pin_memory(), torch.empty_like(v).pin_memory()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for s in range(-warmup, steps):
        if flush_buf is not None:
            flush_buf.zero_()
        if s >= 0:
            ev[s][0].record(stream)
        g.set_state_host(m, x, v)
        g.leapfrog(w.dt, 1, prec)
        g.get_state_host(xo, vo, heliocentric_v=True)  # synchronises
        if s >= 0:
            ev[s][1].record(stream)
        x.copy_(xo); v.copy_(vo)                       # host-side hand-over to the next step
    torch.cuda.synchronize()
    total_ms = float(sum(a.elapsed_time(b) for a, b in ev))
    h2d = m.numel() * 8 + x.numel() * 8 + v.numel() * 8
    d2h = xo.numel() * 8 + vo.numel() * 8
    return total_ms, h2d, d2h


def cpu_oracle_steps(w, steps, warmup=0):
    """The oracle, as it stands, on the host cores: `steps` merged-leapfrog steps (each one full
    O(N^2) oracle force evaluation + Sun-kick + Kepler drift).  Returns (seconds, threads)."""
    import oracle
    p = oracle.Params(G=w.G, M_star=w.M_star, n1=w.n1, n2=w.n2, dt_rcrit=w.dt, pair_rule=w.pair_rule)
    x, v = w.x.copy(), oracle.to_democratic(w.m, w.v, w.M_star)
    times = []
    for s in range(-warmup, steps):
        t0 = time.perf_counter()
        x = oracle.sunkick(w.m, x, v, p, 0.5 * w.dt)
        x, v = oracle.drift(x, v, p, w.dt)
        x = oracle.sunkick(w.m, x, v, p, 0.5 * w.dt)
        v, _ = oracle.kick(w.m, x, v, p, w.dt)
        if s >= 0:
            times.append(time.perf_counter() - t0)
    return times, oracle.num_threads()


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return
    w = make_workload(args, 0)
    steps = max(1, min(args.steps, 3))                 # bounded sample: a few full O(N^2) steps
    times, threads = cpu_oracle_steps(w, steps, warmup=min(args.warmup, 1))
    pairs = w.N * (w.N - 1.0)
    total = sum(times)
    value = pairs * steps / total
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": min(args.warmup, 1), "ms_per_step": 1e3 * total / steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "N": w.N, "dt_days": w.dt, "requested_steps": args.steps,
                   "note": "CPU FP64 oracle (oracle/genga_oracle.c, -O2, OpenMP over i), not a GPU program"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle",
                         "sample": f"{steps} full merged-leapfrog step(s) of the N={w.N} workload"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_cuda(args):
    import torch
    from paper_2309_08217_b200 import binding as B
    from paper_2309_08217_b200 import workloads as W

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the GENGA hot path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    B.load()

    w = make_workload(args, rank)
    N, pairs = w.N, w.N * (w.N - 1.0)
    hkw = dict(weight_mode=1, encounter_mode=1, cand_capacity=64 * w.N) if args.hybrid else {}
    dev = f"cuda:{local_rank}"
    flush = None if args.no_flush else torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    res, e2e, tuned = {}, {}, {}
    sampler = ClockSampler(torch.cuda.current_device() if "CUDA_VISIBLE_DEVICES" not in os.environ else local_rank)
    with sampler:
        for prec, name in ((B.FP32, "fp32"), (B.FP64, "fp64")):
            g = B.from_workload(w, device=dev, **hkw)
            if not args.no_autotune:
                tuned[name] = g.autotune(prec)                 # start-up self-tuning, untimed
            else:
                fixed = args.variant32 if prec == B.FP32 else args.variant64
                tuned[name] = (fixed if fixed is not None else 0, None)
                g.set_tuning(0 if prec == B.FP32 else 1, tuned[name][0])
            g.set_profiling(1)                         # CUDA events around the all-pairs kernel only
            r = time_steps(torch, g, w, prec, args.steps, args.warmup, flush, dist)
            st = g.nearfield_stats()
            r["candidates"], r["overflowed"] = st.candidates, st.overflowed
            r["encounter_pairs"] = int(len(g.encounter_pairs(cap=4 * N + 1024)))
            res[name] = r
            g.close()
    # energy / angular-momentum drift over the timed run length, both precisions (reported)
    drift = {}
    for prec, name in ((B.FP32, "fp32"), (B.FP64, "fp64")):
        g = B.from_workload(w, device=dev, **hkw)
        g.set_tuning(0 if prec == B.FP32 else 1, tuned[name][0])
        E0, L0 = g.energy_angmom()
        g.run(w.dt, args.steps, prec)
        E1, L1 = g.energy_angmom()
        import numpy as np
        drift[name] = {"dE_over_E": E1 / E0 - 1.0,
                       "dL_over_L": float(np.linalg.norm(L1) / np.linalg.norm(L0) - 1.0)}
        g.close()
    e2e_steps = min(args.steps, 50)
    for prec, name in ((B.FP32, "fp32"), (B.FP64, "fp64")):
        g = B.from_workload(w, device=dev, **hkw)
        g.set_tuning(0 if prec == B.FP32 else 1, tuned[name][0])
        ms, h2d, d2h = time_e2e(torch, g, w, prec, e2e_steps, min(args.warmup, 3), flush)
        e2e[name] = (ms, h2d, d2h)
        g.close()

    # max over ranks of the timed totals
    t32, t64, te32, te64 = max_over_ranks(torch, dist, [res["fp32"]["total_ms"], res["fp64"]["total_ms"],
                                                        e2e["fp32"][0], e2e["fp64"][0]], dev)
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    K = args.steps
    def per_prec(name, total_ms, flop, peak):
        r = res[name]
        pps = whole_job_rate(world, pairs, K, total_ms)
        kick_ms = r["kernel_ms"][0]
        tf = flop * pairs / (kick_ms * 1e-3) / 1e12
        return {"pair_interactions_per_s": pps, "steps_per_s": K / (total_ms * 1e-3),
                "body_steps_per_s": world * N * K / (total_ms * 1e-3), "ms_per_step": total_ms / K,
                "kernel_ms": {"kick": r["kernel_ms"][0], "nearfield": r["kernel_ms"][1],
                              "onbody_fused": r["kernel_ms"][3],      # velocity update + S D S + r_crit/packing, one kernel
                              "prep_alone": r["kernel_ms"][2]},        # 0 unless a force evaluation ran outside a step
                "kick_kernel_pairs_per_s": pairs / (kick_ms * 1e-3),
                "kick_kernel_tflops": tf, "kick_kernel_frac_of_peak": tf / peak,
                "step_frac_of_peak": flop * pairs * K / (total_ms * 1e-3) / 1e12 / peak,
                "flop_per_pair": flop, "kernel_variant": B.variant_name(0 if name == "fp32" else 1, tuned[name][0]),
                "nearfield_candidates": r["candidates"],
                "candidate_overflow": r["overflowed"], "encounter_pairs_last": r["encounter_pairs"],
                **drift[name]}
    p32 = per_prec("fp32", t32, FLOP_FP32, PEAK_FP32_TFLOPS)
    p64 = per_prec("fp64", t64, FLOP_FP64, PEAK_FP64_TFLOPS)

    kname32 = "kick32_sym_kernel" if "sym" in p32["kernel_variant"] else "kick32_kernel"
    kname64 = "kick64_sym_kernel" if "sym" in p64["kernel_variant"] else "kick64_kernel"
    tr32 = capture_traffic(p32["kernel_variant"], "fp32")
    tr64 = capture_traffic(p64["kernel_variant"], "fp64")
    line = {
        "metric": METRIC, "value": p32["pair_interactions_per_s"], "unit": UNIT, "n_gpus": world,
        "steps": K, "warmup": args.warmup, "ms_per_step": t32 / K, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "N": N, "dt_days": w.dt, "headline_precision": "fp32",
                   "step": "S(dt/2) D(dt) S(dt/2) K(dt): one force evaluation per step",
                   "l2": "inputs are L2-resident by nature (1.6 MB); L2 flushed by a 256 MiB write between timed steps"
                         if flush is not None else "no flush",
                   "per_rank": "independent system per rank, no data-path collective",
                   **({"encounter_mode": 1, "note": "--hybrid: the opt-in hybrid step (NEXT-1), not the headline configuration"}
                      if args.hybrid else {})},
        "precisions": {"fp32": p32, "fp64": p64},
        "roofline": {"bound": "alu", "kernel": kname32, "achieved": p32["kick_kernel_tflops"],
                     "peak": PEAK_FP32_TFLOPS, "unit": "TFLOP/s", "frac": p32["kick_kernel_frac_of_peak"],
                     "traffic": tr32[0], "traffic_source": tr32[1],
                     "pipe_busy_pct_capture": tr32[2],       # the FMA pipe's busy cycles in that capture (what 'frac' is NOT: see convention)
                     "peak_source": "derived: 148 SMs x 128 FP32 lanes x 2 flop x 1.965 GHz (DESIGN.md section 7); "
                                    "MEASURED_PEAKS.json has no FP32/FP64 ALU figure.  'frac' (the headline) divides by this "
                                    "derived peak; 'frac_of_measured' by the FFMA2 / DFMA rate the in-library probe reached "
                                    "in this very run ('peak_measured')",
                     "flop_per_pair": FLOP_FP32,
                     "convention": "achieved = 18 (25) flop x N (N - 1) ordered pairs / kernel time: the flops of the plain "
                                   "per-ordered-pair sequence (SURVEY.md 8(d)).  The symmetric kernels evaluate each unordered "
                                   "pair once (16 FP32 / 20 FP64 operations for both directions; 14 / 18 in far tiles between "
                                   "uniform-mass chunks, where G m is factored out of the loop: every far tile of this equal-mass "
                                   "workload), so they execute fewer flops than this convention counts and 'frac' can exceed 1; "
                                   "the time is what is measured",
                     "fp64": {"kernel": kname64, "traffic": tr64[0], "traffic_source": tr64[1], "pipe_busy_pct_capture": tr64[2],
                              "achieved": p64["kick_kernel_tflops"],
                              "peak": PEAK_FP64_TFLOPS, "frac": p64["kick_kernel_frac_of_peak"],
                              "flop_per_pair": FLOP_FP64}},
        "e2e": {"value": whole_job_rate(world, pairs, e2e_steps, te32), "unit": UNIT,
                "h2d_bytes_per_step": e2e["fp32"][1], "d2h_bytes_per_step": e2e["fp32"][2], "steps": e2e_steps,
                "fp64_value": whole_job_rate(world, pairs, e2e_steps, te64),
                "ms_per_step": te32 / e2e_steps, "device_ms_per_step": t32 / K,
                "e2e_over_device": (te32 / e2e_steps) / (t32 / K)},
        "gpu_launches": res["fp32"]["launches"],
        "clocks": sampler.summary(),
    }
    return line, w


def alu_probes():
    """Measured issue rates of this GPU (register-only kernels, genga_peak_probe), as TFLOP/s."""
    from paper_2309_08217_b200 import binding as B
    out = {}
    for which, name, flop in ((0, "ffma_tflops", 2.0), (1, "ffma2_tflops", 2.0), (2, "dfma_tflops", 2.0),
                              (3, "mufu_rsq_gops", 1.0), (4, "mufu_rsq64h_gops", 1.0)):
        ops, _ = B.peak_probe(which, 2048)
        out[name] = ops * flop / (1e12 if flop == 2.0 else 1e9)
    return out


def cpu_oracle_kick(w, **kw):
    """One oracle force evaluation + velocity update (oracle_kick) of workload w on the host cores: the
    oracle timed beside the GPU per config / per sweep N.  Returns (seconds, pairs/s, threads)."""
    import oracle
    pk = dict(G=w.G, M_star=w.M_star, n1=w.n1, n2=w.n2, dt_rcrit=w.dt, pair_rule=w.pair_rule)
    pk.update({k: v for k, v in kw.items() if k in ("n1", "n2", "pair_rule", "n_big", "weight_mode")})
    p = oracle.Params(**pk)
    vd = oracle.to_democratic(w.m, w.v, w.M_star)
    t0 = time.perf_counter()
    oracle.kick(w.m, w.x.copy(), vd, p, w.dt)
    dt = time.perf_counter() - t0
    nb = pk.get("n_big", -1)
    pairs = w.N * (w.N - 1.0) if nb < 0 else (2.0 * nb * (w.N - nb) + nb * (nb - 1.0))
    return dt, pairs / dt, oracle.num_threads()


def run_sweep(args, cpu=True):
    """N = 2^10 .. 2^17 (BASELINE.json configs[4]): N x steps/s per precision, device-timed; every row carries the
    clock record sampled while it ran (a row with 'rejected' does not count)."""
    import torch
    from paper_2309_08217_b200 import binding as B
    from paper_2309_08217_b200 import workloads as W
    out = []
    for n in W.SWEEP_N:
        w = W.config(4, n)
        row = {"N": n}
        steps = 200 if n <= 32768 else 20
        pairs = n * (n - 1.0)
        sampler = ClockSampler(torch.cuda.current_device())
        with sampler:
            for prec, name, flop, peak in ((B.FP32, "fp32", FLOP_FP32, PEAK_FP32_TFLOPS), (B.FP64, "fp64", FLOP_FP64, PEAK_FP64_TFLOPS)):
                g = B.from_workload(w)
                variant = 0 if args.no_autotune else g.autotune(prec)[0]
                r = time_steps(torch, g, w, prec, steps, 3, None, None, profile_timed=False)
                row[name] = {"ms_per_step": r["total_ms"] / steps, "body_steps_per_s": n * steps / (r["total_ms"] * 1e-3),
                             "pair_interactions_per_s": pairs * steps / (r["total_ms"] * 1e-3),
                             "step_frac_of_peak": flop * pairs * steps / (r["total_ms"] * 1e-3) / 1e12 / peak,
                             "kick_kernel_ms": r["kernel_ms"][0], "nearfield_ms": r["kernel_ms"][1],
                             "kick_kernel_frac_of_peak": flop * pairs / (r["kernel_ms"][0] * 1e-3) / 1e12 / peak,
                             "launches_per_step": r["launches"] / steps,
                             "kernel_variant": B.variant_name(0 if prec == B.FP32 else 1, variant)}
                # the same steps as ONE genga_leapfrog(steps) call, as a run issues them (small systems then take whole
                # sequences of steps in one launch: csrc/lean_step.cu)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                g.leapfrog(w.dt, 8, prec)                          # untimed: the first launch of a kernel loads it
                l0 = g.launch_count()
                torch.cuda.synchronize()
                e0.record()
                g.leapfrog(w.dt, steps, prec)
                e1.record()
                torch.cuda.synchronize()
                ms1 = e0.elapsed_time(e1)
                row[name].update({"one_call_ms_per_step": ms1 / steps, "one_call_body_steps_per_s": n * steps / (ms1 * 1e-3),
                                  "one_call_launches_per_step": (g.launch_count() - l0) / steps})
                g.close()
        row["clocks"] = sampler.summary()
        if cpu and not args.no_cpu_baseline:
            sec, pps, thr = cpu_oracle_kick(w)
            row["cpu_oracle_kick"] = {"seconds": sec, "pair_interactions_per_s": pps, "cores": thr}
        out.append(row)
    return out


def run_configs_table(args):
    """north_star: 'report ... at each config'.  BASELINE.json configs 0-3 at their full sizes and step counts (config 4 is
    the headline measurement itself), both precisions, each row with its own clock record: ms per step, rates, fraction
    of peak of the whole step, dE/E and dL/L over the run, encounter pairs of the last evaluation."""
    import numpy as np
    import torch
    from paper_2309_08217_b200 import binding as B
    from paper_2309_08217_b200 import workloads as W
    rows = []
    for cfg in (0, 1, 2, 3):
        w = W.config(cfg)
        pairs = w.N * (w.N - 1.0)
        sampler = ClockSampler(torch.cuda.current_device())
        row = {"config": cfg, "workload": w.name, "N": w.N, "dt_days": w.dt, "steps": w.nsteps}
        with sampler:
            for prec, name, flop, peak in ((B.FP32, "fp32", FLOP_FP32, PEAK_FP32_TFLOPS), (B.FP64, "fp64", FLOP_FP64, PEAK_FP64_TFLOPS)):
                g = B.from_workload(w)
                variant = 0 if args.no_autotune else g.autotune(prec)[0]
                g.run(w.dt, 3, prec)                               # warm-up
                g.close()
                g = B.from_workload(w)
                g.set_tuning(0 if prec == B.FP32 else 1, variant)
                E0, L0 = g.energy_angmom()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                e0.record()
                g.run(w.dt, w.nsteps, prec)                        # K(dt/2) [S D S K(dt)]^(n-1) S D S K(dt/2)
                e1.record()
                torch.cuda.synchronize()
                ms = e0.elapsed_time(e1)
                E1, L1 = g.energy_angmom()
                enc = int(len(g.encounter_pairs(cap=8 * w.N + 4096)))
                g.close()
                evals = w.nsteps + 1
                row[name] = {"ms_per_step": ms / w.nsteps, "body_steps_per_s": w.N * w.nsteps / (ms * 1e-3),
                             "pair_interactions_per_s": pairs * evals / (ms * 1e-3),
                             "step_frac_of_peak": flop * pairs * evals / (ms * 1e-3) / 1e12 / peak,
                             "dE_over_E": E1 / E0 - 1.0, "dL_over_L": float(np.linalg.norm(L1) / np.linalg.norm(L0) - 1.0),
                             "encounter_pairs_last_eval": enc,
                             "kernel_variant": B.variant_name(0 if prec == B.FP32 else 1, variant)}
        row["clocks"] = sampler.summary()
        rows.append(row)
    return rows


def run_report(args):
    """north_star: 'Report pair interactions/s and steps/s per body at each config ... relative energy and
    angular-momentum drift over the run: reported for both precisions' (+ encounter pairs per step, config 1)."""
    import numpy as np
    import torch
    from paper_2309_08217_b200 import binding as B
    from paper_2309_08217_b200 import workloads as W
    B.load()
    cases = [(cfg, W.config(cfg), {}) for cfg in range(5)]
    # NEXT-2: config 3 at the paper's 30 000 planetesimals in TP2 mode
    cases.append(("3-tp2", W.config(3, 30000), {"n_big": 4}))
    # NEXT-4: Eq. 1 as printed (n1 = 3, n2 = 0.4, max rule) on the performance shape, 50 steps
    w4 = W.config(4)
    w4.nsteps = 50
    cases.append(("4-eq1", w4, {"n1": 3.0, "n2": 0.4, "pair_rule": B.PAIR_MAX,
                                "pair_capacity": 40 * w4.N, "cand_capacity": 64 * w4.N}))
    # NEXT-1: the hybrid step (encounter mode, reading R11) on the performance shape, 200 steps
    w5 = W.config(4)
    w5.nsteps = 200
    hyb = {"weight_mode": 1, "encounter_mode": 1, "enc_list_scale": 8.0, "enc_list_vfactor": 1.25}   # groups: Bulirsch-Stoer, tol 1e-12
    cases.append(("4-hybrid", w5, dict(hyb, cand_capacity=64 * w5.N)))
    for c in (1, 2, 3):                                            # ... and on the paper-shaped configs, full length
        wc = W.config(c)
        cases.append((f"{c}-hybrid", wc, dict(hyb, cand_capacity=64 * wc.N, pair_capacity=40 * wc.N)))
    for cfg, w, kw in cases:
        nb = kw.get("n_big", -1)
        if not args.no_cpu_baseline:                               # the oracle beside it: one kick per config
            sec, pps, thr = cpu_oracle_kick(w, **kw)
            print(json.dumps({"report": "cpu_oracle_kick", "config": cfg, "workload": w.name, "N": w.N, "seconds": sec,
                              "pair_interactions_per_s": pps, "cores": thr, "kind": "oracle"}), flush=True)
        pairs = w.N * (w.N - 1.0) if nb < 0 else (2.0 * nb * (w.N - nb) + nb * (nb - 1.0))   # interacting ordered pairs
        for prec, name, flop, peak in ((B.FP32, "fp32", FLOP_FP32, PEAK_FP32_TFLOPS), (B.FP64, "fp64", FLOP_FP64, PEAK_FP64_TFLOPS)):
            g = B.from_workload(w, **kw)
            variant = 0 if args.no_autotune else g.autotune(prec)[0]
            E0, L0 = g.energy_angmom()
            g.run(w.dt, 3, prec)                                   # warm-up (3 steps of the same trajectory)
            g.close()
            g = B.from_workload(w, **kw)
            g.set_tuning(0 if prec == B.FP32 else 1, variant)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            sampler = ClockSampler(torch.cuda.current_device())
            with sampler:                                          # every row carries its own clock record
                e0.record()
                g.run(w.dt, w.nsteps, prec)                        # K(dt/2) [S D S K(dt)]^(n-1) S D S K(dt/2)
                e1.record()
                torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            E1, L1 = g.energy_angmom()
            enc_last = int(len(g.encounter_pairs(cap=max(8 * w.N + 4096, kw.get("pair_capacity", 0)))))
            st = g.nearfield_stats()
            enc_stats = g.encounter_stats() if kw.get("encounter_mode") else None    # missed / status: since the warm-up
            enc_work = g.encounter_work() if kw.get("encounter_mode") else None
            g.close()
            evals = w.nsteps + 1
            line = {"report": "config", "config": cfg, "workload": w.name, "N": w.N, "dt_days": w.dt, "steps": w.nsteps,
                    "precision": name, "n_big": nb,
                    "kernel_variant": "tp2_kernel (FP64)" if nb >= 0 else B.variant_name(0 if prec == B.FP32 else 1, variant),
                    "ms_per_step": ms / w.nsteps, "steps_per_s": w.nsteps / (ms * 1e-3),
                    "body_steps_per_s": w.N * w.nsteps / (ms * 1e-3),
                    "pair_interactions_per_s": pairs * evals / (ms * 1e-3),
                    "step_frac_of_peak": flop * pairs * evals / (ms * 1e-3) / 1e12 / peak,
                    "dE_over_E": E1 / E0 - 1.0,
                    "dL_over_L": float(np.linalg.norm(L1) / np.linalg.norm(L0) - 1.0),
                    "encounter_pairs_last_eval": enc_last, "nearfield_candidates_last_eval": st.candidates,
                    "clocks": sampler.summary()}
            if enc_stats is not None:
                line["encounter_groups_last_drift"] = {"groups": enc_stats[0], "bodies": enc_stats[1], "largest": enc_stats[2],
                                                       "missed_pairs_whole_run": enc_stats[3], "status": enc_stats[4],
                                                       "integrator": (f"RK4 x {kw['enc_nsub']}" if kw.get("enc_nsub") else f"Bulirsch-Stoer tol {kw.get('enc_tol', 1e-12):g}"),
                                                       "rhs_total_max_rejected_last_drift": enc_work,
                                                       "list_scale": kw.get("enc_list_scale"), "list_vfactor": kw.get("enc_list_vfactor")}
            if cfg == 1:                                           # encounter-pair counts per step (untimed second run)
                g = B.from_workload(w, **kw)
                g.set_tuning(0 if prec == B.FP32 else 1, variant)
                g.kick(0.5 * w.dt, prec)
                counts = []
                for _ in range(w.nsteps):
                    g.leapfrog(w.dt, 1, prec)
                    counts.append(len(g.encounter_pairs(cap=8 * w.N + 4096)))
                g.close()
                c = np.array(counts)
                line["encounter_pairs_per_step"] = {"mean": float(c.mean()), "min": int(c.min()), "max": int(c.max()),
                                                    "first": int(c[0]), "last": int(c[-1])}
                # dE/E and dL/L every 100 steps (dE/E alike in both precisions, dL/L of the
                # FP32 run a random walk some orders of magnitude above the FP64 one)
                g = B.from_workload(w, **kw)
                g.set_tuning(0 if prec == B.FP32 else 1, variant)
                g.kick(0.5 * w.dt, prec)
                series = []
                for k in range(w.nsteps // 100):
                    g.leapfrog(w.dt, 100, prec)
                    g.kick(-0.5 * w.dt, prec)                          # synchronise v with x for the diagnostics ...
                    Ek, Lk = g.energy_angmom()
                    g.kick(0.5 * w.dt, prec)                           # ... and go on
                    series.append([100 * (k + 1), Ek / E0 - 1.0, float(np.linalg.norm(Lk) / np.linalg.norm(L0) - 1.0)])
                g.close()
                line["drift_series_step_dE_dL"] = series
            print(json.dumps(line), flush=True)


def run_mergers(args):
    """NEXT-4 (R13): config 4 with radii inflated (bulk density 2 g/cm^3, factor 30, so that the
    200 steps do see collisions), genga_merge after every step.  Timed with CUDA events around the whole run; the pass
    synchronises (it returns N'), so its cost includes that round trip."""
    import numpy as np
    import torch
    from paper_2309_08217_b200 import binding as B
    from paper_2309_08217_b200 import workloads as W
    B.load()
    w = W.config(4)
    steps = args.steps if args.steps else 200
    AU_M, MSUN_KG, RHO, INFL = 1.495978707e11, 1.98892e30, 2000.0, 30.0
    R = INFL * (3.0 * w.m * MSUN_KG / (4.0 * np.pi * RHO)) ** (1.0 / 3.0) / AU_M
    for prec, name in ((B.FP32, "fp32"), (B.FP64, "fp64")):
        res = {}
        for mode in ("plain", "merging"):
            g = B.from_workload(w)
            g.autotune(prec)
            if mode == "merging":
                g.set_radii(torch.from_numpy(R).to(g.device))
            E0, L0 = g.energy_angmom()
            g.run(w.dt, 3, prec)                                     # warm-up; a first pass outside the timed region
            if mode == "merging":
                g.merge(prec)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            merged_timed = 0
            for _ in range(steps):
                g.run(w.dt, 1, prec)
                if mode == "merging":
                    n, status, newidx = g.merge(prec)
                    merged_timed += n
                    assert status == 0, status
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            E1, L1 = g.energy_angmom()
            res[mode] = {"ms_per_step": ms / steps, "N_end": g.N, "merged_in_timed_steps": merged_timed,
                         "dE_over_E": E1 / E0 - 1.0, "dL_over_L": float(np.linalg.norm(L1) / np.linalg.norm(L0) - 1.0)}
            g.close()
        print(json.dumps({"report": "mergers", "workload": w.name, "N": w.N, "steps": steps, "precision": name,
                          "radius_inflation": INFL, "bulk_density_kg_m3": RHO, "R_au": float(R[0]),
                          "plain": res["plain"], "merging": res["merging"],
                          "pass_ms": res["merging"]["ms_per_step"] - res["plain"]["ms_per_step"],
                          "note": "plain: genga_run one step at a time (K(dt/2) ... K(dt/2): two force evaluations per "
                                  "call); merging: the same plus genga_merge after every step"}), flush=True)


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    if args.mergers:
        run_mergers(args)
        return
    if args.report:
        run_report(args)
        return
    got = run_cuda(args)
    if got is None:
        return
    line, w = got
    line["alu_probe"] = alu_probes()
    rf = line["roofline"]
    rf["peak_measured"] = line["alu_probe"]["ffma2_tflops"]
    rf["frac_of_measured"] = rf["achieved"] / rf["peak_measured"]
    rf["fp64"]["peak_measured"] = line["alu_probe"]["dfma_tflops"]
    rf["fp64"]["frac_of_measured"] = rf["fp64"]["achieved"] / rf["fp64"]["peak_measured"]
    if line["n_gpus"] == 1 and not args.no_cpu_baseline:
        times, threads = cpu_oracle_steps(w, 4)          # ~10-20 s of host time at N = 40 000
        pairs = w.N * (w.N - 1.0)
        line["cpu_baseline"] = {"value": pairs * len(times) / sum(times), "unit": UNIT, "cores": threads,
                                "kind": "oracle", "sample": f"{len(times)} full merged-leapfrog steps of the "
                                f"N={w.N} workload ({sum(times):.1f} s of host time)"}
    if line["n_gpus"] == 1 and (args.sweep or not args.no_tables):
        line["sweep"] = run_sweep(args, cpu=args.sweep)           # --sweep: with the oracle's kick timed beside each N
    if line["n_gpus"] == 1 and not args.no_tables:
        line["configs"] = run_configs_table(args)
    print(json.dumps(line), flush=True)
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
