"""bench.py — throughput of the fused LLG + cavity-mode RK45 step (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3|cfg5|cfg4|cfg4_f64|cfg2|cfg2_f64|cfg1|cfg1_sweep|
                     cfg2_sweep|cfg2_sweep_joint|cfg2_sweep_joint_f64|cfg3_nx250|cfg3_demag]
    python bench.py --workload <wl> --full-run    # the config exactly as BASELINE.json states it: time to solution
    python bench.py --impl reference ...          # the fp64 CPU oracle on the host cores

A "step" is one Dormand-Prince RK45 step of the whole coupled system: six fused stage kernels
(field + LLG slope + overlap partials + stage combination + mode ODEs + controller), accepted or
rejected.  The metric is cell-stage updates/s = N_cells x right-hand-side evaluations / second
(SURVEY.md section 8(d)); simulated ns per wall-second is reported beside it.

Default workload: cfg3 = BASELINE.json configs[2] (256x256x32 cells, 8 cavity modes, fp32, adaptive
tol 1e-6) — the configuration the north_star's roofline target is quoted on ("2M+-cell grid with
8 cavity modes").  Inputs are synthetic and seeded (cavmag_workloads); the per-step working set
(11 cell fields + 8 profiles = 344 MB) is larger than the 126 MB L2.

Timing: CUDA events recorded on the stream the library launches on (a torch stream handed over
with cav_set_stream), barrier + synchronize on both sides, max over ranks.  The K timed steps are
ONE cav_run_steps call = one CUDA-graph launch whose WHILE node loops on the device.
N > 1: independent replicas (different seeds) per GPU, no data-path collective ("replicas only",
DESIGN.md) -> weak scaling.

`e2e`: the same metric through the C ABI with HOST buffers - every step of every simulation uploads m and a from
pinned host memory, takes one step and downloads m and a - with E2E_STREAMS independent simulations in flight (one host
thread and one stream each, so the copies of one overlap the step and the opposite-direction copies of the others);
`e2e.single_stream` is one such chain alone.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "cell-stage updates/s"
UNIT = "cell-stage/s"

# dram__bytes_read.sum + dram__bytes_write.sum per stage-kernel launch (mean over the six stages of
# one step) from the `ncu --set full` capture summarised in profiles/ (file named beside each value).
NCU_TRAFFIC_BYTES = {      # cold-cache captures (ncu flushes between replays); algorithmic bytes in brackets
    "cfg3": 208.6e6,       # profiles/r2_cfg3_stage_kernels.md      (222.3 MB)
    "cfg4": 136.1e6,       # profiles/r2_cfg4_stage_kernels.md      (159.4 MB)
    "cfg4_f64": 334.3e6,   # profiles/r2_cfg4_f64_stage_kernels.md  (318.8 MB)
    "cfg5": 3676.6e6,      # profiles/r2_cfg5_stage_kernels.md      (3389.0 MB): the halo
                           # rows / columns of the stage-state tiles miss L2 on a grid this large
}


def make_workload(name: str, rank: int = 0):
    import cavmag_workloads as W
    seed_shift = 17 * rank
    if name == "cfg3":
        return W.cfg3(seed=3000 + seed_shift, dtype=np.float32), "f32"
    if name == "cfg3_nx250":      # cfg3 with rows that are not a multiple of 16 bytes (padded inside the library, TMA path)
        return W.cfg3(nx=250, seed=3000 + seed_shift, dtype=np.float32), "f32"
    if name == "cfg3_demag":      # cfg3 with the optional dipolar field on (FFT convolution before every stage; generic kernels)
        return W.cfg3(seed=3000 + seed_shift, dtype=np.float32), "f32"
    if name == "cfg5":
        return W.cfg5(seed=5000 + seed_shift, dtype=np.float32), "f32"
    if name == "cfg4":
        return W.cfg4(seed=4000 + seed_shift), "f32"
    if name == "cfg4_f64":
        return W.cfg4(seed=4000 + seed_shift), "f64"
    if name == "cfg4d":
        return W.cfg4(seed=4000 + seed_shift, dissipative=True), "f32"
    if name == "cfg1":
        return W.cfg1("b", seed=1000 + seed_shift), "f64"
    if name == "cfg2":
        return W.cfg2(seed=2000 + seed_shift), "f32"
    if name == "cfg2_f64":
        return W.cfg2(seed=2000 + seed_shift), "f64"
    raise SystemExit(f"unknown workload {name}")


def algorithmic_bytes_per_cell_step(n_modes: int, n_sub: int, esize: int) -> int:
    """(111 + 6N) elements per cell per RK45 step, (222 + 6N) for two sublattices (SURVEY.md 8(d),
    DESIGN.md 'Algorithmic bytes'): 75 n_sub + 6N reads, 36 n_sub writes."""
    return (111 * n_sub + 6 * n_modes) * esize


def config_of(w, prec, name, gpus=1):
    """The workload, in the same words for the CUDA arm and the --impl reference arm (what differs between the arms -
    kernel path, launch mode, the oracle's bounded sample - is reported outside `config`)."""
    return {"workload": name, "grid": [w.nx, w.ny, w.nz], "cells": w.n_cells, "n_sub": w.n_sub,
            "parallelism": f"replicas x{gpus} (no collective)",
            "modes": w.n_modes, "cell_nm": w.dx * 1e9, "mode": "adaptive RK45 (Dormand-Prince 5(4))",
            "tol": w.tol, "precision": prec,
            "l2": "working set per step (11 cell fields + mode profiles) exceeds the 126 MB L2"
                  if (11 * 3 * w.n_sub + w.n_modes) * w.n_cells * (4 if prec == "f32" else 8) > 126e6
                  else "working set fits in L2 (latency-bound small case; no roofline claim)"}


# ----------------------------------------------------------------------------------------
# clocks during the timed region
# ----------------------------------------------------------------------------------------
class ClockSampler:
    """Samples SM clock and throttle reasons through NVML every 10 ms in a thread
    (nvidia-smi subprocess as a fallback)."""
    _REASONS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
                0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
                0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def __init__(self, index: int):
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop = threading.Event()
        self._thr = None
        self._nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nvml = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self._nvml = None

    def _once(self):
        if self._nvml is not None:
            p = self._nvml
            self.samples.append(p.nvmlDeviceGetClockInfo(self._h, p.NVML_CLOCK_SM))
            mask = p.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
            for bit, nm in self._REASONS.items():
                if mask & bit and nm != "gpu_idle":
                    self.reasons.add(nm)
        else:
            out = subprocess.run(["nvidia-smi", f"--id={self.index}", "--query-gpu=clocks.sm,clocks.max.sm,"
                                  "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
                                  "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap",
                                  "--format=csv,noheader,nounits"], capture_output=True, text=True).stdout.strip()
            f = [x.strip() for x in out.split(",")]
            if len(f) >= 6:
                self.samples.append(int(f[0])); self.max_mhz = int(f[1])
                for nm, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[2:6]):
                    if v.lower().startswith("active"):
                        self.reasons.add(nm)

    def _loop(self):
        while not self._stop.is_set():
            try:
                self._once()
            except Exception:
                pass
            self._stop.wait(0.01)

    def start(self):
        self._thr = threading.Thread(target=self._loop, daemon=True)
        self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr:
            self._thr.join()
        if not self.samples:
            try:
                self._once()
            except Exception:
                pass
        return {"sm_mhz": (statistics.median(self.samples) if self.samples else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ----------------------------------------------------------------------------------------
# the fp64 CPU oracle, timed as it stands (cpu_baseline leg and --impl reference)
# ----------------------------------------------------------------------------------------
def slab_workload(name: str, nz: int):
    """The workload's recipe on a thinner z-slab of the same x-y plane (bounded CPU sample)."""
    import cavmag_workloads as W
    base = name.split("_")[0]
    kw = dict(nz=nz)
    if base in ("cfg3", "cfg5"):
        kw["dtype"] = np.float64
    return W.by_name(base, **kw)


def time_oracle(w, steps: int, warmup: int, tol: float):
    """Runs warmup + steps adaptive RK45 steps of the oracle; returns (seconds, rhs_evals, sim_time) of the
    timed part."""
    from oracle import Oracle
    orc = Oracle(w)
    m, a, t, dt = w.m0, w.a0, 0.0, 0.0
    if warmup > 0:
        r = orc.run(m, a, t0=t, tol=tol, dt_init=dt, max_steps=warmup)
        m, a, t, dt = r.m, r.a, r.t, r.dt
    t0 = time.perf_counter()
    r = orc.run(m, a, t0=t, tol=tol, dt_init=dt, max_steps=steps)
    sec = time.perf_counter() - t0
    return sec, r.rhs_evals, r.t - t


def cpu_baseline(name: str, w_full, budget_s: float = 15.0):
    """Bounded sample: the oracle on a z-slab of the same workload, sized from a one-step calibration so
    that the timed part takes about budget_s seconds."""
    import oracle
    cores = oracle.get_threads()
    nz_cal = min(2, w_full.nz)
    wc = slab_workload(name, nz_cal)
    sec, evals, _ = time_oracle(wc, 1, 0, w_full.tol)
    per_cs = sec / (evals * wc.n_cells)                       # seconds per cell-stage
    plane = w_full.nx * w_full.ny
    # the whole grid if 3 steps of it fit the budget, else a thinner z-slab; then as many steps as the budget allows
    nz = int(max(1, min(w_full.nz, budget_s / (per_cs * plane * (6 * 3 + 1)))))
    ws = slab_workload(name, nz)
    steps = int(max(3, min(2000, budget_s / (per_cs * ws.n_cells * 6))))
    sec, evals, simt = time_oracle(ws, steps, 0, w_full.tol)
    for _ in range(3):                                        # the one-step calibration includes thread start-up:
        if sec >= 0.5 * budget_s or (nz >= w_full.nz and steps >= 2000):      # re-size from the measured rate
            break
        per_cs = sec / (evals * ws.n_cells)
        nz = int(max(1, min(w_full.nz, budget_s / (per_cs * plane * (6 * 3 + 1)))))
        ws = slab_workload(name, nz)
        steps = int(max(3, min(2000, budget_s / (per_cs * ws.n_cells * 6))))
        sec, evals, simt = time_oracle(ws, steps, 0, w_full.tol)
    out = {"value": ws.n_cells * evals / sec, "unit": UNIT, "cores": cores, "kind": "oracle",
           "sample": f"{name} recipe on a {ws.nx}x{ws.ny}x{ws.nz} slab ({ws.n_cells} cells, {ws.n_modes} modes), "
                     f"{steps} adaptive RK45 steps ({evals} RHS evaluations), fp64, {sec:.1f} s",
           "ms_per_step": 1e3 * sec / steps}
    # the same oracle on ONE thread: a thinner slab, about a third of the budget
    try:
        oracle.set_threads(1)
        per_cs1 = per_cs * cores                                  # first guess: perfect scaling
        nz1 = int(max(1, min(w_full.nz, (budget_s / 3.0) / (per_cs1 * plane * 6 * 3))))
        w1 = slab_workload(name, nz1)
        steps1 = int(max(2, min(200, (budget_s / 3.0) / (per_cs1 * w1.n_cells * 6))))
        sec1, evals1, _ = time_oracle(w1, steps1, 0, w_full.tol)
        out["one_thread"] = {"value": w1.n_cells * evals1 / sec1, "unit": UNIT, "cores": 1,
                             "sample": f"{name} recipe on a {w1.nx}x{w1.ny}x{w1.nz} slab, {steps1} adaptive RK45 steps "
                                       f"({evals1} RHS evaluations), fp64, {sec1:.1f} s"}
    finally:
        oracle.set_threads(cores)
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    name = args.workload
    w_full, prec = make_workload(name)
    cores = oracle.get_threads()
    # calibrate on a 2-plane slab, then size the slab so that warmup+steps take about 2 minutes
    wc = slab_workload(name, min(2, w_full.nz))
    sec, evals, _ = time_oracle(wc, 1, 0, w_full.tol)
    per_cs = sec / (evals * wc.n_cells)
    total_steps = args.steps + args.warmup
    plane = w_full.nx * w_full.ny
    nz = int(max(1, min(w_full.nz, 120.0 / (per_cs * plane * (6 * total_steps + 2)))))
    ws = slab_workload(name, nz)
    sec, evals, simt = time_oracle(ws, args.steps, args.warmup, w_full.tol)
    value = ws.n_cells * evals / sec
    sample = (f"{name} recipe on a {ws.nx}x{ws.ny}x{ws.nz} slab ({ws.n_cells} cells, {ws.n_modes} modes) per step; "
              f"{args.steps} timed adaptive RK45 steps after {args.warmup} warm-up steps, fp64")
    cfg = config_of(w_full, prec, name, args.gpus)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sec / max(args.steps, 1),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": cfg, "sim_ns_per_s": simt * 1e9 / sec,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "impl_config": {"reference_sample": sample, "arithmetic": "f64"},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------
# replicas-only aggregation: no data-path collective, only the timing protocol
# ----------------------------------------------------------------------------------------
def aggregate_over_ranks(ms: float, e2e_s: float, units: float, e2e_units: float, sim_t: float, world: int, device):
    """Whole-job numbers of N independent replicas: time = MAX over ranks, work = SUM over ranks.
    Works on any torch.distributed backend (nccl on the GPUs, gloo in the CPU tests)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms, e2e_s], dtype=torch.float64, device=device)
    u = torch.tensor([units, e2e_units, sim_t], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    ms_max, e2e_max = float(t[0]), float(t[1])
    return {"ms_max": ms_max, "e2e_s_max": e2e_max, "units": float(u[0]), "e2e_units": float(u[1]),
            "sim_t_sum": float(u[2]), "value": float(u[0]) / (ms_max * 1e-3), "e2e_value": float(u[1]) / e2e_max}


# ----------------------------------------------------------------------------------------
# the CUDA path
# ----------------------------------------------------------------------------------------
def hbm_peak():
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_path):
        return float(json.load(open(peaks_path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def demag_bytes_per_evaluation(w, esize):
    """Algorithmic bytes of the dipolar-field chain in front of one stage kernel, every array counted once
    per kernel that must stream it and every 2-D transform as ONE read + ONE write of its array (cuFFT takes two passes):
    gather (state in, nz planes padded in x and y out), R2C, z convolution (spectrum in and out + the real octant of the
    tensor's transform), C2R, scatter (corner in, field out), and the field's three components read by the stage kernel."""
    nx, ny, nz = w.nx, w.ny, w.nz
    Px, Py = (2 * nx if nx > 1 else 1), (2 * ny if ny > 1 else 1)
    Pz = 1
    while Pz < 2 * nz - 1:
        Pz *= 2
    nc, real2, cplx2 = nx * ny * nz, Px * Py * nz, nz * Py * (Px // 2 + 1)
    octant = 6 * (Pz // 2 + 1) * (Py // 2 + 1) * (Px // 2 + 1)
    gather = 3 * w.n_sub * nc + 3 * real2
    r2c = 3 * real2 + 3 * 2 * cplx2
    zconv = 2 * 3 * 2 * cplx2 + octant
    c2r = 3 * 2 * cplx2 + 3 * real2
    scatter = 2 * 3 * nc
    return esize * (gather + r2c + zconv + c2r + scatter + 3 * nc)


def roofline_of(name, w, prec, ms, steps):
    """Algorithmic bytes of one stage-kernel launch (mean of the six stages of a step) over its mean duration."""
    esize = 4 if prec == "f32" else 8
    launch_us = ms * 1e3 / (6 * steps)
    bytes_per_launch = algorithmic_bytes_per_cell_step(w.n_modes, w.n_sub, esize) * w.n_cells / 6.0
    if name.endswith("_demag"):          # one evaluation = the FFT-convolution chain + the stage kernel that adds its field
        bytes_per_launch += demag_bytes_per_evaluation(w, esize)
        achieved = bytes_per_launch / (launch_us * 1e-6) / 1e9
        peak, peak_src = hbm_peak()
        return {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                "peak_source": peak_src, "kernel": "one evaluation: k_demag_gather, cuFFT R2C, k_demag_zconv, cuFFT C2R, "
                "k_demag_scatter, cavmag::k_stage (dipolar-field instantiation)", "launch_us": launch_us,
                "algorithmic_bytes_per_launch": bytes_per_launch, "frac_of_nominal_8TBs": achieved / 8000.0}
    achieved = bytes_per_launch / (launch_us * 1e-6) / 1e9
    peak, peak_src = hbm_peak()
    return {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
            "traffic": NCU_TRAFFIC_BYTES.get(name), "peak_source": peak_src, "kernel": "cavmag::k_stage_tma / k_stage (fused RK45 stage)",
            "launch_us": launch_us, "algorithmic_bytes_per_launch": bytes_per_launch,
            "frac_of_nominal_8TBs": achieved / 8000.0}


def timed_steps(api, torch, h, stream, tol, steps, sampler=None, barrier=None):
    """K steps = ONE cav_run_steps call (one CUDA-graph launch), CUDA events on the launching stream."""
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if barrier:
        barrier()
    if sampler:
        sampler.start()
    ev0.record(stream)
    api.cav_run_steps(h, math.inf, tol=tol, max_steps=steps)
    ev1.record(stream)
    stream.synchronize()
    if barrier:
        barrier()
    clocks = sampler.stop() if sampler else None
    return ev0.elapsed_time(ev1), clocks


E2E_STREAMS = 8     # independent simulations in flight in the end-to-end measurement (one host thread and one stream each)


def e2e_pipelined(api, torch, w, prec, tol, k, spinup, barrier, n_streams=E2E_STREAMS):
    """End to end through the C ABI with host buffers, as a host application that integrates several independent
    simulations would drive it: n_streams simulations of the same workload, one host thread and one CUDA stream each,
    every step of every simulation = cav_set_m / cav_set_a from pinned host memory, cav_run_steps(1), cav_get_m /
    cav_get_a back to the host.  A single chain is bound by upload + step + download in series (PCIe, ~1.2 ms for CFG3);
    with several chains the copies of one overlap the step and the opposite-direction copies of the others.
    Returns (seconds, right-hand-side evaluations of all simulations)."""
    import threading
    N = w.n_modes
    sims, hosts = [], []
    for _ in range(n_streams):
        st = torch.cuda.Stream()
        sim = api.Sim(w, precision=prec, stream=st.cuda_stream)
        sim._stream_keepalive = st
        api.cav_run_steps(sim.h, math.inf, tol=tol, max_steps=spinup)
        mh = torch.empty(sim.shape_m, dtype=torch.float32 if prec == "f32" else torch.float64).pin_memory()
        api.cav_get_m(sim.h, mh)
        sims.append(sim); hosts.append(mh)

    errors = []

    def chain(i, n):
        try:
            h, mh = sims[i].h, hosts[i]
            a = api.cav_get_a(h, N)
            for _ in range(n):
                api.cav_set_m(h, mh)                  # H2D from pinned host memory
                api.cav_set_a(h, a)
                api.cav_run_steps(h, math.inf, tol=tol, max_steps=1)
                api.cav_get_m(h, mh)                  # D2H of the step's result (synchronises this simulation's stream)
                a = api.cav_get_a(h, N)
        except Exception as e:                        # a failed chain must fail the measurement, not shorten it silently
            errors.append(e)

    for i in range(n_streams):
        chain(i, 3)                                   # warm-up of the host-buffer path
    if errors:
        raise errors[0]
    ev0 = [api.cav_get_stats(q.h)["rhs_evals"] for q in sims]
    barrier()
    t0 = time.perf_counter()
    threads = [threading.Thread(target=chain, args=(i, k)) for i in range(n_streams)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    torch.cuda.synchronize()
    seconds = time.perf_counter() - t0
    if errors:
        raise errors[0]
    barrier()
    evals = sum(api.cav_get_stats(q.h)["rhs_evals"] - e for q, e in zip(sims, ev0))
    for q in sims:
        q.close()
    return seconds, evals


def measure_extra(api, torch, name, args, local):
    """One more large workload in the same process (device-resident timing only): value, ms per step, roofline
    fraction and the clocks seen during its timed region."""
    w, prec = make_workload(name, 0)
    stream = torch.cuda.Stream()
    with api.Sim(w, precision=prec, stream=stream.cuda_stream) as sim:
        h = sim.h
        path_used = {api.CAV_PATH_GENERIC: "generic", api.CAV_PATH_TMA: "tma", api.CAV_PATH_BLOCK: "block",
                     api.CAV_PATH_COOP: "coop"}[api.cav_get_kernel_path(h)]
        api.cav_run_steps(h, math.inf, tol=w.tol, max_steps=args.spinup)
        api.cav_run_steps(h, math.inf, tol=w.tol, max_steps=max(args.warmup, 3))
        api.cav_sync(h)
        st0 = api.cav_get_stats(h)
        steps = args.extra_steps
        sampler = ClockSampler(torch.cuda.current_device() if os.environ.get("CUDA_VISIBLE_DEVICES") is None else local)
        ms, clocks = timed_steps(api, torch, h, stream, w.tol, steps, sampler)
        api.cav_sync(h)
        st1 = api.cav_get_stats(h)
        evals = st1["rhs_evals"] - st0["rhs_evals"]
        assert evals == 6 * steps, (name, evals)
        m = sim.get_m()
    assert np.isfinite(m).all() and abs(float(np.abs(np.linalg.norm(m.astype(np.float64), axis=1) - 1).max())) < 1e-5
    return {"value": w.n_cells * evals / (ms * 1e-3), "unit": UNIT, "steps": steps, "ms_per_step": ms / steps,
            "dtype": prec, "config": config_of(w, prec, name), "kernel_path": path_used,
            "accepted": st1["accepted"] - st0["accepted"], "rejected": st1["rejected"] - st0["rejected"],
            "sim_ns_per_s": (st1["t"] - st0["t"]) * 1e9 / (ms * 1e-3),
            "roofline": roofline_of(name, w, prec, ms, steps), "clocks": clocks}


def run_cuda(args):
    import torch
    import torch.distributed as dist
    from paper_2603_03706_b200 import api          # raises if libcavmag.so is missing: no CPU fallback

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    name = args.workload
    w, prec = make_workload(name, rank)
    esize = 4 if prec == "f32" else 8
    tol = w.tol
    stream = torch.cuda.Stream()
    path = {"auto": None, "generic": api.CAV_PATH_GENERIC, "tma": api.CAV_PATH_TMA, "block": api.CAV_PATH_BLOCK, "coop": api.CAV_PATH_COOP}[args.kernel_path]
    sim = api.Sim(w, precision=prec, stream=stream.cuda_stream, path=path)
    h = sim.h
    path_used = {api.CAV_PATH_GENERIC: "generic", api.CAV_PATH_TMA: "tma", api.CAV_PATH_BLOCK: "block", api.CAV_PATH_COOP: "coop"}[api.cav_get_kernel_path(h)]
    if name.endswith("_demag"):
        api.cav_set_demag(h, 1)
        path_used = "generic + FFT convolution (x: cuFFT on the occupied rows; y, z and the product: own kernels; captured into the run graph)"
    if args.no_stage_overlap:
        api.cav_set_stage_overlap(h, 0)
    if args.no_serpentine:
        api.cav_set_sweep_order(h, 0)
    N, nc = w.n_modes, w.n_cells

    # spin-up (setup, untimed): the controller grows dt from 1e-14 s to the stability-limited step
    if args.launch_mode == "stream":                  # profiling aid: host-enqueued stage kernels, same kernels
        api.cav_set_launch_mode(h, api.CAV_LAUNCH_STREAM)
    api.cav_run_steps(h, math.inf, tol=tol, max_steps=args.spinup)
    # warm-up: W steps (both run graphs - one step and four steps per WHILE iteration - are instantiated and uploaded by the
    # first run; the spin-up above has already gone through the long-run graph that the timed launch uses)
    api.cav_run_steps(h, math.inf, tol=tol, max_steps=max(args.warmup, 1))
    api.cav_sync(h)
    st0 = api.cav_get_stats(h)
    n0 = api.cav_get_launch_count(h)
    sampler = ClockSampler(torch.cuda.current_device() if os.environ.get("CUDA_VISIBLE_DEVICES") is None else local)
    ms, clocks = timed_steps(api, torch, h, stream, tol, args.steps, sampler, barrier)
    overlap_active = api.cav_get_stage_overlap(h)
    api.cav_sync(h)                                   # raises on a device-side error status
    st1 = api.cav_get_stats(h)
    n1 = api.cav_get_launch_count(h)
    evals = st1["rhs_evals"] - st0["rhs_evals"]
    steps_done = (st1["accepted"] + st1["rejected"]) - (st0["accepted"] + st0["rejected"])
    # the single-block path (grids up to 1024 cells) re-evaluates k1 at the start of a run: one more evaluation
    assert steps_done == args.steps and evals in (6 * args.steps, 6 * args.steps + 1), (steps_done, evals)
    sim_t = st1["t"] - st0["t"]
    # SURVEY.md 8(d) "median of 5": the same K-step launch five more times (reported beside the contract's one timed region)
    rep_ms = [timed_steps(api, torch, h, stream, tol, args.steps)[0] for _ in range(args.repeats)]
    api.cav_sync(h)

    # ---- e2e: host buffers through the C ABI, copies inside the timed region, every step ----
    k_e2e = min(args.steps, args.e2e_steps)
    m_host = torch.empty(sim.shape_m, dtype=torch.float32 if prec == "f32" else torch.float64).pin_memory()
    api.cav_get_m(h, m_host)
    a_host = api.cav_get_a(h, N)
    for _ in range(3):                                # warm-up of the host-buffer path
        api.cav_set_m(h, m_host); api.cav_set_a(h, a_host)
        api.cav_run_steps(h, math.inf, tol=tol, max_steps=1)
        api.cav_get_m(h, m_host); a_host = api.cav_get_a(h, N)
    se0 = api.cav_get_stats(h)
    barrier()
    t0 = time.perf_counter()
    for _ in range(k_e2e):
        api.cav_set_m(h, m_host)                      # H2D from pinned host memory
        api.cav_set_a(h, a_host)
        api.cav_run_steps(h, math.inf, tol=tol, max_steps=1)
        api.cav_get_m(h, m_host)                      # D2H of the step's result (synchronises)
        a_host = api.cav_get_a(h, N)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    barrier()
    se1 = api.cav_get_stats(h)
    e2e1_evals = se1["rhs_evals"] - se0["rhs_evals"]
    e2e1_s = e2e_s
    io_bytes = int(np.prod(sim.shape_m)) * esize + 16 * N
    sim.close()
    # the same with E2E_STREAMS independent simulations in flight (the end-to-end figure of the line)
    e2e_s, e2e_evals = e2e_pipelined(api, torch, w, prec, tol, k_e2e, args.spinup, barrier)

    # ---- max over ranks, sum of units ----
    agg = aggregate_over_ranks(ms, e2e_s, float(nc * evals), float(nc * e2e_evals), sim_t, world, "cuda")
    ms_max, e2e_max = agg["ms_max"], agg["e2e_s_max"]
    value, e2e_value = agg["value"], agg["e2e_value"]
    units = [agg["units"], agg["e2e_units"], agg["sim_t_sum"]]

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": prec, "data": "synthetic",
            "config": config_of(w, prec, name, world),
            "impl_config": {"launch_mode": args.launch_mode, "kernel_path": path_used,
                            "stage_overlap": bool(overlap_active), "serpentine": not args.no_serpentine},
            "sim_ns_per_s": float(units[2]) * 1e9 / (ms_max * 1e-3) / world,
            "mean_dt_ps": sim_t * 1e12 / max(st1["accepted"] - st0["accepted"], 1),
            "accepted": st1["accepted"] - st0["accepted"], "rejected": st1["rejected"] - st0["rejected"],
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": io_bytes, "d2h_bytes_per_step": io_bytes,
                    "steps": k_e2e, "simulations_in_flight": E2E_STREAMS, "ms_per_step": 1e3 * e2e_max / (k_e2e * E2E_STREAMS),
                    "single_stream": {"value": nc * e2e1_evals / e2e1_s, "ms_per_step": 1e3 * e2e1_s / k_e2e,
                                      "note": "one simulation: upload, step and download in series (this rank)"},
                    "note": "every step of every simulation: cav_set_m/cav_set_a from pinned host memory, cav_run_steps(1), "
                            "cav_get_m/cav_get_a to host; FSAL is lost at each upload (7 RHS evaluations per step); "
                            f"{E2E_STREAMS} independent simulations of the workload, one host thread and one stream each, so "
                            "that the copies of one overlap the step and the opposite-direction copies of the others; "
                            "bytes are per step of one simulation"},
            "gpu_launches": int(n1 - n0),
            "roofline": roofline_of(name, w, prec, ms, args.steps),
        }
        if rep_ms:
            med = statistics.median(rep_ms)
            line["repeats"] = {"n": len(rep_ms), "ms_per_step": [x / args.steps for x in rep_ms],
                               "ms_per_step_median": med / args.steps, "value_median": nc * 6 * args.steps / (med * 1e-3),
                               "roofline_frac_median": roofline_of(name, w, prec, med, args.steps)["frac"],
                               "note": "the same K-step graph launch repeated (this rank), after the contract's timed region"}
        if world == 1 and not args.no_extras and name == "cfg3":
            # the other large configs of BASELINE.json, measured in the same process (device-resident timing)
            line["workloads"] = {}
            for extra in ("cfg4", "cfg4_f64", "cfg5"):
                try:
                    line["workloads"][extra] = measure_extra(api, torch, extra, args, local)
                except Exception as e:              # an extra must never cost the headline line
                    line["workloads"][extra] = {"error": f"{type(e).__name__}: {e}"}
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(name, w)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()



# ----------------------------------------------------------------------------------------
# batched small-grid sweep: --workload cfg1_sweep
# ----------------------------------------------------------------------------------------
FLOP_PER_CELL_STAGE_BATCH = 151.0     # measured: fp64 add + mul + 2 fma of k_batch per cell-stage (profiles/r2_batch_flops.md); the formulas give ~150


def run_batch(args):
    """BASELINE.json configs[0] (8x8x8 cells, one uniform mode, fp64, adaptive tol 1e-8) as a field sweep of
    --replicas independent simulations (41 Kittel frequencies, cyclic) integrated by ONE kernel launch."""
    import torch
    import cavmag_workloads as W
    from paper_2603_03706_b200 import api
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    w = W.cfg1("b")
    n_rep = args.replicas
    ghz = np.linspace(9.6, 10.4, 41)
    B0 = np.array([[0.0, 0.0, W.b0_for_ghz(ghz[r % 41])] for r in range(n_rep)])
    stream = torch.cuda.Stream()
    nc = w.n_cells
    with api.Batch(w, n_rep, precision="f64", B0=B0, stream=stream.cuda_stream) as b:
        b.run(math.inf, tol=w.tol, max_steps=args.spinup)
        b.run(math.inf, tol=w.tol, max_steps=max(args.warmup, 3))
        st0 = b.stats()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        sampler = ClockSampler(torch.cuda.current_device())
        torch.cuda.synchronize()
        sampler.start()
        ev0.record(stream)
        b.run(math.inf, tol=w.tol, max_steps=args.steps)
        ev1.record(stream)
        stream.synchronize()
        clocks = sampler.stop()
        ms = ev0.elapsed_time(ev1)
        st1 = b.stats()
        evals = sum(s1["rhs_evals"] - s0["rhs_evals"] for s0, s1 in zip(st0, st1))
        sim_t = sum(s1["t"] - s0["t"] for s0, s1 in zip(st0, st1))
        # e2e: host buffers through the C ABI, every step
        m_host = b.get_m()
        a_host = b.get_a()
        k_e2e = min(args.e2e_steps, 50)
        se0 = b.stats()
        t0 = time.perf_counter()
        for _ in range(k_e2e):
            api.cav_batch_set_m(b.h, m_host, per_replica=True)
            api.cav_batch_set_a(b.h, a_host, per_replica=True)
            b.run(math.inf, tol=w.tol, max_steps=1)
            m_host = b.get_m()
            a_host = b.get_a()
        e2e_s = time.perf_counter() - t0
        se1 = b.stats()
        e2e_evals = sum(s1["rhs_evals"] - s0["rhs_evals"] for s0, s1 in zip(se0, se1))
    # the same grid through cav_run (one simulation, six kernel launches per step): context for the batch number
    with api.Sim(w, precision="f64", stream=stream.cuda_stream) as sim:
        api.cav_run_steps(sim.h, math.inf, tol=w.tol, max_steps=args.spinup)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        api.cav_run_steps(sim.h, math.inf, tol=w.tol, max_steps=200)
        e1.record(stream)
        stream.synchronize()
        single = nc * 6 * 200 / (e0.elapsed_time(e1) * 1e-3)
    value = nc * evals / (ms * 1e-3)
    flops = value * FLOP_PER_CELL_STAGE_BATCH / 1e12
    peak = 148 * 64 * 2 * 1.965e9 / 1e12          # DFMA: 64 per clock per SM, 1965 MHz
    io = int(m_host.nbytes + a_host.nbytes)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": "cfg1_sweep", "grid": [w.nx, w.ny, w.nz], "cells": nc, "replicas": n_rep, "modes": 1,
                       "mode": "adaptive RK45, one thread block per replica (cav_batch_run)", "tol": w.tol,
                       "l2": "state lives in shared memory and registers (no per-stage global traffic)"},
            "sim_ns_per_s": sim_t * 1e9 / (ms * 1e-3), "clocks": clocks,
            "e2e": {"value": nc * e2e_evals / e2e_s, "unit": UNIT, "h2d_bytes_per_step": io, "d2h_bytes_per_step": io,
                    "steps": k_e2e, "ms_per_step": 1e3 * e2e_s / k_e2e},
            "gpu_launches": 1,
            "roofline": {"bound": "alu", "achieved": flops, "peak": peak, "unit": "TFLOP/s", "frac": flops / peak,
                         "traffic": None, "kernel": "cavmag::k_batch",
                         "note": "fp64 vector peak derived from unit counts; the kernel is barrier/latency-bound "
                                 "(15 block barriers per step on a 512-thread block)"},
            "single_simulation_cell_stage_per_s": single,
            "speedup_vs_one_simulation_at_a_time": value / single}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------
# the 41-point field sweep of configs[1] as concurrent simulations: --workload cfg2_sweep
# ----------------------------------------------------------------------------------------
def run_concurrent_sweep(args):
    """BASELINE.json configs[1] (64x64x16 cells, two sine modes, fp32, adaptive tol 1e-6) at its 41 field values:
    41 independent cav_run graphs on 41 streams, launched back to back (cav_run_steps is asynchronous), timed by
    CUDA events on a master stream that every simulation stream waits on / is waited for."""
    import torch
    import cavmag_workloads as W
    from paper_2603_03706_b200 import api
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    ghz = W.cfg2_sweep_ghz()
    ws = [W.cfg2(f_kittel_ghz=float(f), seed=2000 + i) for i, f in enumerate(ghz)]
    streams = [torch.cuda.Stream() for _ in ws]
    # the generic stage kernels: graphs of different simulations overlap (cooperative grids would serialise)
    sims = [api.Sim(w, precision="f32", stream=st.cuda_stream, path=api.CAV_PATH_GENERIC) for w, st in zip(ws, streams)]
    tol, nc, N = ws[0].tol, ws[0].n_cells, ws[0].n_modes
    master = torch.cuda.Stream()

    def run_all(k):
        ev0 = torch.cuda.Event(enable_timing=True); ev1 = torch.cuda.Event(enable_timing=True)
        ev0.record(master)
        ends = []
        for sim, st in zip(sims, streams):
            st.wait_event(ev0)
            api.cav_run_steps(sim.h, math.inf, tol=tol, max_steps=k)
            e = torch.cuda.Event(); e.record(st); ends.append(e)
        for e in ends:
            master.wait_event(e)
        ev1.record(master)
        master.synchronize()
        return ev0.elapsed_time(ev1)

    run_all(args.spinup)
    run_all(max(args.warmup, 3))
    st0 = [api.cav_get_stats(s.h) for s in sims]
    sampler = ClockSampler(torch.cuda.current_device())
    torch.cuda.synchronize()
    sampler.start()
    ms = run_all(args.steps)
    clocks = sampler.stop()
    st1 = [api.cav_get_stats(s.h) for s in sims]
    evals = sum(b["rhs_evals"] - a["rhs_evals"] for a, b in zip(st0, st1))
    sim_t = sum(b["t"] - a["t"] for a, b in zip(st0, st1))
    # one simulation alone, same graph: the latency-bound single-run number
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(streams[0]); api.cav_run_steps(sims[0].h, math.inf, tol=tol, max_steps=args.steps); e1.record(streams[0])
    streams[0].synchronize()
    single = nc * 6 * args.steps / (e0.elapsed_time(e1) * 1e-3)
    # e2e: host buffers, every step, all simulations
    k_e2e = min(args.e2e_steps, 20)
    hosts = [torch.empty(s.shape_m, dtype=torch.float32).pin_memory() for s in sims]
    for s, hbuf in zip(sims, hosts):
        api.cav_get_m(s.h, hbuf)
    a_hosts = [api.cav_get_a(s.h, N) for s in sims]
    se0 = [api.cav_get_stats(s.h) for s in sims]
    t0 = time.perf_counter()
    for _ in range(k_e2e):
        for i, s in enumerate(sims):
            api.cav_set_m(s.h, hosts[i]); api.cav_set_a(s.h, a_hosts[i])
            api.cav_run_steps(s.h, math.inf, tol=tol, max_steps=1)
        for i, s in enumerate(sims):
            api.cav_get_m(s.h, hosts[i]); a_hosts[i] = api.cav_get_a(s.h, N)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    se1 = [api.cav_get_stats(s.h) for s in sims]
    e2e_evals = sum(b["rhs_evals"] - a["rhs_evals"] for a, b in zip(se0, se1))
    launches = sum(api.cav_get_launch_count(s.h) for s in sims)
    for s in sims:
        s.close()
    value = nc * evals / (ms * 1e-3)
    bytes_per_cs = algorithmic_bytes_per_cell_step(N, 1, 4) / 6.0
    achieved = value * bytes_per_cs / 1e9
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    peak = float(json.load(open(peaks_path))["hbm_gbs"]) if os.path.exists(peaks_path) else 6650.0
    io = int(np.prod(sims[0].shape_m)) * 4 * len(sims) + 16 * N * len(sims)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": "cfg2_sweep", "grid": [ws[0].nx, ws[0].ny, ws[0].nz], "cells": nc, "simulations": len(sims),
                       "modes": N, "mode": "adaptive RK45; 41 cav_run graphs on 41 streams", "tol": tol,
                       "l2": "41 x 8.7 MB of cell fields = 355 MB in total exceeds the 126 MB L2"},
            "sim_ns_per_s": sim_t * 1e9 / (ms * 1e-3), "clocks": clocks,
            "e2e": {"value": nc * e2e_evals / e2e_s, "unit": UNIT, "h2d_bytes_per_step": io, "d2h_bytes_per_step": io,
                    "steps": k_e2e, "ms_per_step": 1e3 * e2e_s / k_e2e},
            "gpu_launches": int(launches),
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": None, "kernel": "cavmag::k_stage (generic path, 128 blocks per launch, 41 concurrent graphs)"},
            "single_simulation_cell_stage_per_s": single,
            "speedup_vs_one_simulation_at_a_time": value / single}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------
# --full-run: the configuration exactly as BASELINE.json states it, from t = 0 to its t_end
# ----------------------------------------------------------------------------------------
def run_joint_sweep(args):
    """BASELINE.json configs[1] at its 41 field values through cav_sweep_run: ONE device-side loop over all 41
    simulations - their plane-tiles form one work list for the persistent TMA grid, every simulation keeps its own step
    size and accept/reject decisions."""
    import torch
    import cavmag_workloads as W
    from paper_2603_03706_b200 import api
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    prec = "f64" if args.workload.endswith("_f64") else "f32"            # configs[1]: "fp32 and fp64"
    esize = 4 if prec == "f32" else 8
    tdtype = torch.float32 if prec == "f32" else torch.float64
    ghz = W.cfg2_sweep_ghz()
    ws = [W.cfg2(f_kittel_ghz=float(f), seed=2000 + i) for i, f in enumerate(ghz)]
    stream = torch.cuda.Stream()
    sims = [api.Sim(w, precision=prec, stream=stream.cuda_stream) for w in ws]
    sw = api.cav_sweep_create(sims)
    tol, nc, N = ws[0].tol, ws[0].n_cells, ws[0].n_modes

    def run_all(k):
        ev0 = torch.cuda.Event(enable_timing=True); ev1 = torch.cuda.Event(enable_timing=True)
        ev0.record(stream)
        api.cav_sweep_run(sw, math.inf, tol=tol, max_steps=k)
        ev1.record(stream)
        stream.synchronize()
        return ev0.elapsed_time(ev1)

    run_all(args.spinup)
    run_all(max(args.warmup, 3))
    st0 = [api.cav_get_stats(s.h) for s in sims]
    sampler = ClockSampler(torch.cuda.current_device())
    torch.cuda.synchronize()
    sampler.start()
    ms = run_all(args.steps)
    clocks = sampler.stop()
    st1 = [api.cav_get_stats(s.h) for s in sims]
    rep_ms = [run_all(args.steps) for _ in range(args.repeats)]
    evals = sum(b["rhs_evals"] - a["rhs_evals"] for a, b in zip(st0, st1))
    sim_t = sum(b["t"] - a["t"] for a, b in zip(st0, st1))
    assert evals == 6 * args.steps * len(sims), evals
    # e2e: host buffers of all simulations every step
    k_e2e = min(args.e2e_steps, 20)
    hosts = [torch.empty(s.shape_m, dtype=tdtype).pin_memory() for s in sims]
    for s, hbuf in zip(sims, hosts):
        api.cav_get_m(s.h, hbuf)
    a_hosts = [api.cav_get_a(s.h, N) for s in sims]
    se0 = [api.cav_get_stats(s.h) for s in sims]
    t0 = time.perf_counter()
    for _ in range(k_e2e):
        for i, s in enumerate(sims):
            api.cav_set_m(s.h, hosts[i]); api.cav_set_a(s.h, a_hosts[i])
        api.cav_sweep_run(sw, math.inf, tol=tol, max_steps=1)
        for i, s in enumerate(sims):
            api.cav_get_m(s.h, hosts[i]); a_hosts[i] = api.cav_get_a(s.h, N)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    se1 = [api.cav_get_stats(s.h) for s in sims]
    e2e_evals = sum(b["rhs_evals"] - a["rhs_evals"] for a, b in zip(se0, se1))
    api.cav_sweep_destroy(sw)
    for s in sims:
        s.close()
    value = nc * evals / (ms * 1e-3)
    bytes_per_cs = algorithmic_bytes_per_cell_step(N, 1, esize) / 6.0
    achieved = value * bytes_per_cs / 1e9
    peak, peak_src = hbm_peak()
    io = int(np.prod(sims[0].shape_m)) * esize * len(sims) + 16 * N * len(sims)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": prec, "data": "synthetic",
            "config": {"workload": args.workload, "grid": [ws[0].nx, ws[0].ny, ws[0].nz], "cells": nc, "simulations": len(sims),
                       "modes": N, "mode": "adaptive RK45; 41 simulations in one device-side loop (cav_sweep_run)", "tol": tol,
                       "precision": prec,
                       "l2": f"41 x {8.7 * esize / 4:.1f} MB of cell fields = {355 * esize // 4} MB in total exceeds the 126 MB L2"},
            "sim_ns_per_s": sim_t * 1e9 / (ms * 1e-3), "clocks": clocks,
            "e2e": {"value": nc * e2e_evals / e2e_s, "unit": UNIT, "h2d_bytes_per_step": io, "d2h_bytes_per_step": io,
                    "steps": k_e2e, "ms_per_step": 1e3 * e2e_s / k_e2e},
            "gpu_launches": 6 * args.steps + 4 + len(sims),
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": None, "peak_source": peak_src, "kernel": "cavmag::k_stage_tma_sweep (joint launch over 41 simulations)"}}
    if rep_ms:
        med = statistics.median(rep_ms)
        line["repeats"] = {"n": len(rep_ms), "ms_per_step_median": med / args.steps, "roofline_frac_median": achieved / peak * ms / med}
    print(json.dumps(line), flush=True)


def run_full(args):
    """Time to solution of one BASELINE.json config (adaptive tol, its own duration): ONE cav_run call = one launch of the
    device-side step loop; wall time by CUDA events; |m| = 1, finiteness and the step statistics are checked."""
    import torch
    from paper_2603_03706_b200 import api
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    name = args.workload
    w, prec = make_workload(name)
    stream = torch.cuda.Stream()
    with api.Sim(w, precision=prec, stream=stream.cuda_stream) as sim:
        api.cav_set_trace(sim.h, w.t_end / 1000.0, 1000)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        ev0.record(stream)
        api.cav_run(sim.h, w.t_end, tol=w.tol)
        ev1.record(stream)
        stream.synchronize()
        sec = ev0.elapsed_time(ev1) * 1e-3
        st = api.cav_get_stats(sim.h)
        m = sim.get_m()
        a = sim.get_a()
        tr = api.cav_get_trace(sim.h)
        path_used = api.cav_get_kernel_path(sim.h)
    norm_err = float(np.abs(np.linalg.norm(m.astype(np.float64), axis=1) - 1.0).max())
    assert st["t"] == w.t_end and np.isfinite(m).all() and np.isfinite(a).all() and tr.shape[0] == 1000
    line = {"metric": "time to solution", "value": sec, "unit": "s", "higher_is_better": False, "n_gpus": 1,
            "dtype": prec, "data": "synthetic",
            "config": dict(config_of(w, prec, name), t_end_ns=w.t_end * 1e9),
            "impl_config": {"kernel_path": {1: "generic", 2: "tma", 3: "block", 4: "coop"}[path_used]},
            "accepted": st["accepted"], "rejected": st["rejected"], "rhs_evals": st["rhs_evals"],
            "mean_dt_ps": w.t_end * 1e12 / max(st["accepted"], 1), "dt_min_ps": st["dt_min"] * 1e12, "dt_max_ps": st["dt_max"] * 1e12,
            "sim_ns_per_s": w.t_end * 1e9 / sec, "cell_stage_per_s": w.n_cells * st["rhs_evals"] / sec,
            "max_norm_error": norm_err, "max_abs_a": float(np.abs(a).max()) if a.size else 0.0, "trace_rows": int(tr.shape[0])}
    print(json.dumps(line), flush=True)


def run_full_sweep(args):
    """BASELINE.json configs[1] exactly as stated: B0 swept over 41 values, each run 50 ns from t = 0, adaptive - all 41
    simulations in ONE cav_sweep_run call (one launch of the joint device-side loop), a 1000-sample spectrum pair per
    simulation accumulated on the device (cav_set_spectrum) instead of 41 traces."""
    import torch
    import cavmag_workloads as W
    from paper_2603_03706_b200 import api
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    prec = "f64" if args.workload.endswith("_f64") else "f32"
    ghz = W.cfg2_sweep_ghz()
    ws = [W.cfg2(f_kittel_ghz=float(f), seed=2000 + i) for i, f in enumerate(ghz)]
    stream = torch.cuda.Stream()
    sims = [api.Sim(w, precision=prec, stream=stream.cuda_stream) for w in ws]
    t_end, tol, nc, N = ws[0].t_end, ws[0].tol, ws[0].n_cells, ws[0].n_modes
    K = 401
    for s in sims:
        api.cav_set_trace(s.h, t_end / 1000.0, 1000)
        api.cav_set_spectrum(s.h, K, 2 * math.pi * 9.5e9, 2 * math.pi * 10.5e9)
    sw = api.cav_sweep_create(sims)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    ev0.record(stream)
    api.cav_sweep_run(sw, t_end, tol=tol)
    ev1.record(stream)
    stream.synchronize()
    sec = ev0.elapsed_time(ev1) * 1e-3
    stats = [api.cav_get_stats(s.h) for s in sims]
    samples = [api.cav_get_spectrum(s.h, K, N)[1] for s in sims]
    norm_err = 0.0
    for s in sims:
        m = s.get_m()
        assert np.isfinite(m).all()
        norm_err = max(norm_err, float(np.abs(np.linalg.norm(m.astype(np.float64), axis=1) - 1.0).max()))
    api.cav_sweep_destroy(sw)
    for s in sims:
        s.close()
    assert all(st["t"] == t_end for st in stats) and all(n == 1000 for n in samples)
    evals = sum(st["rhs_evals"] for st in stats)
    line = {"metric": "time to solution", "value": sec, "unit": "s", "higher_is_better": False, "n_gpus": 1, "dtype": prec,
            "data": "synthetic",
            "config": {"workload": args.workload, "grid": [ws[0].nx, ws[0].ny, ws[0].nz], "cells": nc, "simulations": len(sims),
                       "modes": N, "t_end_ns": t_end * 1e9, "tol": tol, "precision": prec,
                       "mode": "adaptive RK45; 41 field points in one device-side loop (cav_sweep_run), spectra on the device"},
            "accepted": [min(st["accepted"] for st in stats), max(st["accepted"] for st in stats)],
            "rejected": sum(st["rejected"] for st in stats), "rhs_evals": evals,
            "sim_ns_per_s": len(sims) * t_end * 1e9 / sec, "cell_stage_per_s": nc * evals / sec, "max_norm_error": norm_err,
            "spectrum_samples_per_simulation": 1000}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3000)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--e2e-steps", type=int, default=300)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the cfg4 / cfg4_f64 / cfg5 sub-records of the default cfg3 run")
    ap.add_argument("--extra-steps", type=int, default=300, help="timed steps of each extra workload")
    ap.add_argument("--repeats", type=int, default=5, help="extra repetitions of the K-step launch (median reported)")
    ap.add_argument("--spinup", type=int, default=40, help="untimed setup steps that let dt settle")
    ap.add_argument("--launch-mode", default="graph", choices=["graph", "stream"])
    ap.add_argument("--kernel-path", default="auto", choices=["auto", "generic", "tma", "block", "coop"])
    ap.add_argument("--replicas", type=int, default=1184, help="cfg1_sweep: replicas in the batch")
    ap.add_argument("--full-run", action="store_true",
                    help="run the workload as BASELINE.json states it (t = 0 .. t_end, adaptive) and report the time to solution")
    ap.add_argument("--no-serpentine", action="store_true", help="every stage sweeps forward (A/B aid)")
    ap.add_argument("--no-stage-overlap", action="store_true", help="full dependencies between stage kernels (A/B aid)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "cuda":
        args.warmup = 3
    if args.full_run and args.workload in ("cfg2_sweep_joint", "cfg2_sweep_joint_f64"):
        run_full_sweep(args)
    elif args.full_run:
        run_full(args)
    elif args.impl == "reference":
        run_reference(args)
    elif args.workload == "cfg1_sweep":
        run_batch(args)
    elif args.workload == "cfg2_sweep":
        run_concurrent_sweep(args)
    elif args.workload in ("cfg2_sweep_joint", "cfg2_sweep_joint_f64"):
        run_joint_sweep(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
