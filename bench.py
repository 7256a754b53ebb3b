#!/usr/bin/env python
"""bench.py -- throughput of the batched spectra + NLL hot path (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config k] [--impl ours|reference]

A step = one phylino_nll call over the whole batch of parameter points of a workload (all rows of
SURVEY.md 8(a): per-point derivation, oscillation weights, energy scale + binning, scatter-add,
deterministic reduction, expectation assembly, NLL reduction).

Headline workload (`value`, `roofline`, `e2e`, `clocks`): BASELINE.json names no config for its metric, so
it is the LARGEST single-GPU one, configs[4] (sterile grid scan: 2 x 1e6 events x 4096 points = 8.19e9
event x point per step), timed for exactly K steps.  At one GPU the line also carries `configs`: all five
BASELINE.json configs measured in the same run, each with value, median / min / mean ms per step, the spectra
kernel's own duration and roofline fraction, dram traffic and end-to-end numbers; config 1 (one point, 1e5
events: launch-latency bound) with its single-call latencies; config 3 with the wall time of the 603-point
gradient step, dense and with cross-point caching.  `--config k` makes config k the headline and skips the rest.

N > 1 (torchrun): the path shards by parameter point with no data-path collective -- every rank
holds the event store and evaluates its own batch of points ("weak" scaling).
`--impl reference` times the CPU oracle (oracle/) on the host cores instead; that and the
`cpu_baseline` leg are the only places this file touches oracle/.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "oscillated event x param-point/s (batched spectra+NLL)"
UNIT = "event*point/s"
HEADLINE_CONFIG = 5
# ALGORITHMIC fp64-pipe instructions per event x point, unit-weight datasets (every
# BASELINE.json config).  Per oscillation term: 3 range reduction + 1 square + 5 Horner + the last Horner step; the
# two-term model accumulates with that last step itself (devmath.cuh half_cos_accumulate: 10), the three-term models
# form g and add it (11).  The SASS of the hot loop has exactly these (profiles/r2f_hot_loop_sass.md).  The
# bin/weight bookkeeping is per batch of events and per run, not per event x point.
def fp64_per_general_term(S: int) -> int:
    return 10 if S == 2 else 11
# ... and 6 for the LAST term where its phase stays below an eighth of a half-turn for every event and point of a
# group (no range reduction, a cubic instead of a quintic, accumulated with its last Horner step: devmath.cuh
# half_cos_small_accumulate); the library reports the fraction of event x point evaluations that took it
# (phylino_last_small_phase), the roofline counts what ran
FP64_SMALL_TERM = 6
# ... and 8 for the FIRST term where its phase cannot wrap for any event of a work item and any point of the group (no
# range reduction, no sign: devmath.cuh half_cos_medium_accumulate; phylino_last_medium_phase reports the fraction)
FP64_MEDIUM_TERM = 8
# nominal fp64 pipe, derived in DESIGN.md section 7 (the guide has no fp64 row): 64 fp64 lanes/clk/SM (one DFMA
# per lane and clock) x SMs x the SM clock nvidia-smi reports as maximum
FP64_LANES_PER_SM = 64
L2_FLUSH_BYTES = 256 << 20
EVENT_BYTES = 12            # unit-weight store: x fp64 + E_vis fp32 (every BASELINE.json config)


def n_terms(model) -> int:
    return 2 if model.osc_model == 0 else 3


def fp64_inst_per_evpt(model) -> int:
    S = n_terms(model)
    return fp64_per_general_term(S) * S


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown",
               0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake"}

    def __init__(self, index: int, period_s: float = 0.005):
        super().__init__(daemon=True)
        self.index, self.period = index, period_s
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._halt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self._halt.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                get = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
                    nv.nvmlDeviceGetCurrentClocksThrottleReasons
                bits = int(get(self.h))
                for b, name in self.REASONS.items():
                    if bits & b:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._halt.set()
        if self.is_alive():
            self.join()
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def physical_gpu_index(local: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local])
        except Exception:
            return local
    return local


def traffic_from_profile(config: int):
    """(dram bytes read + written per launch of the spectra kernel, where the number comes from) for this config,
    from the committed summary of the `ncu --set full` captures (profiles/spectra_kernel_traffic.csv); (None, why)
    if there is no row.  A number taken under a profiler is never a bench value: this is the ONE quantity of the
    line that is not measured in this run, and `traffic_source` says so."""
    import csv
    p = os.path.join(ROOT, "profiles", "spectra_kernel_traffic.csv")
    try:
        rows = [r for r in csv.DictReader(open(p)) if int(r["config"]) == config]
        r = rows[-1]
        return (int(r["dram_bytes_read"]) + int(r["dram_bytes_write"]),
                f"profiles/spectra_kernel_traffic.csv, capture {r['capture']} ({r['kernel']}; ncu --set full, one launch; "
                "not measured in this run)")
    except Exception:
        return None, "no ncu capture of this config under profiles/"


def stats_ms(ms):
    return {"mean": sum(ms) / len(ms), "median": statistics.median(ms), "min": min(ms), "max": max(ms)}


def oracle_rates(wl, data, n_all=64, n_one=4):
    """The CPU oracle as it stands, on a bounded sample of this workload: all host cores (OpenMP over points) and
    one thread.  Test infrastructure: only the cpu_baseline leg comes here."""
    import oracle
    orc = oracle.Oracle(wl.model, wl.events)
    P = wl.n_points
    n_all = min(P, n_all)
    t0 = time.perf_counter()
    nll_o = orc.nll(wl.params[:n_all], data)
    dt_all = time.perf_counter() - t0
    n_one = min(P, n_one)
    t0 = time.perf_counter()
    orc.nll(wl.params[:n_one], data, n_threads=1)
    dt_one = time.perf_counter() - t0
    return {"value": wl.n_events * n_all / dt_all, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle",
            "sample": f"all {wl.n_events} events x first {n_all} of {P} points, one call, {dt_all:.2f} s",
            "single_thread": {"value": wl.n_events * n_one / dt_one, "unit": UNIT, "cores": 1,
                              "sample": f"all {wl.n_events} events x first {n_one} of {P} points, one call, {dt_one:.2f} s"}}, nll_o


def measure(pkg, torch, dist, k, steps, warmup, local, rank, world, flush, tuning, sample_clocks, measured_peak,
            with_oracle):
    """All numbers of one config: K device-timed steps (CUDA events per step, L2 flushed in between), the same K steps
    with the library's events around each kernel, the end-to-end host-buffer call, the cached host call."""
    wl = workloads.make_config(k)
    params = wl.params.copy()
    if rank > 0:    # every rank: the same event store, its own batch of points (sharded by parameter point)
        rng = np.random.Generator(np.random.PCG64(wl.seed + 1000 * rank))
        spread = np.abs(wl.params - wl.theta0[None, :]).max(axis=0)
        params = wl.theta0[None, :] + rng.uniform(-1, 1, wl.params.shape) * spread[None, :]
    ph = pkg.Phylino(device=local)
    ph.load_workload(wl)
    if any(tuning):
        ph.set_tuning(*tuning)
    P, NPAR, TB = wl.n_points, wl.model.n_params, ph.total_bins
    ph.reserve(P)
    d_params = torch.as_tensor(params, device="cuda")
    # pseudo-data: Poisson counts around the expectation at theta0.  Where the oracle leg runs (rank 0 at N = 1, the
    # only place its NLLs are compared with the library's) the expectation is the ORACLE's, so that no input of the
    # checker comes from the checked; elsewhere it is the library's own (input synthesis only, nothing is compared).
    if with_oracle:
        import oracle
        orc0 = oracle.Oracle(wl.model, wl.events)
        th0 = wl.theta0[None, :].copy()
        mu0 = orc0.expectation(th0, orc0.spectra(th0))[0]
        data_from = "oracle expectation at theta0"
    else:
        mu0 = ph.expectation(torch.as_tensor(wl.theta0[None, :].copy(), device="cuda")).cpu().numpy()[0]
        data_from = "library expectation at theta0 (no oracle leg in this run)"
    data = workloads.poisson_counts(mu0, wl.seed + 7)
    d_data = torch.as_tensor(data, device="cuda")
    d_nll = torch.empty(P, dtype=torch.float64, device="cuda")

    def barrier():
        if world > 1:
            dist.barrier()

    # ---- device-resident timed region: K steps, CUDA events per step, L2 flushed in between.  The library's
    # own per-kernel events are OFF here (with them off the kernels of a call go out as programmatic dependent
    # launches) ----
    ph.set_timing(False)
    for _ in range(warmup):
        ph.nll(d_params, d_data, d_nll)
        flush.zero_()
    starts = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    ends = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    sampler = ClockSampler(physical_gpu_index(local)) if sample_clocks else None
    launches0 = ph.launch_count
    barrier()
    torch.cuda.synchronize()
    if sampler:
        sampler.start()
    for i in range(steps):
        starts[i].record()
        ph.nll(d_params, d_data, d_nll)
        ends[i].record()
        flush.zero_()
    torch.cuda.synchronize()
    launches = ph.launch_count - launches0
    barrier()
    step_ms = [s.elapsed_time(e) for s, e in zip(starts, ends)]
    total_ms = sum(step_ms)
    # ---- the same K steps with the library's events around each of the kernels of a call (recorded on the
    # stream the kernels run on): the per-kernel durations the roofline uses ----
    ph.set_timing(True)
    su_ms, sp_ms, fin_ms, inst_ms = [], [], [], []
    for i in range(steps):
        s0, e0 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record()
        ph.nll(d_params, d_data, d_nll)
        e0.record()
        a, b, c = ph.last_kernel_ms()       # waits for this step; per-kernel device times
        su_ms.append(a)
        sp_ms.append(b)
        fin_ms.append(c)
        inst_ms.append(s0.elapsed_time(e0))
        flush.zero_()
    torch.cuda.synchronize()
    small_frac = ph.last_small_phase()
    medium_frac = ph.last_medium_phase()
    clocks = sampler.stop() if sampler else None
    barrier()
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    ms_per_step = total_ms / steps
    evpt_step = wl.n_events * P
    value = world * evpt_step / (ms_per_step * 1e-3)

    # ---- end to end through the host-buffer entry point: params + data in, kernels, nll out, every step ----
    ph.set_timing(False)
    h_params = params.copy()
    out = np.empty(P)
    for _ in range(warmup):
        ph.nll_host(h_params, data, out)
    barrier()
    torch.cuda.synchronize()
    e2e_ms = []
    for i in range(steps):
        h_params[:, 0] = params[:, 0] * (1.0 + 1e-9 * i)     # a fresh batch every step
        flush.zero_()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ph.nll_host(h_params, data, out)
        e2e_ms.append((time.perf_counter() - t0) * 1e3)
    e2e_s = sum(e2e_ms) * 1e-3
    if world > 1:
        t = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    e2e_value = world * evpt_step * steps / e2e_s

    # ---- cross-point caching, reported beside the dense numbers, never instead of
    # them: the same host-buffer call with phylino_set_caching(1); wall time of one whole batch (config 3: one
    # central-difference gradient step; config 5: one grid scan), every step a fresh batch.
    cached = None
    ph.set_caching(True)
    ph.nll_host(h_params, data, out)
    vp, classes = ph.last_plan()
    if vp > 0:
        for _ in range(warmup):
            ph.nll_host(h_params, data, out)
        torch.cuda.synchronize()
        c_ms = []
        for i in range(steps):
            h_params[:, 0] = params[:, 0] * (1.0 + 1e-9 * (i + 1))
            flush.zero_()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            ph.nll_host(h_params, data, out)
            c_ms.append((time.perf_counter() - t0) * 1e3)
        dense_ref = np.empty(P)
        ph.set_caching(False)
        ph.nll_host(h_params, data, dense_ref)
        cached = {"ms_per_step": stats_ms(c_ms), "virtual_points": vp, "energy_scale_classes": classes,
                  "points": P, "max_abs_nll_diff_vs_dense": float(np.nanmax(np.abs(out - dense_ref))),
                  "note": "phylino_nll_host with phylino_set_caching(1): H2D + plan + kernels + D2H, host wall time; "
                          "not comparable with the dense roofline (fewer event x point evaluations are executed)"}
    ph.set_caching(False)

    res = None
    if rank == 0:
        inst_general = fp64_inst_per_evpt(wl.model)
        small = P <= 16 and not (n_terms(wl.model) == 3 and P > 4)      # the small-batch kernel (setup fused in) ran
        if small:
            # the single-launch kernel keeps the unfolded forms: 11 per general term, 7 for a small-phase last term
            inst_general = 11 * n_terms(wl.model)
            inst = inst_general - (11 - 7) * small_frac
        else:
            gen = fp64_per_general_term(n_terms(wl.model))
            inst = inst_general - (gen - FP64_SMALL_TERM) * small_frac - (gen - FP64_MEDIUM_TERM) * medium_frac   # executed
        sp = stats_ms(sp_ms)
        sm_max_mhz = (clocks or {}).get("sm_max_mhz") or 1965.0
        sm_count = torch.cuda.get_device_properties(local).multi_processor_count
        peak_nominal = FP64_LANES_PER_SM * sm_count * sm_max_mhz * 1e6
        achieved = inst * evpt_step / (sp["mean"] * 1e-3)
        traffic, traffic_source = traffic_from_profile(k)
        hbm_bytes = EVENT_BYTES * wl.n_events + 8 * P * NPAR + 8 * P
        roofline = {
            "bound": "alu", "kernel": "spectra_fused_kernel" if small else "spectra_kernel",
            "achieved": achieved / 1e9, "peak": peak_nominal / 1e9, "unit": "fp64 Ginst/s",
            "frac": achieved / peak_nominal, "frac_of": "nominal fp64 pipe",
            "peak_source": f"nominal: {FP64_LANES_PER_SM} fp64 lanes/clk/SM x {sm_count} SMs x {sm_max_mhz:.0f} MHz "
                           "(derived in DESIGN.md section 7; MEASURED_PEAKS.json and the profiling guide hold no fp64 figure)",
            "measured_dfma_peak": None if measured_peak is None else measured_peak / 1e9,
            "frac_of_measured_dfma_peak": None if not measured_peak else achieved / measured_peak,
            "traffic": traffic, "traffic_source": traffic_source,
            "fp64_inst_per_event_point": inst, "fp64_inst_general_form": inst_general,
            "small_phase_fraction": small_frac, "medium_phase_fraction": medium_frac, "kernel_ms": sp["mean"], "kernel_ms_median": sp["median"],
            "kernel_ms_min": sp["min"],
            "kernel_share_of_step": sp["mean"] / (sum(inst_ms) / steps),
            "kernel_timing": f"second pass of {steps} steps with CUDA events around each kernel on the library's "
                             f"stream ({sum(inst_ms) / steps:.4f} ms per instrumented step)",
            "setup_kernel_ms": sum(su_ms) / steps, "finalize_kernel_ms": sum(fin_ms) / steps,
            "hbm_bytes_per_launch": hbm_bytes,
            "hbm_frac_if_bandwidth_bound": None,
        }
        if small:
            # one point over the store is bound by the event bytes (and, at 1e5 events, by launch latency): the same
            # kernel time against the HBM roofline of MEASURED_PEAKS.json
            hbm_gbs = measured_hbm_gbs()
            roofline["hbm_frac_if_bandwidth_bound"] = hbm_bytes / (sp["mean"] * 1e-3) / (hbm_gbs * 1e9)
            roofline["hbm_peak_gbs"] = hbm_gbs
        st = stats_ms(step_ms)
        res = {
            "config": k, "workload": f"{wl.name} (BASELINE.json configs[{k - 1}])", "events": wl.n_events,
            "points_per_gpu": P, "n_params": NPAR, "total_bins": TB, "steps": steps, "warmup": warmup,
            "value": value, "unit": UNIT, "ms_per_step": ms_per_step, "ms_per_step_median": st["median"],
            "ms_per_step_min": st["min"], "gpu_launches": launches,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 8 * (P * NPAR + TB),
                    "d2h_bytes_per_step": 8 * P, "ms_per_step": e2e_s / steps * 1e3,
                    "ms_per_step_median": statistics.median(e2e_ms), "ms_per_step_min": min(e2e_ms),
                    "call": "phylino_nll_host: pinned staging, parameters + data to the device, kernels, nll[P] back, "
                            "one synchronise; host wall clock, L2 flushed before every call"},
            "roofline": roofline, "clocks": clocks,
        }
        if cached is not None:
            res["cached"] = cached
        if evpt_step <= 10_000_000:
            # launch-latency-bound workload (config 1): one host call against the empty-kernel floor, cold (L2
            # flushed before the call: the e2e numbers above) and warm (back to back, as a minimiser calls it)
            warm = []
            for i in range(max(steps, 50)):
                t0 = time.perf_counter()
                ph.nll_host(h_params, data, out)
                warm.append((time.perf_counter() - t0) * 1e6)
            res["latency"] = {"host_call_us_cold_median": statistics.median(e2e_ms) * 1e3, "host_call_us_cold_min": min(e2e_ms) * 1e3,
                              "host_call_us_warm_median": statistics.median(warm), "host_call_us_warm_min": min(warm),
                              "device_step_us_median": st["median"] * 1e3, "device_step_us_min": st["min"] * 1e3,
                              "launch_plus_sync_floor_us": ph.launch_floor(200),
                              "note": "a call is 2 launches (spectra with the setup fused in; finalize, overlapped) "
                                      "+ 1 synchronise; no copy engine (parameters ride with the kernel arguments)"}
        if with_oracle:
            res["cpu_baseline"], nll_o = oracle_rates(wl, data)
            res["cpu_baseline"]["pseudo_data_from"] = data_from
            res["cpu_baseline"]["max_abs_nll_diff_vs_gpu"] = float(np.abs(nll_o - d_nll.cpu().numpy()[:len(nll_o)]).max())
    ph.close()
    return res


def sharded_steps(evaluate, params, n_events, steps, warmup, dist, before_step, timer, check_against=None, tol=1e-9):
    """The STRONG arm of a multi-rank run: ONE batch of points is cut across the ranks
    with sharding.shard_points, every rank evaluates its slice, and nll[P] is all-gathered INSIDE the timed region
    (sharding.sharded_eval).  The step time is the maximum over ranks; value = n_events x P / that time.
    Device-agnostic so that the CPU test can drive it with gloo: `evaluate(slice) -> one row per point`,
    `before_step()` = flush + synchronise + barrier, `timer` = object with start() / stop() -> milliseconds on the
    device the evaluator runs on.  check_against: the unsharded result on this rank (rank 0), compared to `tol`
    (a slice is a batch of another size, so the rows agree to rounding, not bit for bit)."""
    import torch
    from paper_2502_15253_b200 import sharding
    world = dist.get_world_size() if dist.is_initialized() else 1
    rank = dist.get_rank() if dist.is_initialized() else 0
    P = int(params.shape[0])
    ms, out = [], None
    for it in range(warmup + steps):
        before_step()
        timer.start()
        out = sharding.sharded_eval(evaluate, params)
        t = torch.tensor([timer.stop()], dtype=torch.float64, device=params.device)
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        if it >= warmup:
            ms.append(float(t.item()))
    if tuple(out.shape[:1]) != (P,):
        raise RuntimeError("the gathered result does not have one row per point")
    res = {"points": P, "slices": sharding.shard_sizes(P, world), "steps": steps, "warmup": warmup,
           "ms_per_step": sum(ms) / len(ms), "ms_per_step_min": min(ms),
           "value": n_events * P / (sum(ms) / len(ms) * 1e-3), "unit": UNIT, "scaling": "strong",
           "collective": "all_gather of nll[P] inside the timed region (padded to the largest slice)"}
    if check_against is not None and rank == 0:
        err = float((out - check_against).abs().max()) if P else 0.0
        res["max_abs_nll_diff_vs_one_gpu"] = err
        if not err <= tol:
            raise RuntimeError(f"sharded NLLs differ from the one-GPU batch by {err} > {tol}")
    return res


class CudaEventTimer:
    """milliseconds between start() and stop() on torch's current CUDA stream (the library's stream in bench.py)"""
    def __init__(self, torch):
        self.torch = torch
        self.a, self.b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def start(self):
        self.a.record()

    def stop(self):
        self.b.record()
        self.b.synchronize()
        return self.a.elapsed_time(self.b)


def sharded_arm(pkg, torch, dist, k, steps, warmup, local, rank, world, flush):
    """config k's whole batch sharded over the ranks (603 points over 8 ranks: 76 / 75, the uneven case)"""
    wl = workloads.make_config(k)
    ph = pkg.Phylino(device=local)
    ph.load_workload(wl)
    ph.reserve(wl.n_points if rank == 0 else max(1, -(-wl.n_points // world)))
    d_params = torch.as_tensor(wl.params, device="cuda")
    mu0 = ph.expectation(torch.as_tensor(wl.theta0[None, :].copy(), device="cuda")).cpu().numpy()[0]
    d_data = torch.as_tensor(workloads.poisson_counts(mu0, wl.seed + 7), device="cuda")
    whole = ph.nll(d_params, d_data).clone() if rank == 0 else None     # the one-GPU call, for the check only

    def before_step():
        flush.fill_(1)
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()

    def evaluate(p):
        if p.shape[0] == 0:
            return torch.empty(0, dtype=torch.float64, device="cuda")
        return ph.nll(p, d_data)

    res = sharded_steps(evaluate, d_params, wl.n_events, steps, warmup, dist, before_step, CudaEventTimer(torch), whole)
    res["workload"] = f"{wl.name} (BASELINE.json configs[{k - 1}])"
    ph.close()
    return res


def measured_hbm_gbs() -> float:
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"])
    except Exception:
        return 6553.6       # the profiling guide's fallback for this pool's B200s


def gradient_step_wall(pkg, torch, local, flush, steps=10):
    """north_star: "wall time for a full gradient step" -- BASELINE.json configs[2] (3 x 2e6 events, 301
    parameters, 603 central-difference points) through the host call a minimiser makes (H2D + kernels + D2H),
    dense and with cross-point caching; a fresh batch every step, L2 flushed in between."""
    wl = workloads.make_config(3)
    ph = pkg.Phylino(device=local)
    ph.load_workload(wl)
    mu0 = ph.expectation(torch.as_tensor(wl.theta0[None, :].copy(), device="cuda")).cpu().numpy()[0]
    data = workloads.poisson_counts(mu0, wl.seed + 7)
    out = np.empty(wl.n_points)
    res = {"workload": f"{wl.name} (BASELINE.json configs[2])", "events": wl.n_events, "points": wl.n_points,
           "n_params": wl.model.n_params, "steps": steps}
    for key, on in (("dense_ms", False), ("cached_ms", True)):
        ph.set_caching(on)
        h = wl.params.copy()
        for _ in range(3):
            ph.nll_host(h, data, out)
        torch.cuda.synchronize()
        ts = []
        for i in range(steps):
            h[:, 0] = wl.params[:, 0] * (1.0 + 1e-9 * (i + 1))
            flush.zero_()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            ph.nll_host(h, data, out)
            ts.append((time.perf_counter() - t0) * 1e3)
        res[key] = sum(ts) / steps
        res[key + "_median"] = statistics.median(ts)
        res[key + "_min"] = min(ts)
        if on:
            res["virtual_points"], res["energy_scale_classes"] = ph.last_plan()
    # the same step with the batch formed and differenced ON THE DEVICE (phylino_nll_gradient: theta and steps in,
    # gradient out; with caching the plan comes from the batch's structure, so nothing is copied back and nothing
    # synchronises): device time between CUDA events
    N = wl.model.n_params
    theta0 = wl.params[0].copy()
    d_theta = torch.as_tensor(theta0, device="cuda")
    d_step = torch.as_tensor(np.array([wl.params[1 + 2 * j, j] - theta0[j] for j in range(N)]), device="cuda")
    d_data0 = torch.as_tensor(data, device="cuda")
    g0 = torch.empty(1, dtype=torch.float64, device="cuda")
    gg = torch.empty(N, dtype=torch.float64, device="cuda")
    for key, on in (("device_gradient_dense_ms", False), ("device_gradient_cached_ms", True)):
        ph.set_caching(on)
        for _ in range(3):
            ph.nll_gradient(d_theta, d_step, d_data0, g0, gg)
        ts = []
        for i in range(steps):
            flush.zero_()
            s0, e0 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            s0.record()
            ph.nll_gradient(d_theta, d_step, d_data0, g0, gg)
            e0.record()
            torch.cuda.synchronize()
            ts.append(s0.elapsed_time(e0))
        res[key] = sum(ts) / steps
        res[key + "_median"] = statistics.median(ts)
        res[key + "_min"] = min(ts)
    ph.set_caching(False)
    # a minimiser's SINGLE evaluation on the same store (one point over 6e6 events): bound by the event bytes over
    # HBM, not by arithmetic -- the small-batch kernel (setup fused in) + the overlapped finalize kernel
    d_data = torch.as_tensor(data, device="cuda")
    single = {}
    for n_pts in (1, 4, 16):
        dp = torch.as_tensor(wl.params[:n_pts].copy(), device="cuda")
        d_out = torch.empty(n_pts, dtype=torch.float64, device="cuda")
        for _ in range(3):
            ph.nll(dp, d_data, d_out)
        ts = []
        for i in range(max(steps, 20)):
            flush.zero_()
            s0, e0 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            s0.record()
            ph.nll(dp, d_data, d_out)
            e0.record()
            torch.cuda.synchronize()
            ts.append(s0.elapsed_time(e0) * 1e3)
        hs = []
        hp, ho = wl.params[:n_pts].copy(), np.empty(n_pts)
        for i in range(max(steps, 20)):
            flush.zero_()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            ph.nll_host(hp, data, ho)
            hs.append((time.perf_counter() - t0) * 1e6)
        # L2-WARM: what a line search sees -- the 72 MB store fits the 126 MB L2 and nothing else runs in between
        # (SURVEY.md 8(d) "may even sit in L2"): back-to-back calls, no flush
        tw, hw = [], []
        for i in range(max(steps, 20)):
            s0, e0 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            s0.record()
            ph.nll(dp, d_data, d_out)
            e0.record()
            torch.cuda.synchronize()
            tw.append(s0.elapsed_time(e0) * 1e3)
        for i in range(max(steps, 20)):
            t0 = time.perf_counter()
            ph.nll_host(hp, data, ho)
            hw.append((time.perf_counter() - t0) * 1e6)
        single[str(n_pts)] = {"device_step_us_median": statistics.median(ts), "device_step_us_min": min(ts),
                              "host_call_us_median": statistics.median(hs), "host_call_us_min": min(hs),
                              "warm": {"device_step_us_median": statistics.median(tw), "device_step_us_min": min(tw),
                                       "host_call_us_median": statistics.median(hw), "host_call_us_min": min(hw),
                                       "l2": "not flushed: back-to-back calls over a store that fits L2"}}
    store_bytes = EVENT_BYTES * wl.n_events
    floor_us = ph.hbm_read_floor(store_bytes, 10)
    hbm = measured_hbm_gbs()
    res["single_evaluation"] = {
        "points": single, "event_store_bytes": store_bytes, "l2": "flushed before every call",
        "hbm_time_at_measured_peak_us": store_bytes / (hbm * 1e9) * 1e6, "hbm_peak_gbs": hbm,
        "hbm_read_floor_us": floor_us,
        "hbm_read_floor_note": "device time of one kernel that only reads the store's bytes from HBM (L2 flushed), "
                               "launch ramp included (phylino_hbm_read_floor)",
        "frac_of_hbm_roofline_1pt": store_bytes / (hbm * 1e9) * 1e6 / single["1"]["device_step_us_median"],
        "frac_of_read_floor_1pt": floor_us / single["1"]["device_step_us_median"]}
    ph.close()
    return res


def run_reference(args, wl, rank):
    """--impl reference: the CPU oracle, as it stands, on the host cores (bounded sample per step)."""
    if rank != 0:
        return
    import oracle
    orc = oracle.Oracle(wl.model, wl.events)
    n_pts = min(wl.n_points, args.ref_points)
    params = wl.params[:n_pts]
    data = np.full(orc.total_bins, 100.0)
    cores = oracle.max_threads()
    for _ in range(args.warmup):
        orc.nll(params, data)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        orc.nll(params, data)
    dt = time.perf_counter() - t0
    evpt = wl.n_events * n_pts
    value = evpt * args.steps / dt
    sample = f"all {wl.n_events} events x first {n_pts} of {wl.n_points} points per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": f"{wl.name} (BASELINE.json configs[{args.config - 1}])",
                                        "events": wl.n_events, "points": n_pts},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=0,
                    help="BASELINE.json config, 1-based, as the headline and only workload (default: config 5 as the "
                         "headline plus all five in `configs`)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--other-steps", type=int, default=20, help="steps per config of the `configs` array")
    ap.add_argument("--unit-events", type=int, default=0, help="tuning: events per unit of the event store")
    ap.add_argument("--chunk-groups", type=int, default=0, help="tuning: groups of 32 points per work item")
    ap.add_argument("--max-warps", type=int, default=0, help="tuning: cap on the persistent grid's warps")
    ap.add_argument("--ref-points", type=int, default=16, help="points per step of --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sharded-arm", action="store_true", help="N > 1: skip the strong (sharded batch) arm")
    ap.add_argument("--sharded-arm", action="store_true", help="run the strong arm also at N = 1 (one slice, no collective)")
    ap.add_argument("--no-gradient-step", action="store_true",
                    help="skip the wall time of config 3's 603-point gradient step that the default run adds")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    all_configs = args.config == 0
    if all_configs:
        args.config = HEADLINE_CONFIG

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        run_reference(args, workloads.make_config(args.config), rank)
        return

    import torch
    import torch.distributed as dist
    import paper_2502_15253_b200 as pkg

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (this path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device="cuda")
    tuning = (args.unit_events, args.chunk_groups, args.max_warps)

    measured_peak = None
    if rank == 0:
        try:
            with pkg.Phylino(device=local) as ph0:
                measured_peak = ph0.peak_fp64(8192)
        except Exception:
            measured_peak = None

    with_oracle = world == 1 and not args.no_cpu_baseline
    head = measure(pkg, torch, dist, args.config, args.steps, args.warmup, local, rank, world, flush, tuning, True,
                   measured_peak, with_oracle)
    others = []
    if all_configs and world == 1:
        for k in (1, 2, 3, 4):
            others.append(measure(pkg, torch, dist, k, args.other_steps, args.warmup, local, rank, world, flush, tuning,
                                  False, measured_peak, with_oracle))

    # N > 1: besides the weak arm above (every rank its own batch), the STRONG arm -- the configured batch cut across
    # the ranks and gathered inside the timed region: config 5's 4096 points and config 3's 603 (uneven slices)
    sharded = []
    if (world > 1 and not args.no_sharded_arm) or args.sharded_arm:
        for k in (HEADLINE_CONFIG, 3):
            sharded.append(sharded_arm(pkg, torch, dist, k, min(args.steps, args.other_steps), args.warmup, local, rank,
                                       world, flush))
    if rank == 0:
        line = {
            "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": head["ms_per_step"], "ms_per_step_median": head["ms_per_step_median"],
            "ms_per_step_min": head["ms_per_step_min"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": head["workload"] + (": the largest single-GPU config (BASELINE.json's metric names none)"
                                                       if all_configs else ""),
                       "events": head["events"], "points_per_gpu": head["points_per_gpu"], "n_params": head["n_params"],
                       "total_bins": head["total_bins"],
                       "l2": f"flushed between timed iterations ({L2_FLUSH_BYTES >> 20} MiB write)",
                       "sharding": "by parameter point, event store replicated, no collective"},
            "clocks": head["clocks"], "gpu_launches": head["gpu_launches"],
            "e2e": head["e2e"], "roofline": head["roofline"],
        }
        for key in ("cached", "latency", "cpu_baseline"):
            if key in head:
                line[key] = head[key]
        if others:
            line["configs"] = sorted(others + [head], key=lambda r: r["config"])
        if world == 1 and all_configs and not args.no_gradient_step:
            line["gradient_step"] = gradient_step_wall(pkg, torch, local, flush)
        if sharded:
            line["sharded"] = sharded
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
