#!/usr/bin/env python
"""bench.py -- throughput of the batched spectra + NLL hot path (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config k] [--impl ours|reference]

A step = one phylino_nll call over the whole batch of parameter points of the workload (all rows of
SURVEY.md 8(a): per-point derivation, oscillation weights, energy scale + binning, scatter-add,
deterministic reduction, expectation assembly, NLL reduction).  Default workload: BASELINE.json
configs[1] (Double Chooz FD+ND, 2 x 1e6 events, 64 points).  Prints ONE JSON line (rank 0).

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
# ALGORITHMIC fp64-pipe instructions per event x point: per oscillation term
# 10 for 1/2 cos(2 phase) (3 range reduction, 1 square, 6 Horner) + 1 multiply-accumulate into the run;
# the SASS of the hot loop has exactly these (9 DFMA + 1 DADD + 1 DMUL per event x point x term).
# The bin/weight bookkeeping is per batch of events and per run, not per event x point.
FP64_PER_TERM = 11
# nominal fp64 pipe: 64 lanes/clk/SM x 148 SMs x 1.965 GHz (B200_PROFILING.md table)
PEAK_FP64_INST = 64 * 148 * 1.965e9
L2_FLUSH_BYTES = 256 << 20


def fp64_inst_per_evpt(model) -> int:
    S = 2 if model.osc_model == 0 else 3
    return FP64_PER_TERM * S


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
    """dram bytes (read + write) per launch of the spectra kernel for this config, from the committed
    summary of the ncu --set full capture (profiles/spectra_kernel_traffic.csv), or None."""
    import csv
    p = os.path.join(ROOT, "profiles", "spectra_kernel_traffic.csv")
    try:
        rows = [r for r in csv.DictReader(open(p)) if int(r["config"]) == config]
        return int(rows[-1]["dram_bytes_read"]) + int(rows[-1]["dram_bytes_write"])
    except Exception:
        return None


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
        t = 0.0
        for i in range(steps):
            h[:, 0] = wl.params[:, 0] * (1.0 + 1e-9 * (i + 1))
            flush.zero_()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            ph.nll_host(h, data, out)
            t += time.perf_counter() - t0
        res[key] = t / steps * 1e3
        if on:
            res["virtual_points"], res["energy_scale_classes"] = ph.last_plan()
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
        "data": "synthetic", "config": {"workload": wl.name, "events": wl.n_events, "points": n_pts},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config, 1-based (default 2 = configs[1])")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--unit-events", type=int, default=0, help="tuning: events per unit of the event store")
    ap.add_argument("--chunk-groups", type=int, default=0, help="tuning: groups of 32 points per work item")
    ap.add_argument("--max-warps", type=int, default=0, help="tuning: cap on the persistent grid's warps")
    ap.add_argument("--ref-points", type=int, default=16, help="points per step of --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-gradient-step", action="store_true",
                    help="skip the wall time of config 3's 603-point gradient step that the default run adds")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    wl = workloads.make_config(args.config)

    if args.impl == "reference":
        run_reference(args, wl, rank)
        return

    import torch
    import torch.distributed as dist
    import paper_2502_15253_b200 as pkg

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (this path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    # every rank: the same event store, its own batch of points (sharded by parameter point)
    params = wl.params.copy()
    if rank > 0:
        rng = np.random.Generator(np.random.PCG64(wl.seed + 1000 * rank))
        spread = np.abs(wl.params - wl.theta0[None, :]).max(axis=0)
        params = wl.theta0[None, :] + rng.uniform(-1, 1, wl.params.shape) * spread[None, :]
    ph = pkg.Phylino(device=local)
    ph.load_workload(wl)
    if args.unit_events or args.chunk_groups or args.max_warps:
        ph.set_tuning(args.unit_events, args.chunk_groups, args.max_warps)
    P, NPAR, TB = wl.n_points, wl.model.n_params, ph.total_bins
    d_params = torch.as_tensor(params, device="cuda")
    # pseudo-data: Poisson counts around the product's own expectation at theta0 (input synthesis only)
    mu0 = ph.expectation(torch.as_tensor(wl.theta0[None, :].copy(), device="cuda")).cpu().numpy()[0]
    data = workloads.poisson_counts(mu0, wl.seed + 7)
    d_data = torch.as_tensor(data, device="cuda")
    d_nll = torch.empty(P, dtype=torch.float64, device="cuda")
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device="cuda")

    def barrier():
        if world > 1:
            dist.barrier()

    for _ in range(args.warmup):
        ph.nll(d_params, d_data, d_nll)
        flush.zero_()
    torch.cuda.synchronize()

    # ---- device-resident timed region: K steps, CUDA events per step, L2 flushed in between.  The library's
    # own per-kernel events are OFF here (they sit between the three launches and cost ~10 us per step; with
    # them off the spectra and finalize kernels go out as programmatic dependent launches) ----
    starts = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    ends = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    sampler = ClockSampler(physical_gpu_index(local))
    ph.set_timing(False)
    for _ in range(2):
        ph.nll(d_params, d_data, d_nll)
        flush.zero_()
    launches0 = ph.launch_count
    barrier()
    torch.cuda.synchronize()
    sampler.start()
    for i in range(args.steps):
        starts[i].record()
        ph.nll(d_params, d_data, d_nll)
        ends[i].record()
        flush.zero_()
    torch.cuda.synchronize()
    launches = ph.launch_count - launches0
    barrier()
    total_ms = sum(s.elapsed_time(e) for s, e in zip(starts, ends))
    # ---- same K steps again with the library's events around each of the three kernels (recorded on the
    # stream the kernels run on): the per-kernel durations the roofline uses ----
    ph.set_timing(True)
    su_ms, sp_ms, fin_ms = [], [], []
    inst_ms = 0.0
    for i in range(args.steps):
        s0, e0 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record()
        ph.nll(d_params, d_data, d_nll)
        e0.record()
        a, b, c = ph.last_kernel_ms()       # waits for this step; per-kernel device times
        su_ms.append(a)
        sp_ms.append(b)
        fin_ms.append(c)
        inst_ms += s0.elapsed_time(e0)
        flush.zero_()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    barrier()
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    ms_per_step = total_ms / args.steps
    evpt_step = wl.n_events * P
    value = world * evpt_step / (ms_per_step * 1e-3)

    # ---- end to end through the host-buffer entry point: H2D params+data, kernels, D2H nll ----
    ph.set_timing(False)
    h_params = params.copy()
    out = np.empty(P)
    for _ in range(args.warmup):
        ph.nll_host(h_params, data, out)
    barrier()
    torch.cuda.synchronize()
    e2e_s = 0.0
    for i in range(args.steps):
        h_params[:, 0] = params[:, 0] * (1.0 + 1e-9 * i)     # a fresh batch every step
        t0 = time.perf_counter()
        ph.nll_host(h_params, data, out)
        e2e_s += time.perf_counter() - t0
        flush.zero_()
        torch.cuda.synchronize()
    if world > 1:
        t = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    e2e_value = world * evpt_step * args.steps / e2e_s

    # ---- cross-point caching, reported beside the dense numbers, never instead of
    # them: the same host-buffer call with phylino_set_caching(1); wall time of one whole batch (config 3: one
    # central-difference gradient step; config 5: one grid scan), every step a fresh batch.
    cached = None
    ph.set_caching(True)
    ph.nll_host(h_params, data, out)
    vp, classes = ph.last_plan()
    if vp > 0:
        for _ in range(args.warmup):
            ph.nll_host(h_params, data, out)
        torch.cuda.synchronize()
        c_s = 0.0
        for i in range(args.steps):
            h_params[:, 0] = params[:, 0] * (1.0 + 1e-9 * (i + 1))
            t0 = time.perf_counter()
            ph.nll_host(h_params, data, out)
            c_s += time.perf_counter() - t0
            flush.zero_()
            torch.cuda.synchronize()
        dense_ref = np.empty(P)
        ph.set_caching(False)
        ph.nll_host(h_params, data, dense_ref)
        cached = {"ms_per_step": c_s / args.steps * 1e3, "virtual_points": vp, "energy_scale_classes": classes,
                  "points": P, "max_abs_nll_diff_vs_dense": float(np.nanmax(np.abs(out - dense_ref))),
                  "note": "phylino_nll_host with phylino_set_caching(1): H2D + plan + kernels + D2H; "
                          "not comparable with the dense roofline (fewer event x point evaluations are executed)"}
    ph.set_caching(False)

    if rank == 0:
        inst = fp64_inst_per_evpt(wl.model)
        sp_avg = sum(sp_ms) / len(sp_ms)
        achieved = inst * evpt_step / (sp_avg * 1e-3)
        try:
            measured_peak = ph.peak_fp64(8192)
        except Exception:
            measured_peak = None
        roofline = {
            "bound": "alu", "kernel": "spectra_kernel", "achieved": achieved / 1e9, "peak": PEAK_FP64_INST / 1e9,
            "unit": "fp64 Ginst/s", "frac": achieved / PEAK_FP64_INST, "traffic": traffic_from_profile(args.config),
            "peak_source": "nominal: 64 fp64 lanes/clk/SM x 148 SMs x 1.965 GHz (DESIGN.md)",
            "measured_dfma_peak": None if measured_peak is None else measured_peak / 1e9,
            "frac_of_measured": None if not measured_peak else achieved / measured_peak,
            "fp64_inst_per_event_point": inst, "kernel_ms": sp_avg,
            "kernel_share_of_step": sp_avg / (inst_ms / args.steps),
            "kernel_timing": f"second pass of {args.steps} steps with CUDA events around each kernel on the library's "
                             f"stream ({inst_ms / args.steps:.4f} ms per instrumented step)",
            "setup_kernel_ms": sum(su_ms) / len(su_ms), "finalize_kernel_ms": sum(fin_ms) / len(fin_ms),
            "hbm_bytes_per_launch": 24 * wl.n_events + 8 * P * TB,
        }
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{wl.name} (BASELINE.json configs[{args.config - 1}])",
                       "events": wl.n_events, "points_per_gpu": P, "n_params": NPAR, "total_bins": TB,
                       "l2": f"flushed between timed iterations ({L2_FLUSH_BYTES >> 20} MiB write)",
                       "sharding": "by parameter point, event store replicated, no collective"},
            "clocks": clocks, "gpu_launches": launches,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 8 * (P * NPAR + TB),
                    "d2h_bytes_per_step": 8 * P, "ms_per_step": e2e_s / args.steps * 1e3},
            "roofline": roofline,
        }
        if cached is not None:
            line["cached"] = cached
        if wl.n_events * P <= 10_000_000:
            # launch-latency-bound workload (config 1): one host call against the empty-kernel floor
            line["latency"] = {"host_call_us": e2e_s / args.steps * 1e6, "device_step_us": ms_per_step * 1e3,
                               "launch_plus_sync_floor_us": ph.launch_floor(200),
                               "note": "a call is 1 H2D + 3 kernels + 1 D2H + 1 synchronise"}
        if world == 1 and args.config == 2 and not args.no_gradient_step:
            line["gradient_step"] = gradient_step_wall(pkg, torch, local, flush)
        if world == 1 and not args.no_cpu_baseline:
            import oracle                                   # the cpu_baseline leg (test infrastructure)
            orc = oracle.Oracle(wl.model, wl.events)
            n_pts = min(P, 64)
            t0 = time.perf_counter()
            nll_o = orc.nll(wl.params[:n_pts], data)
            dt = time.perf_counter() - t0
            line["cpu_baseline"] = {
                "value": wl.n_events * n_pts / dt, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle",
                "sample": f"all {wl.n_events} events x first {n_pts} of {P} points, one call, {dt:.2f} s",
                "max_abs_nll_diff_vs_gpu": float(np.abs(nll_o - d_nll.cpu().numpy()[:n_pts]).max())}
        print(json.dumps(line))
    ph.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
