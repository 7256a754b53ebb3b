"""bench.py's reference arm runs on the host cores alone (no GPU): its JSON line must carry the contract keys."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_contract_line(oracle_mod):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                          "--steps", "2", "--warmup", "1"], capture_output=True, text=True, cwd=ROOT, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    j = json.loads(lines[0])
    assert j["impl"] == "reference" and j["higher_is_better"] is True and j["vs_baseline"] is None
    assert j["metric"].startswith("oscillated event x param-point/s") and j["unit"] == "event*point/s"
    assert j["n_gpus"] == 1 and j["steps"] == 2 and j["warmup"] == 1 and j["dtype"] == "f64" and j["data"] == "synthetic"
    assert j["value"] > 0 and j["ms_per_step"] > 0 and "workload" in j["config"]
    cb = j["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == j["value"] and cb["sample"]
    assert j["e2e"] == {"value": j["value"], "unit": j["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


def test_reference_arm_other_ranks_stay_silent(oracle_mod):
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                          "--steps", "1", "--warmup", "0", "--gpus", "2"], capture_output=True, text=True, cwd=ROOT,
                         env=env, timeout=600)
    assert out.returncode == 0 and out.stdout.strip() == ""


import pytest  # noqa: E402


@pytest.mark.gpu
def test_own_arm_line_has_roofline_cpu_baseline_e2e_and_all_five_configs(gpu, oracle_mod):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "3", "--warmup", "3",
                          "--other-steps", "3", "--no-gradient-step"], capture_output=True, text=True, cwd=ROOT, timeout=1500)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    j = json.loads(lines[0])
    assert "impl" not in j and j["n_gpus"] == 1 and j["steps"] == 3 and j["scaling"] == "weak" and j["dtype"] == "f64"
    # the headline is the largest single-GPU config, not the smallest batched one
    assert "configs[4]" in j["config"]["workload"] and "l2" in j["config"]
    assert j["config"]["events"] * j["config"]["points_per_gpu"] == 2_000_000 * 4096
    assert j["gpu_launches"] == 9                                   # setup, spectra, finalize per timed step
    assert j["ms_per_step_min"] <= j["ms_per_step_median"] and j["ms_per_step_min"] <= j["ms_per_step"]
    r = j["roofline"]
    assert r["bound"] == "alu" and r["unit"] and 0.3 < r["frac"] < 1.05 and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    assert r["frac_of"] == "nominal fp64 pipe" and r["frac_of_measured_dfma_peak"] >= r["frac"] * 0.9
    assert r["traffic"] is None or r["traffic"] > 12 * j["config"]["events"] * 0.9
    assert r["traffic_source"]
    cb = j["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] > 0 and cb["max_abs_nll_diff_vs_gpu"] <= 1e-6
    assert cb["single_thread"]["cores"] == 1 and 0 < cb["single_thread"]["value"] <= cb["value"] * 1.5
    e = j["e2e"]
    assert 0 < e["value"] <= j["value"] * 1.05 and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0
    assert "sm_mhz" in j["clocks"] and "reasons" in j["clocks"]
    # every BASELINE.json config measured in the same run
    cfgs = j["configs"]
    assert [c["config"] for c in cfgs] == [1, 2, 3, 4, 5]
    for c in cfgs:
        assert c["value"] > 0 and c["ms_per_step_min"] <= c["ms_per_step_median"] and c["e2e"]["value"] > 0
        assert c["roofline"]["kernel_ms"] > 0 and "frac_of_measured_dfma_peak" in c["roofline"]
        assert c["cpu_baseline"]["max_abs_nll_diff_vs_gpu"] <= 1e-6
    lat = cfgs[0]["latency"]
    assert lat["launch_plus_sync_floor_us"] > 0 and lat["host_call_us_warm_min"] <= lat["host_call_us_cold_median"] * 1.5
    assert cfgs[0]["gpu_launches"] == 6                             # small batch: spectra (setup fused in), finalize


# ---- the strong (sharded) arm of bench.py --gpus N: argument and slicing logic on CPU, world_size 2, gloo ------------
def _free_port():
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


class _WallTimer:
    def start(self):
        import time
        self.t0 = time.perf_counter()

    def stop(self):
        import time
        return (time.perf_counter() - self.t0) * 1e3


def _sharded_worker(rank, world, port, n_points, out_dir):
    import numpy as np
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        sys.path.insert(0, ROOT)
        import bench
        import oracle
        import workloads
        wl = workloads.make_tiny(seed=99, n_events=50, n_points=n_points, n_datasets=2)
        orc = oracle.Oracle(wl.model, wl.events)
        data = np.arange(orc.total_bins, dtype=np.float64) + 2.0
        params = torch.as_tensor(wl.params)
        seen, barriers = [], []

        def evaluate(p):                                   # stands in for the rank's libphylino context
            seen.append(int(p.shape[0]))
            return torch.as_tensor(orc.nll(p.numpy(), data)) if p.shape[0] else torch.empty(0, dtype=torch.float64)

        def before_step():
            barriers.append(1)
            dist.barrier()

        whole = torch.as_tensor(orc.nll(wl.params, data)) if rank == 0 else None
        res = bench.sharded_steps(evaluate, params, 50, steps=3, warmup=2, dist=dist, before_step=before_step,
                                  timer=_WallTimer(), check_against=whole)
        assert len(barriers) == 5 and seen == [res["slices"][rank]] * 5
        assert sum(res["slices"]) == n_points and max(res["slices"]) - min(res["slices"]) <= 1
        assert res["scaling"] == "strong" and res["points"] == n_points and res["steps"] == 3
        assert res["ms_per_step"] > 0 and res["ms_per_step_min"] <= res["ms_per_step"]
        assert abs(res["value"] - 50 * n_points / (res["ms_per_step"] * 1e-3)) <= 1e-6 * res["value"]
        if rank == 0:
            assert res["max_abs_nll_diff_vs_one_gpu"] == 0.0          # same evaluator on both sides: identical rows
            # a wrong gathered vector is caught
            bad = whole + 1.0
            try:
                bench.sharded_steps(evaluate, params, 50, 1, 0, dist, before_step, _WallTimer(), bad)
                raise AssertionError("the check against the one-GPU batch did not fire")
            except RuntimeError:
                pass
        else:
            bench.sharded_steps(evaluate, params, 50, 1, 0, dist, before_step, _WallTimer(), None)
        # every rank saw the same max-over-ranks step time
        t = torch.tensor([res["ms_per_step"]], dtype=torch.float64)
        both = [torch.zeros_like(t) for _ in range(world)]
        dist.all_gather(both, t)
        assert both[0].item() == both[1].item()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_points", [7, 4, 1])
def test_sharded_arm_world2_gloo(tmp_path, oracle_mod, n_points):
    """bench.py's strong arm: slices of 4 + 3 (padding), 2 + 2, 1 + 0 (an empty slice); the all-gather
    sits inside the timed region, the step time is the max over ranks, the gathered NLLs are checked on rank 0."""
    import torch.multiprocessing as mp
    mp.spawn(_sharded_worker, args=(2, _free_port(), n_points, str(tmp_path)), nprocs=2, join=True)


@pytest.mark.gpu
def test_sharded_arm_on_one_gpu(gpu):
    """the same arm through the real library at N = 1 (one slice, no collective): configs 5 and 3, checked to 1e-9"""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--config", "1", "--steps", "3", "--warmup", "3",
                          "--other-steps", "3", "--no-cpu-baseline", "--sharded-arm"], capture_output=True, text=True,
                         cwd=ROOT, timeout=900)
    assert out.returncode == 0, out.stderr[-2000:]
    j = json.loads([l for l in out.stdout.splitlines() if l.strip()][-1])
    sh = j["sharded"]
    assert [s["points"] for s in sh] == [4096, 603] and all(s["slices"] == [s["points"]] for s in sh)
    assert all(s["scaling"] == "strong" and s["value"] > 0 and s["max_abs_nll_diff_vs_one_gpu"] <= 1e-9 for s in sh)
