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
