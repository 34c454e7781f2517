"""bench.py's JSON line on a GPU box: the keys the measurement contract asks for, on the small workload."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_bench(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], cwd=ROOT, capture_output=True,
                         text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout[-2000:]
    return json.loads(lines[0])


@pytest.mark.gpu
def test_bench_line_has_the_contract_keys():
    d = run_bench("--workload", "1", "--steps", "5", "--warmup", "3", "--e2e-steps", "2", "--cpu-seconds", "1",
                  "--shock-frac", "0.5", "--compact-frac", "0.25")
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline",
              "parity_checked", "repeats"):
        assert k in d, k
    assert d["n_gpus"] == 1 and d["steps"] == 5 and d["warmup"] == 3 and d["dtype"] == "f64"
    assert d["vs_baseline"] is None and d["scaling"] == "weak" and d["data"] == "synthetic"
    assert d["value"] > 0 and d["gpu_launches"] >= 5 and "workload" in d["config"]
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and r["peak"] > 1000 and r["achieved"] > 0
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and "traffic" in r
    a = r["alu"]
    assert a["bound"] == "alu" and a["peak"] > 1.0 and a["achieved"] > 0 and abs(a["frac"] - a["achieved"] / a["peak"]) < 1e-12
    pc = d["parity_checked"]
    assert pc["ok"] and pc["positions_bit_exact"] and pc["max_rel"] <= 1e-10 and pc["steps"] == 3 + 5 * 5 and pc["particles"] == 1024
    rp = d["repeats"]
    assert rp["passes"] == 5 and len(rp["ms_per_step"]) == 5 and len(rp["clocks"]) == 5
    # the line quotes the median pass, not the best one
    assert d["ms_per_step"] == rp["ms_per_step"][rp["quoted_pass"]] == sorted(rp["ms_per_step"])[2]
    assert d["value"] == rp["value"][rp["quoted_pass"]] and d["clocks"] == rp["clocks"][rp["quoted_pass"]]
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["sample"]
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}
    assert d["shock_update"]["flagged"] > 0 and d["compact"]["np_new"] == 1024 - d["compact"]["deleted"]
    c1, cs = c["single_thread"], c["spectral_update_only"]
    assert c1["cores"] == 1 and c1["value"] > 0 and cs["value"] > 0


@pytest.mark.gpu
def test_bench_workload2_staged_with_time_dependent_fields():
    """configs[1]: the staged calls with the fields re-set between the stages, parity-checked in the line."""
    d = run_bench("--workload", "2", "--steps", "4", "--warmup", "3", "--repeats", "2", "--no-e2e", "--cpu-seconds", "1")
    assert "lp_set_fields" in d["config"]["api"] and d["parity_checked"]["ok"] and d["parity_checked"]["steps"] == 3 + 4 * 2


@pytest.mark.gpu
def test_reference_arm_line():
    d = run_bench("--impl", "reference", "--workload", "1", "--steps", "2", "--warmup", "1")
    assert d["impl"] == "reference" and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0 and d["gpu_launches"] == 0


@pytest.mark.gpu
def test_sweep_points_of_the_small_configs():
    """The `sweep` key of the default run is made of sweep_point entries; the two small configs through the same code
    (configs[0] fused, configs[1] staged with time-dependent fields), each parity-checked on its timed state."""
    import torch
    sys.path.insert(0, ROOT)
    import bench
    import paper_2602_23434_b200 as P
    cache = {}
    for index, steps in ((1, 100), (2, 200)):
        e = bench.sweep_point(P, index, 0, torch.device("cuda", 0), 0, 6500.0, 30.0, cache, nsample=128)
        assert e["steps"] == steps and e["ms_per_step"] > 0 and e["frac"] > 0 and e["alu_frac"] > 0
        assert e["parity_checked"]["ok"] and e["parity_checked"]["steps"] == steps + 3
        assert set(e["clocks"]) >= {"sm_mhz", "reasons"}
