"""The bench.py contract on a GPU box: one JSON line with the keys the driver reads, on a small run."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_bench_prints_one_contract_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--config", "C2", "--steps", "2", "--warmup", "3"],
                       capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "e2e", "gpu_launches", "roofline", "cpu_baseline", "clocks"):
        assert k in d, k
    assert d["n_gpus"] == 1 and d["steps"] == 2 and d["warmup"] >= 3 and d["higher_is_better"] is True
    assert d["dtype"] == "u8" and d["data"] == "synthetic" and d["vs_baseline"] is None and "workload" in d["config"]
    assert d["value"] > 0 and d["gpu_launches"] > 0
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0 and e["value"] < d["value"]
    rf = d["roofline"]
    assert rf["bound"] == "hbm" and rf["unit"] == "GB/s" and abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-9
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] == 1 and cb["value"] > 0 and cb["sample"]
    assert d["check"]["ok"] is True
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}
    assert d["check"]["frames_vs_oracle"] == 16  # every oracle frame of the run is compared, not a sample of them
    t = d["targets"]
    assert set(t) >= {"kernel_60pct_of_8TBs_nominal", "kernel_60pct_of_measured_copy_rate", "e2e_1000_frames_per_s"}
    assert t["kernel_60pct_of_8TBs_nominal"]["met"] == (d["frac_of_8TBs_nominal"] >= 0.6)
    assert d["c4_batches_of_8_one_stream"]["frac"] > 0 and e["frac_of_pcie"] > 0 and e["pcie_copy_only"]["frames_per_s"] > e["value"]
    # config 4 as worded (batches over 3 caller streams), the sustained figures at the top level, the oracle's phase split
    s3 = d["c4_batches_of_8_three_streams"]
    assert s3["frac"] > 0 and s3["n_streams"] == 3 and s3["same_bytes"] is True
    assert d["value_sustained"] > 0 and 0 < d["frac_sustained"] < 1
    assert t["kernel_60pct_of_8TBs_nominal_sustained"]["met"] == (t["kernel_60pct_of_8TBs_nominal_sustained"]["frac"] >= 0.6)
    ph = cb["phases_ms_per_frame"]
    assert ph["hash"] > 0 and ph["derivation"] > 0 and ph["confusion_xor"] > 0


def test_bench_kernel_leg_only_line():
    """The command profiles/ captures under ncu: kernel-only legs, exactly the requested warm-up, one small JSON line."""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--config", "C2", "--steps", "1", "--warmup", "3", "--kernel-leg-only"],
                       capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    d = json.loads([ln for ln in r.stdout.splitlines() if ln.strip()][-1])
    assert d["kernel_leg_only"] is True and d["ok"] is True and d["warmup_steps_run"] == 3 and d["us_per_frame"] > 0
    for direction in ("encrypt", "decrypt"):
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--config", "C2", "--steps", "1", "--warmup", "3", "--kernel-leg-only",
                            "--direction", direction], capture_output=True, text=True, timeout=600)
        assert r.returncode == 0, r.stderr[-2000:]
        d = json.loads([ln for ln in r.stdout.splitlines() if ln.strip()][-1])
        assert d["direction"] == direction and d["ok"] is True and d["us_per_frame"] > 0 and d["launches_per_step"] >= 2
