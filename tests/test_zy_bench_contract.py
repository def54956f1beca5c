"""bench.py's output contract: one JSON line with the keys the driver reads (needs one B200).  The headline leg and the
CPU baseline only; the other legs are switched off to keep the test short."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_bench_line_carries_the_contract_keys():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "1", "--steps", "5", "--warmup", "3", "--configs", "1",
           "--batch", "0", "--no-field", "--no-stage", "--no-seeding", "--no-compare"]
    r = subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.strip().splitlines() if ln.strip()]
    assert len(lines) == 1, "exactly one line on stdout"
    out = json.loads(lines[0])
    assert out["metric"] == "seed_hit_dca_evals_per_s" and out["n_gpus"] == 1 and out["steps"] == 5 and out["warmup"] == 3
    assert out["higher_is_better"] is True and out["scaling"] == "weak" and out["vs_baseline"] is None
    assert out["dtype"] == "f64" and out["data"] == "synthetic" and "configs[1]" in out["config"]["workload"]
    assert out["value"] > 1e9 and 0.1 < out["ms_per_step"] < 100.0 and out["gpu_launches"] > 0
    e2e = out["e2e"]
    assert e2e["value"] > 1e9 and 0 < e2e["h2d_bytes_per_step"] < 100_000 and e2e["d2h_bytes_per_step"] > 0
    assert e2e["value"] != out["value"]                       # measured separately, not a copy of the device figure
    rf = out["roofline"]
    assert rf["bound"] in ("alu", "hbm", "tensor") and rf["unit"] in ("TFLOP/s", "GB/s")
    assert abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-9 and 0.05 < rf["frac"] < 1.0
    assert rf["traffic"] is None or rf["traffic"]["per_step"] > 0
    assert 0.0 < rf["hbm_frac"] < 1.0
    cb = out["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] > 0 and isinstance(cb["sample"], str)
    ck = out["clocks"]
    assert ck["sm_mhz"] > 0 and ck["sm_max_mhz"] >= ck["sm_mhz"] * 0.5 and isinstance(ck["reasons"], list)
