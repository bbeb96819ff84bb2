"""The product arm of bench.py on the GPU box, at a reduced size: the JSON line carries every key of the contract, no
roofline fraction of a measured peak exceeds 1 (a fraction far above 1 means the timed kernel is not doing the work, or
the bound is not the kernel's), the end-to-end leg reproduces the device-resident result, and the library's own kernels
were launched."""
import json
import subprocess
import sys
from pathlib import Path

import pytest
import torch

ROOT = Path(__file__).resolve().parent.parent
pytestmark = pytest.mark.gpu


def test_bench_line_contract_on_a_reduced_workload():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--workload", "cfg3", "--n", str(1 << 23), "--steps", "3",
                        "--warmup", "3", "--e2e-steps", "1"], capture_output=True, text=True, timeout=900, cwd=str(ROOT))
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["metric"].startswith("particles/sec") and d["unit"] == "particles/s" and d["higher_is_better"] is True
    assert d["n_gpus"] == 1 and d["steps"] == 3 and d["warmup"] == 3 and d["scaling"] == "weak" and d["vs_baseline"] is None
    assert d["dtype"] == "int32" and d["data"] == "synthetic" and d["config"]["workload"] == "cfg3"
    assert d["value"] > 0 and abs(d["value"] - (1 << 23) / (d["ms_per_step"] * 1e-3)) < 1e-6 * d["value"]
    assert d["gpu_launches"] > 0
    rf = d["roofline"]
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic", "kernel_ms", "kernel_share_of_step", "path"):
        assert k in rf
    assert rf["bound"] == "alu" and rf["peak"] > 0
    assert rf["frac"] is None or 0 < rf["frac"] <= 1.0          # null only when the ncu capture is stale
    assert 0 < rf["kernel_share_of_step"] < 1 and 0 < rf["hbm"]["frac"] <= 1.0
    assert rf["path"]["frac"] > 0
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] == 1 and cb["value"] > 0 and cb["best_of"] == 3 and "sample" in cb
    e = d["e2e"]
    assert e["value"] > 0 and e["unit"] == "particles/s" and e["h2d_bytes_per_step"] == (1 << 23) * 12
    assert e["d2h_bytes_per_step"] > 0 and e["same_result_as_device_path"] is True
    assert e["two_crossings"]["h2d_bytes_per_step"] == 2 * (1 << 23) * 12 and e["two_crossings"]["same_result_as_device_path"] is True
    assert e["value"] < d["value"], "the end-to-end number includes the PCIe copies"
    c = d["clocks"]
    assert "sm_mhz" in c and "reasons" in c
