"""The measurement contract of bench.py on a GPU box: one JSON line with the keys the driver reads, on the small
configuration (cfg1) so that the test stays short.  The default run (cfg4) differs only in the workload."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], cwd=ROOT, capture_output=True, text=True,
                         timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout[-2000:]
    return json.loads(lines[0])


def test_bench_line_has_the_contract_keys():
    j = _run("--workload", "cfg1", "--steps", "2", "--warmup", "3")
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches", "clocks", "roofline", "cpu_baseline"):
        assert key in j, key
    assert j["n_gpus"] == 1 and j["steps"] == 2 and j["warmup"] == 3 and j["higher_is_better"] is True
    assert j["scaling"] == "weak" and j["vs_baseline"] is None and j["dtype"] == "f32" and j["data"] == "synthetic"
    assert j["config"]["workload"] == "cfg1" and j["value"] > 0 and j["ms_per_step"] > 0
    assert j["gpu_launches"] > 0
    e = j["e2e"]
    assert e["value"] > 0 and e["unit"] == j["unit"] and e["h2d_bytes_per_step"] == 64 * 64 * 5 and e["d2h_bytes_per_step"] == 64 * 64 * 4
    r = j["roofline"]
    assert r["bound"] in ("hbm", "tensor", "alu") and r["unit"] == "GB/s" and r["peak"] > 0
    assert r["frac"] == pytest.approx(r["achieved"] / r["peak"])
    assert set(("sm_mhz", "sm_max_mhz", "reasons")) <= set(j["clocks"])
    c = j["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["unit"] == j["unit"] and c["sample"]
    assert "double_precision" in j and j["double_precision"]["mae_f64"] == pytest.approx(j["double_precision"]["mae_f32"], rel=0.2)


def test_reference_arm_line():
    j = _run("--impl", "reference", "--workload", "cfg1", "--steps", "1", "--warmup", "0")
    assert j["impl"] == "reference" and j["value"] > 0 and j["cpu_baseline"]["kind"] == "oracle"
    assert j["e2e"]["h2d_bytes_per_step"] == 0 and j["e2e"]["d2h_bytes_per_step"] == 0 and j["e2e"]["value"] == j["value"]
