"""bench.py prints ONE JSON line with the keys the measurement contract names."""
import io
import json
import contextlib
import sys

import pytest


@pytest.mark.gpu
def test_bench_line_has_the_contract_keys(monkeypatch):
    import bench
    monkeypatch.setattr(sys, "argv", ["bench.py", "--workload", "synth4m", "--steps", "5", "--warmup", "3"])
    buf = io.StringIO()
    with contextlib.redirect_stdout(buf):
        bench.main()
    lines = [x for x in buf.getvalue().splitlines() if x.strip()]
    assert len(lines) == 1
    j = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "gpu_launches", "clocks"):
        assert k in j, k
    assert j["unit"] == "GB/s" and j["dtype"] == "u8" and j["data"] == "synthetic" and j["vs_baseline"] is None
    assert j["config"]["workload"] == "synth4m" and j["warmup"] >= 3 and j["value"] > 0
    r = j["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-3 and "traffic" in r
    c = j["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["sample"]
    e = j["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] == j["config"]["comp_bytes"] and e["d2h_bytes_per_step"] == j["config"]["raw_bytes"]
    assert j["gpu_launches"] >= 2 * j["steps"]


def test_reference_arm_line_on_cpu(monkeypatch):
    import bench
    monkeypatch.setattr(sys, "argv", ["bench.py", "--impl", "reference", "--workload", "synth4m", "--steps", "2", "--warmup", "1"])
    buf = io.StringIO()
    with contextlib.redirect_stdout(buf):
        bench.main()
    j = json.loads(buf.getvalue().strip().splitlines()[-1])
    assert j["impl"] == "reference" and j["metric"] == bench.METRIC and j["unit"] == "GB/s" and j["value"] > 0
    assert j["cpu_baseline"]["kind"] == "oracle" and j["e2e"]["h2d_bytes_per_step"] == 0 and j["e2e"]["d2h_bytes_per_step"] == 0
