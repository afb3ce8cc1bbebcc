"""The bench line on the GPU: one small run of bench.py through its command line, checked against the contract keys."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_bench_line_has_the_contract_keys():
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--size", "24x16x8", "--steps", "2", "--warmup", "3"],
                       capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert k in d, k
    assert d["n_gpus"] == 1 and d["steps"] == 2 and d["warmup"] >= 3 and d["higher_is_better"] is True
    assert d["dtype"] == "f64" and d["data"] == "synthetic" and d["vs_baseline"] is None and d["scaling"] == "weak"
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["gpu_launches"] > 0 and d["config"]["finite"] is True
    assert "workload" in d["config"] and "model" not in d["config"]
    for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"):
        assert k in d["e2e"], k
    assert d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0 and 0 < d["e2e"]["value"] < d["value"]
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert k in d["roofline"], k
    assert abs(d["roofline"]["frac"] - d["roofline"]["achieved"] / d["roofline"]["peak"]) < 1e-12
    for k in ("value", "unit", "cores", "kind", "sample", "single_thread"):
        assert k in d["cpu_baseline"], k
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] > 0
    assert d["cpu_baseline"]["single_thread"]["cores"] == 1 and d["cpu_baseline"]["single_thread"]["value"] > 0
    # the whole step against SURVEY 8(d)'s two fixed byte counts; no inflatable numerator
    r = d["roofline"]
    assert 0 < r["step_frac_of_peak_32B"] < r["step_frac_of_peak_74B"] and "step_frac_of_peak" not in r
    assert abs(r["step_frac_of_peak_74B"] / r["step_frac_of_peak_32B"] - 74.0 / 32.0) < 1e-9
    # ncu-derived figures are attached only from a committed capture of the running build (hash-matched), never as literals:
    # a --size run has none
    assert r["traffic"] is None and r["issue"] is None and r["l2"] is None
    assert d["config"]["n_fail"] == 0 and 0 < d["config"]["live_fraction"] <= 1
    assert d["config"]["transport_path"][0] in (0, 1)
    for k in ("sm_mhz", "sm_max_mhz", "reasons"):
        assert k in d["clocks"], k


def test_ncu_figures_trace_to_a_committed_capture_of_this_build():
    """bench.py quotes roofline.traffic / issue / l2 only from profiles/*_metrics_c<config>.json whose source hash equals the
    hash of the library sources it runs (paper_2508_15532_b200/ncu_metrics.py); otherwise they are null."""
    import glob
    import json as js
    sys.path.insert(0, ROOT)
    import bench
    from paper_2508_15532_b200.ncu_metrics import source_hash
    classes, path = bench.ncu_metrics(4)
    files = glob.glob(os.path.join(ROOT, "profiles", "*_metrics_c4.json"))
    match = [f for f in files if js.load(open(f)).get("source_hash") == source_hash()]
    if match:
        assert classes is not None and os.path.join(ROOT, path) in match
        assert classes["transport"]["dram_bytes"] > 0 and classes["transport"]["warp_instr"] > 0
    else:
        assert classes is None and path is None
    assert not any(name.startswith("NCU_") for name in dir(bench))
