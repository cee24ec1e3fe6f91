"""bench.py's contract line on a GPU box (a down-scaled config 3 so that it runs in seconds): every key the
driver reads is present and consistent.  The numbers themselves are not judged here."""
import json
import os
import subprocess
import sys

import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*extra):
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--scale", "0.06", "--steps", "4", "--warmup", "3", *extra]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=900)
    assert out.returncode == 0, out.stderr[-3000:]
    lines = [l for l in out.stdout.strip().splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout[-2000:]
    return json.loads(lines[0])


def test_bench_line_has_the_contract_keys():
    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device (no CPU fallback exists)")
    d = _run()
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "gpu_launches", "clocks"):
        assert k in d, k
    assert d["metric"] == "tf_update_latency_ms" and d["unit"] == "ms" and d["higher_is_better"] is False
    assert d["n_gpus"] == 1 and d["steps"] == 4 and d["warmup"] == 3 and d["vs_baseline"] is None
    assert d["dtype"] == "f32" and d["data"] == "synthetic" and "workload" in d["config"] and "model" not in d["config"]
    assert d["value"] > 0 and abs(d["value"] - d["ms_per_step"]) < 1e-9
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and r["kernel"] == "k_colorize"
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9 and r["achieved"] > 0
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["sample"]
    assert d["propagate_host_ms"] > 0 and d["update_incl_tf_upload_ms"] > d["propagate_host_ms"]     # incl. the TF upload
    assert d["tf_upload"]["tf_upload_bytes"] == 16 * d["config"]["leaves"] and "tf_sequence" in d["config"]
    e = d["e2e"]
    # (at this scale an update is tens of microseconds, so the two timings differ by their event overheads in either
    # direction: e2e must be a measurement of its own with its copies declared, not a value above the device-resident one)
    assert e["value"] > 0 and e["value"] != d["value"] and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0
    per_step = d["gpu_launches"] / d["steps"]
    assert per_step == int(per_step) and per_step >= 2                       # propagate launches + one colourise
    assert "sm_mhz" in d["clocks"] and "reasons" in d["clocks"]
    for k in ("packed", "attr", "render", "query"):                             # the NEXT rows report beside it
        assert k in d, k
    assert d["setup_s"].get("front_end_s", 0) > 0                               # device mipmap front end is the default


def test_bench_host_mipmap_and_fp16_variants_agree_on_the_workload():
    a = _run("--host-mipmap", "--no-cpu-baseline", "--no-e2e", "--no-render", "--no-query", "--no-packed", "--no-attr")
    b = _run("--format", "rgba16f", "--no-cpu-baseline", "--no-e2e", "--no-render", "--no-query", "--no-packed", "--no-attr")
    for k in ("mip_voxels", "nodes", "leaves", "topo_depth"):
        assert a["config"][k] == b["config"][k], k
    assert "front_end_s" not in a["setup_s"] and a["config"]["output"] == "rgba8" and b["config"]["output"] == "rgba16f"
    assert b["roofline"]["algorithmic_bytes_per_launch"] == 12 * b["config"]["mip_voxels"]


def test_bench_config5_reports_both_bandwidth_bound_kernels():
    """Config 5 (scaled to 10 M nodes: a 161 MB palette, beyond the L2): loaded with MG_RELABEL by default, both kernels carry a roofline object, the one that takes
    longer is `roofline`; --device-levels changes the setup only."""
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--config", "5", "--scale", "0.15", "--steps", "4", "--warmup", "3",
           "--no-cpu-baseline", "--no-e2e", "--no-packed", "--no-attr"]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=900)
    assert out.returncode == 0, out.stderr[-3000:]
    d = json.loads([l for l in out.stdout.strip().splitlines() if l.startswith("{")][-1])
    assert d["config"]["workload"].startswith("cfg5") and d["value"] > 0
    names = {d["roofline"]["kernel"], d["roofline_second_kernel"]["kernel"]}
    assert "k_level" in names and len(names) == 2
    assert d["roofline"]["avg_launch_ms"] >= d["roofline_second_kernel"]["avg_launch_ms"]
    a = _run("--device-levels", "--no-cpu-baseline", "--no-e2e", "--no-render", "--no-query", "--no-packed", "--no-attr")
    assert a["setup_s"]["device_levels_done"] >= 1 and a["value"] > 0
