"""The bench.py contract on a GPU box: one JSON line with the keys the driver reads, the roofline
and cpu_baseline objects, an end-to-end figure with its byte counts, clocks, and a non-zero count
of the library's own kernel launches.  Small workload (config 2, 64^3) so that it takes seconds;
the numbers themselves are not asserted."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _line(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], cwd=ROOT,
                         capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.strip().split("\n") if l.startswith("{")]
    assert len(lines) == 1, out.stdout[-2000:]
    return json.loads(lines[0])


def test_bench_line_contract():
    d = _line("--config", "2", "--steps", "8", "--warmup", "3")
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step",
              "higher_is_better", "scaling", "vs_baseline", "dtype", "data", "config", "clocks",
              "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert k in d, k
    assert d["metric"] == "two_component_d3q19_mlups" and d["unit"] == "MLUPS"
    assert d["n_gpus"] == 1 and d["steps"] == 8 and d["warmup"] == 3 and d["dtype"] == "f32"
    assert d["vs_baseline"] is None and d["data"] == "synthetic" and d["higher_is_better"] is True
    assert d["config"]["workload"] == "cfg2_contact_64"
    assert d["value"] > 0 and abs(d["value"] - d["config"]["fluid_nodes"] / d["ms_per_step"] / 1e3) < 1e-6 * d["value"]
    assert d["gpu_launches"] == 8 * 3                      # density, wall pass, fused pass per step
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and r["kernel"].startswith("k_collide_stream_bulk<float")
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and r["peak"] > 1000
    assert r["traffic"] is None                            # no ncu capture of this workload is committed
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and "fluid nodes" in c["sample"]
    e = d["e2e"]
    nbytes = 2 * 64 ** 3 * 8
    assert e["unit"] == "MLUPS" and 0 < e["value"] < d["value"]
    assert e["h2d_bytes_per_step"] == nbytes / 8 and e["d2h_bytes_per_step"] == nbytes / 8
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}


def test_reference_arm_line():
    d = _line("--impl", "reference", "--config", "2", "--steps", "2", "--warmup", "1")
    assert d["impl"] == "reference" and d["gpu_launches"] == 0 and d["dtype"] == "f64"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": "MLUPS", "h2d_bytes_per_step": 0,
                        "d2h_bytes_per_step": 0}
