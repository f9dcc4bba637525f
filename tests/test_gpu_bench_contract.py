"""bench.py's output contract on the small configuration: one JSON line on stdout with the keys the driver reads, the
roofline and cpu_baseline objects, a non-zero launch count, and both arms (ours, reference) agreeing on metric / unit /
workload."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(args):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + args, cwd=ROOT, capture_output=True, text=True,
                       timeout=900)
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout[-2000:]
    return json.loads(lines[0])


def test_json_line_of_both_arms():
    ours = _run(["--config", "0", "--steps", "20", "--warmup", "3", "--mp-apertures", "8"])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert key in ours, key
    assert ours["n_gpus"] == 1 and ours["steps"] == 20 and ours["warmup"] == 3 and ours["higher_is_better"] is True
    assert ours["value"] > 0 and abs(ours["value"] * ours["ms_per_step"] * 1e-3 - 1.0) < 1e-6
    assert ours["vs_baseline"] is None and ours["dtype"] == "f32" and ours["data"] == "synthetic"
    assert "workload" in ours["config"] and "model" not in ours["config"]
    assert ours["gpu_launches"] == 4 * 20                            # dose(+objective), partial sum, price(+selection), aperture price
    e2e = ours["e2e"]
    assert e2e["value"] > 0 and e2e["h2d_bytes_per_step"] == 4 * ours["config"]["n_beamlets"] and e2e["d2h_bytes_per_step"] > 0
    assert e2e["value"] != ours["value"]
    rf = ours["roofline"]
    assert rf["bound"] == "hbm" and rf["unit"] == "GB/s" and rf["peak"] > 0 and "traffic" in rf
    assert abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-9
    cb = ours["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] == 1 and cb["value"] > 0 and cb["unit"] == ours["unit"] and cb["sample"]
    assert {"sm_mhz", "sm_max_mhz", "reasons"} <= set(ours["clocks"])
    for section in ("master_problem", "plan_optimisation", "constrained_selection", "plan_optimisation_constrained"):
        assert section in ours, section
    assert ours["plan_optimisation"]["F_end"] < 0.01 * ours["plan_optimisation"]["F_start"]
    sus = ours["sustained"]                                          # the steady-state leg behind the K timed steps
    assert sus["steps"] >= 20 and sus["evals_per_s"] > 0 and sus["seconds"] > 0
    assert abs(sus["evals_per_s"] * sus["ms_per_step"] * 1e-3 - 1.0) < 1e-6
    assert len(sus["kernels"]) == 2 and all(k["ms"] > 0 and k["gbs"] > 0 for k in sus["kernels"])
    assert {"sm_mhz", "sm_max_mhz", "reasons"} <= set(sus["clocks"])
    assert "copied_back" in e2e

    ref = _run(["--impl", "reference", "--config", "0", "--steps", "3", "--warmup", "1"])
    assert ref["impl"] == "reference" and ref["metric"] == ours["metric"] and ref["unit"] == ours["unit"]
    assert ref["config"]["workload"] == ours["config"]["workload"] and ref["higher_is_better"] is True
    assert ref["e2e"] == {"value": ref["value"], "unit": ref["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert ref["cpu_baseline"]["kind"] == "oracle" and ref["cpu_baseline"]["value"] == ref["value"]
    for key in ("n_voxels", "n_beamlets", "nnz", "n_angles", "n_leaf_rows"):        # the whole matrix: the GPU arm's sizes
        assert ref["config"][key] == ours["config"][key], key
