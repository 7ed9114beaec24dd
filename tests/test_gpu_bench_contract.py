"""bench.py prints ONE JSON line with the keys the driver reads (pytest -m gpu; small workload)."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_bench_line_has_the_contract_keys():
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--workload", "W3", "--steps", "20", "--warmup", "3",
                        "--cpu-steps", "1", "--quick", "--compare", "--sweep", "W1,W3,P1"], capture_output=True, text=True, timeout=900)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "gpu_launches", "roofline", "cpu_baseline", "e2e"):
        assert k in d, k
    assert d["unit"] == "MLUPS" and d["n_gpus"] == 1 and d["steps"] == 20 and d["dtype"] == "f32" and d["vs_baseline"] is None
    assert d["config"]["workload"] == "W3" and "model" not in d["config"]
    assert d["gpu_launches"] > 20 * 15                 # a coupled W3 step is ~20 kernels of this library (one of them the whole MDF loop)
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    assert 0.3 < r["frac"] < 1.2
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] > 0
    e = d["e2e"]
    assert e["unit"] == "MLUPS" and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0
    assert 0 < e["value"] <= d["value"] * 1.05          # end to end cannot beat the resident step
    assert d["serial_chain"]["value"] > 0 and 0.0 <= d["ibm_share"] < 1.0
    assert d["comparisons_ms_per_step"]["default"] > 0
    # the whole step against the HBM roofline, and the kernel with the largest time share (the tile pass)
    rs, ri = d["roofline_step"], d["roofline_ibm"]
    assert rs["bound"] == "hbm" and abs(rs["frac"] - rs["achieved"] / rs["peak"]) < 1e-12 and 0.0 < rs["frac"] < 1.0
    assert abs(rs["achieved"] - rs["algorithmic_bytes_per_step"] / (d["ms_per_step"] * 1e-3) / 1e9) < 1e-6 * rs["achieved"]
    assert ri["bound"] == "alu" and ri["unit"] == "TFLOP/s" and 0.0 < ri["frac"] < 1.0 and "k_mdf_tiles" in ri["kernel"]
    assert r["traffic"] is None or "not measured in this run" in r["traffic_source"]
    assert e["changed_table_value"] > 0 and e["with_fields_every_10_steps_value"] > 0 and e["blocking_read_value"] > 0
    assert d["cpu_baseline"]["same_config_as_gpu_arm"] is True and d["cpu_baseline"]["pure_lbm_value"] > 0
    assert d["cpu_baseline"]["host"]["nproc"] >= 1
    # the metric as a curve: one entry per workload of the sweep, the main workload's entry = the headline
    sw = {x["workload"]: x for x in d["density_sweep"]}
    assert set(sw) == {"W1", "W3", "P1"}
    for x in sw.values():
        assert abs(x["coupled_over_pure"] - x["pure_ms_per_step"] / x["ms_per_step"]) < 1e-12
        assert 0.0 < x["step_hbm_frac"] < 1.0 and 0.0 <= x["ibm_share"] < 1.0 and x["markers_per_active_cell"] > 0
    assert sw["W3"]["ms_per_step"] == d["ms_per_step"] and sw["P1"]["paper_context"]["mlups"] == 893.0
