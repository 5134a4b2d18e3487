"""-m gpu: bench.py's JSON contract on the GPU arm, on the smallest workload (config 1) so that it takes seconds."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_gpu_arm_prints_one_json_line_with_the_contract_keys():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--config", "1", "--no-per-config", "--steps", "3",
                          "--warmup", "3", "--cpu-seconds", "1"], capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["metric"] == "coupled photon-electron histories/s" and d["unit"] == "histories/s"
    assert d["higher_is_better"] is True and d["scaling"] == "weak" and d["data"] == "synthetic" and d["dtype"] == "f32"
    assert d["n_gpus"] == 1 and d["steps"] == 3 and d["warmup"] == 3 and d["vs_baseline"] is None
    assert d["config"]["workload"] == "cfg1_2MeV_photon_pencil_water32" and "l2" in d["config"]
    assert d["value"] > 0 and d["ch_steps_per_s"] > 0 and d["ms_per_step"] > 0
    assert d["value"] == pytest.approx(1e5 / (d["ms_per_step"] * 1e-3), rel=1e-6)
    assert d["gpu_launches"] == 3                                   # one persistent kernel per step
    r = d["roofline"]
    assert r["bound"] == "alu" and r["unit"] == "thread-inst/s" and 0 < r["frac"] < 1
    assert r["frac"] == pytest.approx(r["achieved"] / r["peak"]) and r["traffic"] > 0
    assert 0.5 < r["kernel_share_of_step"] <= 1.0                   # CUDA events inside the library vs around gpumcd_run
    t = d["roofline_tally"]
    assert t["bound"] == "l2_atomic" and 0 < t["frac"] < 1 and t["peak"] > 1e9
    e = d["e2e"]
    assert e["unit"] == "histories/s" and 0 < e["value"] < d["value"]
    assert e["h2d_bytes_per_step"] >= 5 * 32 ** 3 and e["d2h_bytes_per_step"] == 4 * 32 ** 3
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and "sample" in c
    k = d["clocks"]
    assert k["sm_mhz"] > 0 and k["sm_max_mhz"] >= k["sm_mhz"] and isinstance(k["reasons"], list)
