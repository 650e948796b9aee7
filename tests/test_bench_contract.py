"""The bench.py contract: one JSON line with the keys the driver reads, for both arms.  The
reference arm (the oracle on the host cores) needs no GPU; our arm runs on a small copy of the
headline workload under -m gpu."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
COMMON = ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
          "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches", "cpu_baseline")


def _run(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                         timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, out.stdout
    return json.loads(lines[0])


def test_reference_arm_prints_one_json_line():
    d = _run("--impl", "reference", "--workload", "c3_small", "--steps", "1", "--warmup", "1")
    for k in COMMON:
        assert k in d, k
    assert d["impl"] == "reference" and d["gpu_launches"] == 0 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"]
    assert d["config"]["workload"] == "c3_collision_16"


@pytest.mark.gpu
def test_our_arm_prints_one_json_line_with_roofline_and_e2e():
    d = _run("--workload", "c3_small", "--steps", "2", "--warmup", "3")
    for k in COMMON + ("roofline", "clocks", "e2e_stepping"):
        assert k in d, k
    r = d["roofline"]
    assert r["bound"] == "alu" and r["unit"] == "TFLOP/s" and 0 < r["frac"] < 1.2
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    assert d["gpu_launches"] == 2 * 3                       # 2 steps x (pre-pass, pairwise, epilogue)
    assert d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0
    assert d["e2e"]["value"] != d["value"] and d["dtype"] == "f32" and d["scaling"] == "weak"
    assert d["cpu_baseline"]["kind"] == "oracle"
    ref = _run("--impl", "reference", "--workload", "c3_small", "--steps", "1", "--warmup", "1")
    assert ref["config"] == d["config"]                    # the two arms describe the same workload
