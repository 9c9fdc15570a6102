"""bench.py's constants and its reference arm (-m "not gpu")."""
import json
import os
import subprocess
import sys

import oracle as o

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_flops_per_photon_step_is_the_oracle_tally():
    sys.path.insert(0, ROOT)
    import bench
    y = o.init_ray(0.7, 1000.0, 45.0, 3.0, 4.0)
    for name, rule in (("rel", o.STEP_REL), ("eq2", o.STEP_EQ2)):
        t = o.op_tally(0.7, y, 1 / 32, rule)
        assert bench.FLOPS_PER_PHOTON_STEP[name] == t["add"] + t["mul"] + t["div"] + t["sqrt"] + t["sin"] + t["cos"]
    assert abs(bench.PEAK_TFLOPS["f32"] - 74.45) < 0.05 and abs(bench.PEAK_TFLOPS["f64"] - 37.2) < 0.05


def test_reference_arm_prints_one_json_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0",
                          "--ref-log2n", "9", "--log2n", "20"], capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    j = json.loads(lines[0])
    assert j["impl"] == "reference" and j["unit"] == "photon-steps/s" and j["value"] > 1e5
    assert j["cpu_baseline"]["kind"] == "oracle" and j["e2e"]["h2d_bytes_per_step"] == 0
