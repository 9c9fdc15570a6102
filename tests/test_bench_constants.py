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
        t = o.op_tally(0.7, y, 1 / 32, rule, o.SYS_REDUCED)
        assert bench.FLOPS_PER_PHOTON_STEP_REDUCED[name] == t["add"] + t["mul"] + t["div"] + t["sqrt"] + t["sin"] + t["cos"]
        # the reduced oracle = the full one + five (k^t, k^phi) reconstructions: 4 stages + the final state
        assert t["sin"] == 9 and t["cos"] == 9
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


def test_launcher_command_starts_one_rank_per_gpu(monkeypatch):
    # `python bench.py --gpus N` by hand must start N ranks itself (row (e) of the scope table)
    sys.path.insert(0, ROOT)
    import argparse

    import bench
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    a = argparse.Namespace(gpus=4, impl="gray")
    cmd = bench.launcher_command(a, ["--gpus", "4", "--steps", "2"], port=29999)
    assert cmd[1:4] == ["-m", "torch.distributed.run", "--nnodes=1"] and "--nproc-per-node=4" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "29999"
    assert cmd[-4:] == ["--gpus", "4", "--steps", "2"] and cmd[-5].endswith("bench.py")
    assert bench.launcher_command(argparse.Namespace(gpus=1, impl="gray"), []) is None
    assert bench.launcher_command(argparse.Namespace(gpus=4, impl="reference"), []) is None
    monkeypatch.setenv("WORLD_SIZE", "4")                    # already inside torchrun (the driver's launch): no re-launch
    assert bench.launcher_command(a, []) is None


def test_profile_csv_readers():
    sys.path.insert(0, ROOT)
    import bench
    b, src = bench.ncu_dram_bytes_per_photon()
    assert src is not None and 74.0 <= b <= 76.0          # 74 B algorithmic per photon (fp32): DESIGN.md "Data layout"
    assert bench.variant_name("f32", "eq2", "realistic", 0.0, "full", 0) == "f32_eq2"
    assert bench.variant_name("f64", "eq2", "realistic", 1e-3, "full", 0) == "f64_eq2_xi"
    assert bench.variant_name("f32", "rel", "peak", 0.0, "full", 0) == "f32_rel_frozen"
    # executed FP operations per issued lane-step (ncu): below the oracle's nominal tally, above the FMA-only floor
    for variant, lo, hi in (("f32_eq2", 400, 787), ("f64_eq2", 500, 787), ("f32_eq2_xi", 450, 900), ("f32_rel_frozen", 400, 777),
                            ("f32x1_eq2", 400, 787)):
        e = bench.executed_flops_per_lane_step(variant)
        assert e is not None and lo < e < hi, (variant, e)
    assert bench.executed_flops_per_lane_step("no_such_variant") is None
