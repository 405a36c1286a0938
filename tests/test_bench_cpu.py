"""bench.py without a GPU: the reference arm (the oracle on the host cores) prints the contract's JSON line, and the
roofline's `traffic` comes from the committed ncu table, not from a constant."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "C1", "--steps", "2",
                          "--warmup", "1"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "gravity_interactions_per_s" and line["unit"] == "interactions/s"
    assert line["higher_is_better"] is True and line["steps"] == 2 and line["warmup"] == 1 and line["dtype"] == "f64"
    assert line["config"]["workload"].startswith("C1: plummer N=16384")
    assert line["value"] > 0 and line["ms_per_step"] > 0
    cb = line["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == line["value"] and "groups" in cb["sample"]
    assert line["e2e"] == {"value": line["value"], "unit": line["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert line["gpu_launches"] == 0


def test_reference_arm_other_ranks_do_no_work():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "C1", "--gpus", "2"],
                         capture_output=True, text=True, timeout=120, cwd=ROOT, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_traffic_comes_from_the_committed_profile():
    sys.path.insert(0, ROOT)
    import bench
    t, src = bench.committed_traffic("C5", "walk_gravity_ws_kernel")
    assert t is not None and t > 1e9 and "profiles/" in src          # one ncu launch at C5: a few GB
    t2, why = bench.committed_traffic("C5:custom", "walk_gravity_ws_kernel")
    assert t2 is None and "no row" in why
    assert bench.BUILD_BYTES_PER_PARTICLE == 370                       # SURVEY 8(d)'s figure
