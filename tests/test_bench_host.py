"""Host-side pieces of bench.py that need no GPU: the figures it reads from the committed ncu summary (roofline.traffic,
fp64_pipe_pct, l2_hit_pct), the bounded oracle sample, and the reference arm on a small workload (the CPU oracle timed
as it stands)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_profile_figures_come_from_the_committed_summary():
    sys.path.insert(0, ROOT)
    import bench
    f = bench.profile_file()
    assert f and f.startswith("profiles/") and os.path.exists(os.path.join(ROOT, f))
    traffic = bench.profiled_traffic()
    assert traffic is not None and 7.38e9 < traffic < 3e10          # above the compulsory bytes of a config-4 launch
    assert 0.0 < bench.profiled_traffic(key="fp64_pipe_pct") < 100.0
    assert 0.0 < bench.profiled_traffic(key="l2_hit_pct") < 100.0
    assert isinstance(bench.cpu_model(), str) and bench.cpu_model()
    assert bench.FULL_2D_REPLICA_STEPS == 16383


def test_reference_arm_prints_one_json_line_on_a_small_workload():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "cfg3s",
                          "--steps", "2", "--warmup", "1"], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-500:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "cell-updates/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["gpu_launches"] == 0
