"""bench.py contract pieces that run without a GPU: the reference arm (the oracle on the host cores) prints one
JSON line with the keys the driver reads; the algorithmic byte / flop counts are the ones SURVEY.md 8d tabulates."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_json_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "C1",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "Mvox/s" and d["higher_is_better"] is True
    assert d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["gpu_launches"] == 0


def test_algorithmic_counts_match_the_survey_table():
    sys.path.insert(0, ROOT)
    import bench
    from paper_1706_02261_b200 import workloads as wl
    # C4 8.39 MB HBM, 50.3 MB L2, 251.7 MFLOP per step; C5 summed 2.10 MB, 138.4 MB, 922.7 MFLOP; per-field 17.8 MB
    hbm, l2, flop = bench.algorithmic_per_step(wl.config("C4"))
    assert abs(hbm / 1e6 - 8.39) < 0.01 and abs(l2 / 1e6 - 50.3) < 0.1 and abs(flop / 1e6 - 251.7) < 0.1
    hbm, l2, flop = bench.algorithmic_per_step(wl.config("C5"))
    assert abs(hbm / 1e6 - 2.10) < 0.01 and abs(l2 / 1e6 - 138.4) < 0.1 and abs(flop / 1e6 - 922.7) < 0.1
    hbm, l2, flop = bench.algorithmic_per_step(wl.config("C5"), per_field_intensity=True)
    assert abs(hbm / 1e6 - 17.8) < 0.1
