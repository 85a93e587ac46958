"""Host-side logic of bench.py that needs no GPU: the byte accounting of P:333-335, the committed traffic table,
the roofline arithmetic, and the reference arm (the oracle timed on the host cores) end to end."""
import csv
import json
import os
import re
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def test_bytes_per_cell_match_the_papers_counts():
    import bench
    assert bench.bytes_per_cell(15, 27) == (280, 488)          # P:333, P:335 (D3Q15 phase, D3Q27 hydro, fp64)
    assert bench.bytes_per_cell(15, 19) == (280, 360)
    assert bench.bytes_per_cell(27, 27) == (472, 488)
    assert bench.bytes_per_cell(27, 27, 4) == (236, 244)
    assert sum(bench.bytes_per_cell(15, 19)) == 640 and sum(bench.bytes_per_cell(27, 27, 4)) == 480


def test_traffic_table_rows_carry_the_commit_of_their_build():
    import bench
    rows = list(csv.DictReader(open(os.path.join(ROOT, "profiles", "traffic.csv"))))
    assert len(rows) >= 6
    for r in rows:
        assert re.fullmatch(r"[0-9a-f]{7,40}", r["commit"]), r
        assert float(r["dram_bytes_per_launch"]) > 1e9
    t, commit = bench.traffic_row("hydro_kernel", 3, "f64")
    assert commit and 0.95 < t / (360 * 256 ** 3) < 1.05       # traffic = algorithmic bytes within 5 %
    t, commit = bench.traffic_row("hydro_kernel", 5, "f32")
    assert commit and 0.95 < t / (244 * 256 ** 3) < 1.05
    assert bench.traffic_row("hydro_kernel", 99, "f64") == (None, None)
    # moment representation: 128 + 216 B per cell whatever the lattices
    assert bench.bytes_per_cell_moments() == (128, 216)
    for cfg in (3, 5):
        t, commit = bench.traffic_row("hydro_mom_kernel", cfg, "f64")
        assert commit and 0.95 < t / (216 * 256 ** 3) < 1.05
        t, commit = bench.traffic_row("phase_mom_kernel", cfg, "f64")
        assert commit and 0.95 < t / (128 * 256 ** 3) < 1.05


def test_roofline_arithmetic():
    import argparse
    import bench
    N = 256 ** 3
    r = {"hydro_ms": 0.9, "phase_ms": 0.7, "b_hydro": 360, "b_phase": 280, "N": N, "ms": 1.6 * 20}
    args = argparse.Namespace(unfused=False)
    roof, step_gbs, peak = bench.roofline_of(args, 3, "f64", r, 20)
    assert roof["kernel"] == "hydro_kernel" and roof["bound"] == "hbm" and roof["unit"] == "GB/s"
    assert abs(roof["achieved"] - 360 * N / 0.9e-3 / 1e9) < 1e-6
    assert abs(roof["frac"] - roof["achieved"] / peak) < 1e-12
    assert abs(roof["frac_of_nominal"] - roof["achieved"] / 8000.0) < 1e-12
    assert roof["peak_is_lower_bound"] == (roof["achieved"] > peak)
    assert abs(step_gbs - 640 * N / 1.6e-3 / 1e9) < 1e-6
    assert abs(roof["kernel_share_of_step"] - 0.9 / 1.6) < 1e-12
    m = {"hydro_ms": 0.9, "phase_ms": 0.62, "b_hydro": 216, "b_phase": 128, "N": N, "ms": 1.52 * 20, "moments": True}
    roof, step_gbs, peak = bench.roofline_of(args, 3, "f64", m, 20)
    assert roof["kernel"] == "hydro_mom_kernel" and roof["traffic"] and abs(roof["achieved"] - 216 * N / 0.9e-3 / 1e9) < 1e-6


def test_reference_arm_prints_one_json_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "MLUPS" and d["value"] > 0 and d["higher_is_better"] is True
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["gpu_launches"] == 0
