"""bench.py contract checks that need no GPU: the reference arm (the oracle timed on the host cores) prints
one JSON line with the keys the driver reads, and the roofline helpers read the committed profile data."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_json_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    j = json.loads(lines[0])
    assert j["impl"] == "reference" and j["metric"] == "sscn_steps_per_s" and j["unit"] == "steps/s"
    assert j["higher_is_better"] is True and j["vs_baseline"] is None and j["dtype"] == "f64"
    assert j["value"] > 0 and abs(j["ms_per_step"] * j["value"] - 1e3) < 1e-6 * 1e3
    assert j["cpu_baseline"]["kind"] == "oracle" and j["cpu_baseline"]["cores"] == 1
    assert j["e2e"] == {"value": j["value"], "unit": "steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "C4" in j["config"]["workload"] and "512x512x512" in j["config"]["workload"]


def test_traffic_table_names_the_kernels_of_the_step():
    sys.path.insert(0, ROOT)
    import bench
    for name in ("K1 dens_r2c(z)", "K3 fft_x*Udd*ifft_x", "K5+K8 c2r(z)+nonlinear+sweep_z", "K7 sweep_y(+norm)"):
        t = bench.ncu_traffic(name)
        assert t is not None and 1e9 < t < 1e10, name
        r = bench.ncu_traffic(name, rpsi=True)             # the real-valued path has its own capture
        assert r is not None and 1e9 < r <= t, name
    assert bench.ncu_traffic("no such kernel") is None
    peak, src = bench.load_peaks()
    assert 3000 < peak < 9000 and ("measured" in src or "fallback" in src)


def test_committed_ncu_tables_pair_the_step_kernels_with_the_right_cuda_kernels():
    """profiles/r2_*_ncu_full.md pairs the kernels of a step (bench.py names) with ncu's launches by ORDER: a kernel missing
    from the ncu filter shifts every row after it (it happened once).  Each row must name the kernel family of its stage."""
    import glob
    want = {"K1": "k_z_r2c", "K2": "k_fft", "K3": "k_fft", "K4": "k_fft", "K5+K8": "k_z_main", "K6": "k_sweep", "K7": "k_sweep"}
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "r2_*_ncu_full.md")))
    assert len(files) >= 3
    for path in files:
        rows = [l for l in open(path) if l.startswith("| K")]
        assert len(rows) == 7, path
        for line in rows:
            cells = [c.strip() for c in line.split("|")]
            stage, kernel = cells[1].split(" ")[0], cells[2]
            assert want[stage] in kernel, (path, stage, kernel)
            algorithmic, read, write = float(cells[6]), float(cells[4]), float(cells[5])
            assert 0.9 * algorithmic <= read + write <= 1.15 * algorithmic, (path, stage, read, write, algorithmic)


def test_measured_full_size_oracle_step_comes_from_the_golden_headers():
    """bench.py's cpu_baseline.measured_full_size_s_per_step is the oracle's measured time for one FULL-SIZE step, recorded in
    the headers of the goldens the oracle wrote offline (tests/golden/make_fullsize_goldens.py)."""
    sys.path.insert(0, ROOT)
    import bench
    from paper_1610_05329_b200 import inputs
    c4 = bench.measured_full_size(inputs.CONFIGS["C4"])
    c2 = bench.measured_full_size(inputs.CONFIGS["C2"])
    assert c4 is not None and 60.0 < c4 < 1000.0            # 512^3: minutes per step on one core
    assert c2 is not None and 0.5 < c2 < 30.0 and c2 < c4   # 128^3: seconds
    assert bench.measured_full_size(inputs.CONFIGS["C1"]) is None      # no full-size golden run for C1 (the tests run it live)
