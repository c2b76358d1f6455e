"""The reference arm of bench.py (the oracle timed on the host cores) prints the contract's JSON line; runs on CPU."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_contract_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "fresnel_surface_propagations_per_sec"
    assert d["unit"] == "surface-propagations/s" and d["higher_is_better"] is True and d["vs_baseline"] is None
    assert d["value"] > 0 and d["steps"] == 1 and d["n_gpus"] == 1 and d["gpu_launches"] == 0
    assert d["config"]["workload"] == "cfg3_spc_2048_c128"
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == d["value"] and "sample" in cb
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


def test_profile_formatters_run_without_a_gpu(tmp_path):
    """bench.py --format-sweep / --launch-summary: the committed commands behind profiles/*_sweep.md and *_launches.md."""
    sweep = {"peak_gbs": 6537.0, "sweep": [{"N": 2048, "complex": "c128", "us_mean": 82.9, "us_sigma": 0.1, "row_us": 43.0, "col_us": 44.8,
                                            "frac_4S_of_peak": 0.495, "frac_6S_model_at_8TBs": 0.607, "cufft_unfused_us": 210.4}],
             "small_trains": [{"workload": "cfg1", "N": 256, "surfaces": 1, "passes": 2, "eager_us": 33.0, "graph_us": 12.3}],
             "mft": [{"na": 1024, "nb": 256, "complex": "c128", "batch": 1, "us": 260.0, "flops": 2.68e9, "tflops": 10.3, "frac_of_peak": 0.35}],
             "accumulate_intensity": [{"N": 4096, "complex": "c64", "batch": 16, "us": 421.8, "frac_of_peak": 0.83}]}
    f = tmp_path / "sweep.json"
    f.write_text(json.dumps(sweep) + "\n")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--format-sweep", str(f)], capture_output=True, text=True, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    assert "| 2048 | c128 | 82.9 | 0.1 | 43.0 | 44.8 | 0.495 | 0.607 | 210.4 |" in r.stdout
    assert "| cfg1 | 256 | 1 | 2 | 33.0 | 12.3 |" in r.stdout and "| 1024 → 256 | c128 | 1 | 260.0 |" in r.stdout
    hdr = '"ID","Process ID","Process Name","Host Name","Kernel Name","Context","Stream","Block Size","Grid Size","Device","CC","Section Name","Metric Name","Metric Unit","Metric Value"\n'
    row = '"{i}","1","python","h","{k}","1","13","(128, 1, 1)","(16, 1, 1)","0","10.0","s","gpu__time_duration.sum","ns","{ns}"\n'
    c = tmp_path / "launches.csv"
    c.write_text(hdr + row.format(i=0, k="kern_a", ns=3000) + row.format(i=1, k="kern_a", ns=5000) + row.format(i=2, k="kern_b", ns=2000))
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--launch-summary", str(c)], capture_output=True, text=True, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    assert "| `kern_a` | 2 | 8.0 | 4.0 | 0.800 |" in r.stdout and "| `kern_b` | 1 | 2.0 | 2.0 | 0.200 |" in r.stdout
