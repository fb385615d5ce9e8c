"""bench.py's JSON contract, checked on the CPU through the reference arm (the CUDA arm needs a GPU)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_json_line_with_the_contract_keys():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0", "--ref-sample", "32"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
              "scaling", "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert k in d, k
    assert d["impl"] == "reference" and d["metric"] == "pcmd_model_evals_per_s" and d["unit"] == "evals/s"
    assert d["vs_baseline"] is None and d["data"] == "synthetic" and d["config"]["workload"] == "c3"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"] > 0


def test_roofline_constants():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.i_alg(3) == 16 and bench.i_alg(2) == 15
    peaks, which = bench.measured_peaks()
    assert peaks["hbm_gbs"] > 1000 and which in ("measured", "fallback")
