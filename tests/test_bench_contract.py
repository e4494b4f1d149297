"""bench.py contract on the CPU side: the reference arm (the oracle timed on the host cores) prints one JSON line with the
keys the driver reads, for a fit and for a build workload (small overrides so that it runs in seconds)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
KEYS = {"impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
        "dtype", "data", "config", "cpu_baseline", "e2e", "gpu_launches"}


def run(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0", *args],
                         capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    return json.loads(lines[0])


def test_reference_arm_fit():
    d = run("--workload", "fit_c1", "--tracks", "20000", "--ref-sample", "5000")
    assert KEYS <= set(d) and d["impl"] == "reference" and d["metric"] == "tracks_fitted_per_s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["vs_baseline"] is None
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0 and d["gpu_launches"] == 0
    assert d["config"]["workload"] == "fit_c1"


def test_reference_arm_build():
    d = run("--workload", "build_c3", "--events", "2", "--ref-events", "1")
    assert KEYS <= set(d) and d["metric"] == "seeds_built_per_s" and d["unit"] == "seeds/s" and d["value"] > 0
    assert d["config"]["workload"] == "build_c3"


def test_reference_arm_build_on_the_cylinder_with_lids():
    d = run("--workload", "build_lids_two_step", "--events", "1", "--ref-events", "1")
    assert KEYS <= set(d) and d["metric"] == "seeds_built_per_s" and d["value"] > 0 and d["config"]["layers"] == 18
