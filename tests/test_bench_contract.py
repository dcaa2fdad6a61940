"""bench.py keeps the driver's contract: one JSON line with the required keys, on the small config
(GPU), and the site-update accounting used by both arms (CPU)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_site_update_accounting():
    sys.path.insert(0, ROOT)
    import bench
    n, R, M, nt, n_p = 1000, 2, 3000, 1, 42
    lit = bench.site_updates(n, R, M, nt, n_p)
    dbl = bench.site_updates(n, R, M, nt, n_p, doubling=True)
    per = n * R
    assert lit["dos"] == (M - 1) * per                                        # Alg. 5: M - 1 applications
    assert lit["vac"] == (1 + 2 * (1 + M - 1) + 2 * (n_p - 1)) * per          # Alg. 2, two time points
    assert lit["msd"] == ((M - 1) + 2 * (n_p - 1)) * per                      # Alg. 3, pair recursion; row 0 = 0 is not computed
    assert dbl["dos"] == (M // 2) * per
    assert dbl["vac"] == (1 + M // 2 + (1 + 2 * (M // 2)) + 2 * (n_p - 1)) * per   # row 0: one column; row 1: both chains
    assert dbl["msd"] == ((M // 2) + 2 * (n_p - 1)) * per
    assert bench.mom_bytes_per_update(1) == 108.0 and bench.mom_bytes_per_update(8) == 69.5
    assert bench.mom_bytes_per_update(2, phi_l_stream=False) == 70.0


@pytest.mark.gpu
def test_bench_line_on_small_config():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--config", "1", "--steps", "2",
                          "--warmup", "3", "--no-cpu-baseline"], capture_output=True, text=True, cwd=ROOT,
                         timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1                                                    # exactly one JSON line
    b = json.loads(lines[0])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
                "scaling", "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline"):
        assert key in b, key
    assert b["n_gpus"] == 1 and b["steps"] == 2 and b["warmup"] == 3 and b["higher_is_better"] is True
    assert b["scaling"] == "weak" and b["data"] == "synthetic" and b["vs_baseline"] is None
    assert "workload" in b["config"] and b["value"] > 0 and b["gpu_launches"] > 0
    assert set(("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step")) <= set(b["e2e"])
    assert b["e2e"]["h2d_bytes_per_step"] > 0 and b["e2e"]["d2h_bytes_per_step"] > 0
    r = b["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    assert 0 < r["job_weighted"]["frac"] and "timed_as" in r and "second_kernel" in r
    assert b["setup"]["create_s"] > 0 and b["setup"]["first_step_s"] > 0


def test_reference_arm_line_on_the_cpu():
    """`bench.py --impl reference` (the oracle timed on the host cores) prints ONE JSON line with the driver's keys,
    the oracle described in cpu_baseline, and an e2e block repeating the value; no GPU involved."""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--shrink", "25",
                          "--steps", "2", "--warmup", "1"], capture_output=True, text=True, cwd=ROOT, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    b = json.loads(lines[0])
    assert b["impl"] == "reference" and b["steps"] == 2 and b["warmup"] == 1 and b["higher_is_better"] is True
    for key in ("metric", "value", "unit", "n_gpus", "ms_per_step", "scaling", "vs_baseline", "dtype", "data", "config",
                "cpu_baseline", "e2e", "gpu_launches"):
        assert key in b, key
    assert b["value"] > 0 and b["gpu_launches"] == 0 and b["vs_baseline"] is None
    cb = b["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] == 1 and cb["value"] == b["value"] and "recursion + dot" in cb["sample"]
    assert cb["cpu_model"] and cb["host_cores_available"] >= 1
    assert b["e2e"] == {"value": b["value"], "unit": b["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
