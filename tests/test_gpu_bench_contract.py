"""bench.py prints ONE JSON line with the keys the driver reads (small workloads, so that the test takes seconds)."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
             "vs_baseline", "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "clocks", "gpu_launches"}


def run_bench(*args):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + list(args), capture_output=True, text=True,
                       cwd=ROOT, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, lines
    return json.loads(lines[0])


@pytest.mark.parametrize("workload", ["cfg2", "cfg4", "solve", "tree"])
def test_bench_line(workload):
    extra = ["--ncell", "32"] if workload != "solve" else ["--ncell", "32"]
    d = run_bench("--workload", workload, "--steps", "2", "--warmup", "1", "--e2e-steps", "1", "--ref-seconds", "0.2", *extra)
    assert BASE_KEYS <= set(d), BASE_KEYS - set(d)
    assert d["metric"] == "fmm_cell_interactions_per_s" and d["unit"] == "interactions/s" and d["dtype"] == "f64"
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["higher_is_better"] is True and d["vs_baseline"] is None
    assert d["warmup"] >= 3 and d["n_gpus"] == 1 and "workload" in d["config"]
    r = d["roofline"]
    assert {"bound", "achieved", "peak", "unit", "frac", "traffic"} <= set(r) and r["bound"] == "alu"
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    c = d["cpu_baseline"]
    assert {"value", "unit", "cores", "kind", "sample"} <= set(c) and c["kind"] == "oracle" and c["cores"] >= 1
    if workload in ("cfg2", "cfg4"):
        assert c["single_thread"]["cores"] == 1 and c["single_thread"]["value"] > 0
        assert "kernel_version" in r
    if workload == "tree":
        assert d["config"]["host_entry_bit_identical"] is True and d["config"]["net_force_over_sum_abs_force"] < 1e-13
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0
    assert e["value"] < d["value"] * 1.5                       # copies are inside the e2e region
    assert {"sm_mhz", "sm_max_mhz", "reasons"} <= set(d["clocks"]) and d["gpu_launches"] > 0


@pytest.mark.parametrize("halo", ["exchange", "peer"])
def test_coupled_line(halo):
    """--coupled (one problem in z-slabs, f4) carries the full key set in both halo modes; at N = 1 there are no neighbours."""
    d = run_bench("--coupled", "--halo", halo, "--workload", "cfg2", "--ncell", "32", "--steps", "2", "--warmup", "1",
                  "--e2e-steps", "1", "--ref-seconds", "0.2")
    assert BASE_KEYS <= set(d), BASE_KEYS - set(d)
    assert d["value"] > 0 and d["n_gpus"] == 1 and d["scaling"] == "weak" and d["roofline"]["bound"] == "alu"
    assert ("peer memory" in d["config"]["parallelism"]) == (halo == "peer")
    assert d["e2e"]["value"] > 0 and d["e2e"]["h2d_bytes_per_step"] > 0 and d["gpu_launches"] > 0
