"""The measurement contract of bench.py, run as the driver runs it (a subprocess, one JSON line on stdout): required
keys, the roofline / cpu_baseline / e2e objects, both modes in one line, and the reference arm. Small configuration so
that the whole test takes seconds; the numbers themselves are not asserted (they belong to the B200 the driver uses)."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _line(*flags):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *flags], capture_output=True, text=True, timeout=600,
                       cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, r.stdout[-1000:]
    return json.loads(lines[0])


def test_gpu_arm_line_has_the_contract_keys():
    d = _line("--config", "3", "--steps", "2", "--warmup", "3", "--other-mode-steps", "1")
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "gpu_launches", "clocks"):
        assert k in d, k
    assert d["unit"] == "updates/s" and d["dtype"] == "f64" and d["n_gpus"] == 1 and d["vs_baseline"] is None
    assert d["value"] > 0 and d["gpu_launches"] > 0 and d["finite"] is True
    assert "workload" in d["config"] and "model" not in d["config"]
    rf = d["roofline"]
    assert rf["bound"] == "hbm" and rf["unit"] == "GB/s" and 0 < rf["frac"] < 1.2 and abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-9
    assert "traffic" in rf and d["roofline_ghost"]["kernel"] == "ghost_dense_prolong"
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] > 0 and "SAMPLE" in cb["sample"] or "all" in cb["sample"]
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0 and e["value"] < d["value"]
    sv = d["sub_vs_uniform"]
    assert sv["speedup_vs_uniform"] > 1.0 and abs(sv["level_work_ratio"] - 32.0 / 15.0) < 1e-9
    assert set(d["stream_ceiling"]) >= {"R1W1", "R2W2", "R4W3"} and d["graph"]["instantiations"] >= 1
    assert d["clocks"]["sm_max_mhz"] > 0


def test_gpu_arm_takes_the_next_row_options():
    d = _line("--config", "1", "--steps", "2", "--warmup", "3", "--other-mode-steps", "0", "--no-cpu-baseline", "--integrator", "3",
              "--outer-bc", "1", "--fd-order", "8", "--sigma", "0.2")
    c = d["config"]
    assert c["integrator"] == 3 and c["outer_bc"] == 1 and c["fd_order"] == 8 and c["ghost"] == 5 and d["finite"] is True


def test_reference_arm_line():
    d = _line("--impl", "reference", "--config", "1", "--steps", "1", "--warmup", "0")
    assert d["impl"] == "reference" and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    c = d["config"]  # cfg 1 has two levels: the oracle times all of it, and the config says so
    assert c["sampled"] is False and c["sample_levels"] == 2 and c["sample_updates_per_step"] == c["updates_per_step"]


def test_reference_arm_says_when_it_timed_a_sample():
    """The reference arm prints the GPU arm's config, but on deep hierarchies it times the first levels only: the
    config carries the sample (identical configs on different work must not pass silently)."""
    d = _line("--impl", "reference", "--config", "1", "--steps", "1", "--warmup", "0", "--oracle-levels", "1")
    c = d["config"]
    assert c["sampled"] is True and c["sample_levels"] == 1 and 0 < c["sample_updates_per_step"] < c["updates_per_step"]
    assert "SAMPLE" in c["ms_per_step_is"] and "SAMPLE" in d["cpu_baseline"]["sample"]
    # value is the sample's rate: updates of the sample / time of the sample
    assert abs(d["value"] * d["ms_per_step"] * 1e-3 / c["sample_updates_per_step"] - 1.0) < 1e-6
