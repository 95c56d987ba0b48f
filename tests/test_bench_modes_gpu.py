"""The commands profiles/ cites must keep running: bench.py's diagnostic modes on the small config (one GPU)."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(args, timeout=600):
    r = subprocess.run([sys.executable, "bench.py"] + args, cwd=ROOT, capture_output=True, text=True, timeout=timeout)
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    return json.loads(lines[0])


def test_default_mode_prints_one_parseable_contract_line(tmp_path):
    """The driver's own invocation shape (default mode) on the small config: exactly one stdout line starts with '{', it is
    strict JSON under 3 kB with the contract's keys, and the long material is in the --detail file."""
    detail = tmp_path / "detail.json"
    r = subprocess.run([sys.executable, "bench.py", "--config", "tiny", "--steps", "2", "--warmup", "1", "--per-config", "none",
                        "--detail", str(detail)], cwd=ROOT, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1 and r.stdout.rstrip().endswith(lines[0]) and len(lines[0].encode()) < 3000

    def bad(c):
        raise ValueError(c)
    d = json.loads(lines[0], parse_constant=bad)
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "dtype", "data",
              "config", "roofline", "cpu_baseline", "e2e", "clocks", "gpu_launches"):
        assert k in d, k
    assert d["value"] > 0 and d["steps"] == 2 and d["n_gpus"] == 1 and d["gpu_launches"] > 0
    assert d["config"]["workload"] == "tiny" and d["roofline"]["frac"] > 0 and d["cpu_baseline"]["value"] > 0
    assert d["e2e"]["value"] > 0 and d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0
    full = json.loads(detail.read_text())
    assert full["line"]["value"] == d["value"] and "policy" in full["headline"] and "alone" in full["headline"]


def test_gemm_only_mode_reports_plan_and_times():
    d = _run(["--mode", "gemm-only", "--config", "tiny", "--tile-k", "32"])
    assert d["mode"] == "gemm-only" and d["plan"]["tile_k"] == 32 and d["gemm_ms_burst"] > 0 and d["gemm_ms_sustained"] > 0


def test_power_table_mode_writes_rows(tmp_path):
    out = tmp_path / "power.md"
    d = _run(["--mode", "power-table", "--config", "tiny", "--loop-s", "0.05", "--table", str(out)])
    assert d["mode"] == "power-table" and len(d["rows"]) > 10 and all(r["runs"] >= 30 and r["ms_per_iter"] > 0 for r in d["rows"])
    assert out.read_text().count("\n") == len(d["rows"]) + 2
