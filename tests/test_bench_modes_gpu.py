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


def test_gemm_only_mode_reports_plan_and_times():
    d = _run(["--mode", "gemm-only", "--config", "tiny", "--tile-k", "32"])
    assert d["mode"] == "gemm-only" and d["plan"]["tile_k"] == 32 and d["gemm_ms_burst"] > 0 and d["gemm_ms_sustained"] > 0


def test_power_table_mode_writes_rows(tmp_path):
    out = tmp_path / "power.md"
    d = _run(["--mode", "power-table", "--config", "tiny", "--loop-s", "0.05", "--table", str(out)])
    assert d["mode"] == "power-table" and len(d["rows"]) > 10 and all(r["runs"] >= 30 and r["ms_per_iter"] > 0 for r in d["rows"])
    assert out.read_text().count("\n") == len(d["rows"]) + 2
