"""bench.py's stdout contract: ONE line, strict JSON, small enough to survive a reader that keeps only the last 3 kB of
stdout, carrying every key the driver checks.  Round 2's line (~28 kB, five full per-config documents inside it) could not
be parsed by the driver; everything beyond the contract now goes to the --detail file.  CPU only: contract_line is fed a
canned measure_config result (the shape bench.py produces, values from a real cb-ar run)."""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench      # noqa: E402
import ra_inputs  # noqa: E402

REQUIRED = ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
            "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "clocks", "gpu_launches")


def canned(cfg, compute_bound=True, nan=False):
    setting = {"smem_reserve_bytes": 65536, "sm_budget": 148, "tiles_per_cta": 0, "priority": "on", "coll_sm_budget": 32,
               "coll_smem_bytes": 0, "coll_variant": 0, "coll_ctas_per_sm": 0, "use_graph": 0, "l2_persist_bytes": 0}
    alone = {"gemm_ms": 0.68, "coll_ms": 0.17, "gemm_tflops": 1349.1234567, "gemm_tflops_burst": 1691.8479234160661,
             "gemm_frac_of_bf16_peak_burst": 1.0096967793125247, "gemm_frac_of_bf16_peak_sustained": 0.9632040069053964,
             "gemm_gbs": 548.1359223565202, "gemm_frac_of_hbm_peak": 0.08497440894746537, "coll_gbs": 6100.123456,
             "coll_frac_of_hbm_peak": 0.9327, "library_gemm_same_box": {"burst_tflops": 1656.0, "sustained_tflops": 1390.0},
             "gemm_plan": {"grid": 148, "stages": 4}}
    return {
        "workload": cfg.name, "gemm": [cfg.M, cfg.N, cfg.K], "collective": cfg.coll, "P": cfg.P, "n_iters_per_step": 20, "steps": 20,
        "ms_per_step": 17.436712, "value": 1147.0165432, "overlap_ms_per_iter": 0.8718356, "serial_ms_per_iter": 0.9612345,
        "sweep_serial_ms_per_iter": 0.97, "time_ratio_same": 0.907, "time_ratio_best": 1.0257,
        "norm_time_priority": float("nan") if nan else 1.0058016200047752, "overlap_rate": 0.93,
        "gemm_in_step_ms": 0.815659019947052, "coll_in_step_ms": 0.21, "instrumented_ms_per_iter": 0.88, "alone": alone,
        "combined_roofline_ms": {"burst": 0.6561897993411315, "sustained": 0.7856460362815291},
        "overlap_vs_roofline": {"burst": 1.3285378140468624, "sustained": 1.1096256091898926},
        "best_setting": setting, "plan": {"grid": 148, "stages": 4, "tile_m": 512, "tile_n": 256}, "sweep": "quick",
        "policy": {"setting": setting, "final": {"settings": [setting] * 4, "ms_per_iter": [0.87] * 4}, "settings_in_sweep": 67},
        "clocks": {"sm_mhz": 1305.0, "sm_max_mhz": 1965.0, "reasons": ["sw_power_cap"], "samples": 12, "power_w_max": 608.73},
        "gemm_max_ctas_on_one_sm": 1, "wall_ms_timed_region": 353.7236349999944, "gpu_launches": 800, "compute_bound": compute_bound,
        "residency": {"gemm_sms": 148, "coll_sms": 32, "big": list(range(400))},
        "e2e": {"value": 1155.5276988640796, "unit": "iter/s", "h2d_bytes_per_step": 805306368, "d2h_bytes_per_step": 201326592,
                "api": "ra_overlap_run_host " + "x" * 200, "gpu_ms_per_step": 17.3},
    }


def _line(nan=False, compute_bound=True):
    cfgs = {c.name: c for c in ra_inputs.CONFIGS[:5]}
    cfg = cfgs["cb-ar" if compute_bound else "mb-ar"]
    per = {n: canned(c, compute_bound=c.name.startswith("cb")) for n, c in cfgs.items() if n != cfg.name}
    peaks = {"hbm_gbs": 6540.2, "bf16_tflops": 1675.6, "bf16_tflops_sustained": 1399.5, "source": "measured"}
    cpu = {"value": 0.0273, "unit": "iter/s", "cores": 16, "kind": "oracle", "sample": "full: oracle.gemm over all C entries " * 10,
           "seconds_per_iter": 36.6, "timed": "full"}
    line, detail = bench.contract_line(cfg, canned(cfg, compute_bound, nan), per, peaks, cpu, 1, 20, 5, "quick",
                                       total_bench_s=101.6, detail_path="gpurun_out/bench_detail.json")
    return bench.dumps_line(line), detail


def _strict_loads(s):
    def bad(c):
        raise ValueError("non-finite constant " + c)
    return json.loads(s, parse_constant=bad)


def test_contract_line_is_small_strict_json_with_every_key():
    for cb in (True, False):
        s, detail = _line(compute_bound=cb)
        assert "\n" not in s and s.startswith("{") and len(s.encode()) < 3000, len(s)
        d = _strict_loads(s)
        for k in REQUIRED:
            assert k in d, k
        assert d["value"] > 0 and d["higher_is_better"] is True and d["vs_baseline"] is None and d["dtype"] == "bf16"
        r = d["roofline"]
        assert r["bound"] == ("tensor" if cb else "hbm") and r["unit"] == ("TFLOP/s" if cb else "GB/s")
        assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-4 and "traffic" in r
        assert set(d["cpu_baseline"]) == {"value", "unit", "cores", "kind", "sample"} and d["cpu_baseline"]["kind"] == "oracle"
        assert d["e2e"]["value"] > 0 and d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0
        assert {"sm_mhz", "sm_max_mhz", "reasons"} <= set(d["clocks"])
        assert d["config"]["workload"] == ("cb-ar" if cb else "mb-ar") and "model" not in d["config"]
        assert sum(k.startswith("cfg.") for k in d["config"]) == 5            # one short string per BASELINE config
        assert all(len(v) <= 400 for k, v in d["config"].items() if k.startswith("cfg."))
        # the long material is in the detail document, not in the line
        assert set(detail["per_config"]) == set(c.name for c in ra_inputs.CONFIGS[:5]) - {d["config"]["workload"]}
        assert "policy" in detail["headline"] and "residency" in detail["headline"] and "peaks" in detail
        json.dumps(bench._finite(detail), allow_nan=False)


def test_contract_line_never_prints_nan():
    s, _ = _line(nan=True)
    d = _strict_loads(s)
    assert d["norm_time_priority"] is None
