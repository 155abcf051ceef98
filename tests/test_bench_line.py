"""bench.py prints ONE short JSON line (the 20.5 KB line of that round did not reach the driver's record).
The line is built by bench.headline_line from the per-config result dicts; here it is fed dicts of the shape measure_config
returns, with the longest strings and widest numbers a real run produces, and must stay under 3 KB, be strict JSON (no NaN /
Infinity) and carry every key the bench contract names."""
import json
import math
import subprocess
import sys
import os
from types import SimpleNamespace

import bench

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _result(cfg, bad=False):
    roof = lambda kernel, unit: {"kernel": kernel, "bound": "alu", "achieved": 7.234567891234, "peak": 35.1612345678, "unit": unit,
                                 "frac": 0.20571234567, "frac_mufu": 0.156123456, "speedup_from_skipping": 16.4812345,
                                 "ops_per_sample": 20.0, "executed_samples": 16678123456, "ms": 46.1234567,
                                 "peak_source": "FP32 issue peak (FFMA), radt_pipe_peak in this run at 1965 MHz",
                                 "traffic": 2234567890.0}
    e2e = {"value": 4.0712345678e12, "unit": "samples/s", "h2d_bytes_per_step": 2153775104, "d2h_bytes_per_step": 6291464,
           "ms_per_step": 67.5123456, "steps": 5, "api": "radt_fit_step_host (pinned host buffers)"}
    return {"config": {"workload": "cfg5_batch16_axisym256x128_img512_c128_n512", "rays": 4194304, "channels": 128,
                       "steps_per_ray": 512, "grid": [256, 128, 1], "batch": 16, "nominal_samples_per_step": 274877906944,
                       "parallelism": "independent disks x1", "l2": "flushed between timed steps (256 MiB fill)"},
            "value": float("nan") if bad else 4.3012345678e12, "unit": "samples/s", "steps": 20, "warmup": 5,
            "ms_per_step": 63.9123456789, "fwd_value": 1.6e13, "fwd_ms": 17.2345678, "bwd_ms": 46.1234567,
            "roofline": roof("k_march_bwd (adjoint march + gradient unpack, setup reused from the forward)", "T FP32 lane-op/s"),
            "roofline_other": roof("k_march_fwd (includes the fused setup launch)", "T MUFU lane-op/s"),
            "e2e": e2e, "e2e_render": dict(e2e, unit="samples/s (forward only)"),
            "gpu_launches": 120, "launches_per_step": 6,
            "clocks": {"sm_mhz": 1965, "sm_max_mhz": 1965, "reasons": ["sw_power_cap", "sw_thermal_slowdown"], "samples": 64},
            "loss": float("inf") if bad else 0.93, "wall_s": 1.3,
            "cpu_baseline": {"value": 9.0812345e8, "unit": "samples/s", "cores": 16, "kind": "oracle",
                             "sample": "cfg5_batch16_axisym256x128_img512_c128_n512: 2 passes over every 11th row and column of "
                                       "all 16 item(s) (2.27e+09 samples), fp64 forward + adjoint, 12.5 s wall",
                             "value_1thread": 6.1e7}}


def test_headline_line_is_short_strict_json_with_the_contract_keys():
    configs = [1, 2, 3, 4, 5, 6]
    results = {c: _result(c) for c in configs}
    args = SimpleNamespace(steps=20, warmup=5)
    line = bench.headline_line(results[5], results, configs, 1, args)
    text = json.dumps(line, allow_nan=False, separators=(",", ":"))
    assert len(text) < bench.MAX_LINE_BYTES <= 3000
    d = json.loads(text)
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "clocks", "gpu_launches"):
        assert key in d, key
    assert set(("bound", "achieved", "peak", "unit", "frac", "traffic")) <= set(d["roofline"])
    assert set(("value", "unit", "cores", "kind", "sample")) <= set(d["cpu_baseline"])
    assert set(("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step")) <= set(d["e2e"])
    assert d["config"]["workload"].startswith("cfg5") and "model" not in d["config"]
    assert d["value"] > 0 and math.isclose(d["roofline"]["frac"], 0.205712, rel_tol=1e-5)
    assert d["per_config_ms"]["cfg3"][:3] == [63.9123, 17.2346, 46.1235]


def test_non_finite_numbers_never_reach_the_line():
    results = {5: _result(5, bad=True)}
    line = bench.headline_line(results[5], results, [5], 1, SimpleNamespace(steps=3, warmup=3))
    text = json.dumps(line, allow_nan=False)                     # raises on NaN / Infinity
    assert json.loads(text)["value"] is None


def test_dry_run_prints_one_short_line():
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--dry-run", "--steps", "2"], capture_output=True,
                         text=True, timeout=300, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = res.stdout.splitlines()
    assert len(lines) == 1 and len(lines[0]) < 3000
    assert json.loads(lines[0])["dry_run"] is True
