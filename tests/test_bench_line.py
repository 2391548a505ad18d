"""bench.py's headline: ONE line of strict JSON under 2000 bytes, whatever strings the run produced.

Round 2 lost its driver record to a 21 KB line (the driver keeps ~3 KB of stdout and parses the last line), so the line
builder is tested on worst-case content here, without a GPU.
"""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import bench  # noqa: E402


def _full(long):
    roof = {"bound": "tensor", "achieved": 2073.123456789, "peak": 3185.2, "unit": "TOPS", "frac": 0.650123456, "traffic": 4005750000.0,
            "traffic_source": "profiles/r2b_ncu_final.md (ncu capture)" + long, "kernel": "xtc::xengine_pair_kernel<1>",
            "kernel_ms": 1.0651234567, "exec_over_useful": 1.2451361867, "hbm_write_peak_gbs": 4234.56789,
            "tensor": {"frac_of_nominal": 0.4606941, "frac_on_executed_ops": 0.8101234}, "hbm": {"frac": 0.57891234},
            "peak_source": long, "roof_ms": {"tensor": 0.693, "hbm": 0.615}}
    return {
        "metric": bench.METRIC, "value": 2073.123456789, "unit": bench.UNIT, "n_gpus": 1, "steps": 20, "warmup": 5,
        "ms_per_step": 4.26049382716, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "s8 x s8 -> s32", "data": "synthetic",
        "config": {"workload": bench.describe(bench.workload("cfg4")) + long, "l2": "inputs (8192 MiB per step) larger than L2" + long,
                   "parallelism": "replicas only (x1)" + long, "visibilities_per_s": 1.2345e11, "input_sha256": ["f" * 64] * 4},
        "clocks": {"sm_mhz": 1207.5, "sm_max_mhz": 1965.0, "power_w_max": 1003.39, "samples": 17,
                   "reasons": ["hw_slowdown", "hw_thermal_slowdown", "sw_power_cap", "sw_thermal_slowdown"]},
        "e2e": {"value": 55.123456789, "unit": bench.UNIT, "h2d_bytes_per_step": 8589934592, "d2h_bytes_per_step": 1077936128,
                "steps": 5, "ms_per_step": 160.123456789, "how": long},
        "gpu_launches": 80, "roofline": roof,
        "sustained": {"steps": 517, "seconds": 2.2, "ms_per_step": 4.9, "value": 1790.123456, "unit": bench.UNIT,
                      "clocks": {"sm_mhz": 1147.5, "reasons": ["sw_power_cap"]}, "roofline": dict(roof, frac=0.6598765)},
        "cpu_baseline": {"value": 0.107149805, "unit": bench.UNIT, "cores": 16, "kind": "oracle", "sample": "channels 0..15 of call 0" + long,
                         "threads_1": {"value": 0.0071234567}, "cpu_model": "Intel(R) Xeon(R) Platinum 8570" + long, "compiler": long},
    }


def _others(long):
    names = ["cfg1", "cfg2", "cfg3"] + ["cfg5_n%d" % n for n in (32, 64, 128, 256, 512, 1024)] + ["cross_n256"]
    recs = [{"workload": bench.describe(bench.workload(n)) + long, "value": 852.512345, "unit": bench.UNIT, "input_sha256": ["a" * 64],
             "roofline": {"frac": 0.5412345, "bound": "hbm"}} for n in names]
    recs.append({"workload": "dumps: N=256, 2 pol" + long, "value": 352.19333, "hbm": {"frac": 0.4712345}})
    recs.append({"metric": "corner_turn_gbs", "value": 5386.123, "config": {"workload": long}, "roofline": {"frac": 0.82, "bound": "hbm"}})
    recs.append({"metric": "fengine_gbs", "value": 5543.2, "config": {"workload": "F-engine: -> 128 complex fp16"}, "roofline": {"frac": 0.85, "bound": "hbm"}})
    recs.append({"metric": "fengine_gbs", "value": 3394.2, "config": {"workload": "F-engine: -> int8 (requantised, scale 1/20)"},
                 "roofline": {"frac": 0.52, "bound": "hbm"}})
    recs.append({"error": "RuntimeError('" + long + "')"})
    return recs


def test_headline_fits_and_round_trips():
    for long in ("", " lorem ipsum" * 400):
        text = bench.compact_headline(_full(long), _others(long))
        assert "\n" not in text
        assert len(text.encode()) < bench.HEADLINE_MAX_BYTES, len(text.encode())
        line = json.loads(text, parse_constant=lambda c: (_ for _ in ()).throw(ValueError(c)))      # strict: no NaN / Infinity
        for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "dtype",
                    "data", "gpu_launches", "config", "clocks", "e2e", "roofline", "cpu_baseline"):
            assert key in line, key
        assert line["value"] > 0 and line["roofline"]["frac"] > 0 and line["cpu_baseline"]["value"] > 0
        assert set(line["e2e"]) >= {"value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"}
        assert set(line["roofline"]) >= {"bound", "achieved", "peak", "unit", "frac", "traffic"}
        assert line["config"]["workload"] is None or line["config"]["workload"].startswith("cfg4")


def test_headline_normal_case_keeps_everything():
    line = json.loads(bench.compact_headline(_full(""), _others("")))
    assert line["workloads"]["cfg3"] == [852.5, 0.541, "hbm"]
    assert set(line["workloads"]) >= {"cfg1", "cfg2", "cfg3", "cfg5_n1024", "cross_n256", "dumps", "corner_turn", "fengine_f16", "fengine_ci8"}
    assert line["sustained"]["frac"] == 0.66 and line["roofline"]["exec_over_useful"] == 1.245
    assert line["roofline"]["frac_on_executed_ops"] == 0.81


def test_headline_survives_missing_legs_and_nan():
    full = _full("")
    full.update(e2e=None, sustained=None, cpu_baseline=None, clocks=None)
    full["roofline"]["traffic"] = float("nan")
    line = json.loads(bench.compact_headline(full, None))
    assert line["e2e"] is None and line["workloads"] is None and line["roofline"]["traffic"] is None
