"""bench.py's last stdout line must stay small enough for the driver to parse (round 2's grew to 23 KB and was
recorded as `parsed: null`): the formatter is run on a canned record with every key at a realistic size."""
import argparse
import json
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import bench  # noqa: E402
from paper_2603_29785_b200 import inputs  # noqa: E402


def canned():
    args = argparse.Namespace(workload="cfg4", overlap=1.0)
    cfg = inputs.CONFIGS["cfg4"]
    return {
        "metric": bench.METRIC, "value": 9572345678.123456, "unit": bench.UNIT, "n_gpus": 1, "steps": 20, "warmup": 5,
        "ms_per_step": 1.7527123456, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic", "config": bench.workload_config(args, cfg, cfg["batch"], None),
        "clocks": {"sm_mhz": 1965, "sm_max_mhz": 1965, "reasons": ["sw_power_cap"], "samples": 37,
                   "sm_mhz_min": 1920, "source": "nvml"},
        "e2e": {"value": 7123456789.0123, "unit": bench.UNIT, "h2d_bytes_per_step": 67108864,
                "d2h_bytes_per_step": 67108864, "ms_per_step": 2.3512345678, "chunks": 2,
                "equals_device_resident_result": True},
        "gpu_launches": 340,
        "roofline": {"bound": "hbm", "kernel": "rows_split16_inv", "achieved": 1845.123456789, "peak": 6546.2,
                     "unit": "GB/s", "frac": 0.281861234, "traffic": 668512345.0,
                     "traffic_source": "profiles/r3_dram_traffic.csv (ncu --set full, csrc 0123456789abcdef)",
                     "algo_bytes_per_launch": 436207616.0, "design_bytes_per_launch": 546123456.0,
                     "peak_source": "measured (MEASURED_PEAKS.json hbm_gbs)", "avg_launch_ms": 0.23651234,
                     "share_of_step": 0.3871234},
        "path": {"compulsory_bytes_per_step": 2933456789, "achieved_gbs": 1674.123456, "frac_of_peak": 0.25571234,
                 "ms_per_step_cuda_graph": 1.7012345},
        "round_trip_err": 6.9123456e-07,
        "cpu_baseline": {"value": 2061234.5678, "unit": bench.UNIT, "cores": 16, "kind": "oracle",
                         "sample": "24 segments of the same workload, one pass (12.2 s), oracle FFT engine fp64"},
        "csrc_hash": "9e339b9c3b4d03ab", "detail": "gpurun_out/bench_detail.json",
    }


def test_headline_is_one_short_parseable_line():
    text = bench.headline_json(canned())
    assert "\n" not in text and len(text) < bench.HEADLINE_LIMIT == 2048
    back = json.loads(text)
    assert back["value"] > 0 and back["roofline"]["frac"] > 0 and back["e2e"]["value"] > 0
    assert back["cpu_baseline"]["kind"] == "oracle" and back["config"]["baseline_config_index"] == 3
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert key in back
    # the tables belong in the detail file, not here
    for key in ("kernels", "configs", "largest_batch", "cufft_side_by_side"):
        assert key not in back


def test_headline_refuses_to_grow():
    rec = canned()
    rec["kernels"] = [{"name": f"k{i}", "avg_ms": 0.1 * i, "share": 0.01} for i in range(200)]
    with pytest.raises(ValueError):
        bench.headline_json(rec)


def test_detail_file_round_trips(tmp_path):
    where = bench.write_detail(str(tmp_path / "sub" / "detail.json"), {"kernels": [1, 2, 3], "configs": {"cfg2": {}}})
    assert json.load(open(os.path.join(bench.ROOT, where)))["kernels"] == [1, 2, 3]
