"""-m "not gpu": bench.py's final stdout line stays small enough for the driver's capture (round 2's 20 KB line was cut in the
middle and parsed as nothing) and still carries every key of the contract; everything else lands in the extras."""
import json

import bench


def canned():
    big_rows = [{"batch_jets": 2 ** i, "ms_p50": 0.1234567 * i, "ms_p99": 0.2 * i, "jets_per_s": 1e6 * i, "frac_of_bf16_peak": 0.4}
                for i in range(12)]
    return {
        "metric": bench.METRIC, "value": 3058391.123456, "unit": bench.UNIT, "n_gpus": 1, "steps": 200, "warmup": 20,
        "ms_per_step": 0.33481789, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
        "data": "synthetic",
        "config": {"workload": bench.WORKLOAD, "batch_jets": 1024, "particles_per_batch": [40851, 40857, 40863, 40920],
                   "entry": "gnn_infer (ragged, device-resident)", "precision": "bf16", "parallelism": "1 GPU",
                   "l2": "flushed between steps (256 MiB memset outside the per-step CUDA events); 4 batches rotate"},
        "roofline": {"bound": "tensor", "kernel": "edge_kernel<256> (stage edgeconv2: EdgeConv block 3, per-edge layers 2-3)",
                     "achieved": 1094.123456789, "peak": 1665.7, "unit": "TFLOP/s", "frac": 0.65712345, "traffic": 69621248,
                     "traffic_source": "profiles/r02_traffic.json (earlier ncu capture, not this run)",
                     "peak_source": "measured (MEASURED_PEAKS.json), burst cuBLAS bf16", "flops_per_launch": 171.3e9,
                     "flops_per_launch_block_min": 1.8e11, "flops_per_launch_block_stated": 2.6e11, "ms_per_launch": 0.1566,
                     "forwards_averaged": 200},
        "forward": {"flops_min": 235.2e9, "flops_stated": 3.4e11, "achieved_tflops": 702.4, "frac_of_bf16_peak": 0.4217,
                    "t_roof_us": 141.2},
        "stages_ms": {"ingest": 0.0116, "knn0": 0.0196, "edgeconv0": 0.0368, "knn1": 0.0277, "edgeconv1": 0.0633,
                      "knn2": 0.0381, "edgeconv2": 0.1566, "pool_head": 0.0179},
        "stages_pass": {"ms_per_step": 0.37, "note": "x" * 200},
        "gpu_launches": 2200, "wall_s_timed_region": 0.4,
        "two_in_flight": {"value": 3.4e6, "unit": bench.UNIT, "ms_per_step": 0.3, "entry": "y" * 150},
        "e2e": {"value": 2.57e6, "unit": bench.UNIT, "h2d_bytes_per_step": 1474796, "d2h_bytes_per_step": 8192,
                "entry": "gnn_infer_host: one blocking call per step from pinned host buffers (H2D + forward + D2H + sync), wall clock",
                "ms_per_step": 0.398, "pipelined": {"value": 3.32e6, "ms_per_step": 0.308,
                                                    "entry": "gnn_infer_host_begin / _end, two slices on two streams in flight"}},
        "latency_b16": {"p50_us": 58.8, "p99_us": 63.1, "iterations": 1000, "entry": "gnn_infer, 16 jets device-resident, CUDA events"},
        "serving": {"value": 1.08e6, "rows": big_rows}, "ragged_4096_f9": {"value": 3.1e6}, "perf_sweep": {"rows": big_rows * 2},
        "colocation": {"rows": big_rows}, "autoscale": {"scale_up_times_s": list(range(40))}, "sweep": {"particlenet": big_rows, "wide": big_rows},
        "clocks": {"sm_mhz": 1965.0, "sm_max_mhz": 1965, "reasons": [], "samples": 310},
        "cpu_baseline": {"value": 172.5, "unit": bench.UNIT, "cores": 16, "kind": "oracle",
                         "sample": "first 2070 jets of batch 0 (82731 particles), one oracle.forward call, 12.0 s",
                         "one_thread": {"value": 11.9, "sample": "first 36 jets, nthreads=1, 3.0 s"}},
        "bdt": {"rows": big_rows}, "fig4": {"cumulative_wall_ms": list(range(10))},
    }


def test_final_line_is_small_complete_and_round_trips():
    out = canned()
    line, extras = bench.split_line(out)
    text = json.dumps(line, separators=(",", ":"))
    assert len(text) < 4096
    back = json.loads(text)
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "clocks", "gpu_launches", "forward", "latency_b16"):
        assert k in back, k
    assert set(("bound", "achieved", "peak", "unit", "frac", "traffic")) <= set(back["roofline"])
    assert set(("value", "unit", "cores", "kind", "sample")) <= set(back["cpu_baseline"])
    assert set(("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step")) <= set(back["e2e"])
    assert back["config"]["workload"] == bench.WORKLOAD and "model" not in back["config"]
    assert abs(back["value"] - out["value"]) / out["value"] < 1e-5            # six significant digits survive
    assert back["roofline"]["frac"] == float("%.6g" % out["roofline"]["frac"])
    # nothing measured is lost: every key dropped from the line is in the extras, in full
    for k in ("stages_ms", "serving", "sweep", "perf_sweep", "colocation", "autoscale", "bdt", "fig4", "two_in_flight", "ragged_4096_f9"):
        assert k not in back and extras[k] == out[k]
    assert extras["config"]["particles_per_batch"] == out["config"]["particles_per_batch"]
    assert extras["roofline"]["forwards_averaged"] == 200


def test_reference_arm_line_is_small():
    """--impl reference prints its own line; it has no extras and is far below the limit by construction."""
    line = {"impl": "reference", "metric": bench.METRIC, "value": 170.0, "unit": bench.UNIT, "config": {"workload": bench.WORKLOAD, "sample": "s" * 80}}
    assert len(json.dumps(line)) < 1024
