"""Host-side arithmetic of bench.py: the algorithmic bytes / flops per launch it divides by (DESIGN.md section 6 table,
SURVEY.md 8(d)) and the pipeline roofline (slowest of link, HBM, flops).  No GPU."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402
from paper_2606_05495_b200.workloads import baseline_workload  # noqa: E402


def test_algorithmic_work_per_launch_matches_the_design_table():
    alg = {c: bench.stage_algorithmic(baseline_workload(c), (1280, 720, 1, 1)) for c in range(5)}
    assert alg[0] == [("scan_i32", "hbm", 32768), ("hist_mod64", "hbm", 16640)]
    assert [w for _, _, w in alg[1]] == [131072, 196608, 131072, 131072, 65540]
    assert len(alg[2]) == 10 and set(alg[2]) == {("jacobi5_f32", "hbm", 134217728)}       # read + write of a 64 MiB grid
    assert alg[3] == [("gemm_bias_gelu_bf16", "tensor", 2 * 2048 ** 3)]
    px = 1280 * 720
    assert [w for _, _, w in alg[4]] == [4 * px, 2 * px, px + 1024]
    # per job totals of SURVEY.md 8(d): config 1 = 655,364 bytes, config 4 = 7 bytes per pixel + 1024
    assert sum(w for _, _, w in alg[1]) == 655364
    assert sum(w for _, _, w in alg[4]) == 7 * px + 1024


def test_pipeline_roofline_picks_the_slowest_bound():
    link = {"duplex": {"h2d_gbs": 50.0, "d2h_gbs": 50.0}}
    pk = {"hbm_gbs": 6542.7, "bf16_tflops_sustained": 1402.6}
    wl = baseline_workload(1)
    r = bench.pipeline_roofline(wl, 131072, 4, link, pk, (1, 1, 1, 1))
    assert r["e2e_bound_by"] == "link"
    assert abs(r["t_link_us"] - 131072 / 50e3) < 1e-3                                      # 2.62 us of wire time per job
    assert abs(r["e2e_bound_jobs_per_s"] - 1e6 / (131072 / 50e3)) < 1.0
    assert abs(r["t_hbm_us"] - 655364 / 6542.7e3) < 1e-3
    # config 3: link 16.8 MB in / 8.4 MB out, 17.18 GFLOP
    wl3 = baseline_workload(3)
    r3 = bench.pipeline_roofline(wl3, 16785408, 8388608, link, pk, (1, 1, 1, 1))
    assert r3["e2e_bound_by"] == "link" and abs(r3["t_flop_us"] - 2 * 2048 ** 3 / 1402.6e6) < 1e-2
    assert r3["device_bound_jobs_per_s"] <= 1e6 / (2 * 2048 ** 3 / 1402.6e6) + 1.0
    # with a very fast link the GEMM becomes tensor-bound
    fast = {"duplex": {"h2d_gbs": 1e5, "d2h_gbs": 1e5}}
    assert bench.pipeline_roofline(wl3, 16785408, 8388608, fast, pk, (1, 1, 1, 1))["e2e_bound_by"] == "tensor"


def _fake_arm(jps, io):
    return {"jobs": 10000, "ms_per_step": 1e7 / jps, "jobs_per_s": jps, "in_bytes": 1310720000, "out_bytes": 40000,
            "h2d_bytes": 0 if io == "device" else 1310720000, "d2h_bytes": 0 if io == "device" else 40000, "kernel_launches": 2000000, "mismatches": 0,
            "host_us_per_job": {"submit": 1.91234567, "bind": 1.01234, "launch": 2.2345678, "callback": 0.2123456, "sync": 0.0},
            "stats": {"cuda_streams": 16}, "step_ms": [1.0] * 20}


def test_stdout_line_is_compact_and_complete():
    """the driver keeps only the tail of stdout, so the one JSON line must stay small (< 2 KB aimed, 4 KB hard)
    and carry every key the contract and the tier ask for; everything else lives in the detail file."""
    import json
    wl = baseline_workload(1)
    pk = {"hbm_gbs": 6541.8, "bf16_tflops": 1604.2, "bf16_tflops_sustained": 1375.2, "source": "measured (MEASURED_PEAKS.json)"}
    krow = {"kernel": "block_sum_f32", "bound": "hbm", "avg_us": 1.843, "algorithmic": 65540, "achieved": 35.56, "peak": 6541.8, "unit": "GB/s",
            "frac": 0.0054, "launches_per_job": 1, "total_us": 1.843, "traffic": 12345.0, "launch_floor_us": 0.942}
    gaps = {"jobs": 30000, "gaps": 29000, "gap_mean_us": 14.71234, "gap_p50_us": 12.0, "gap_p99_us": 39.12345, "gap_max_us": 200.0, "job_mean_us": 24.0,
            "span_us": 46000.0, "stream_busy_frac": 0.63, "busy_union_us": 45800.0, "idle_frac": 0.004, "overhead_frac": 0.0312345, "jobs_per_s": 191000.0}
    side = {"workload": "x" * 60, "e2e": 812.3, "value": 4000.1, "speedup_vs_batch_sync_e2e": 1.031, "pipeline_roofline": {"e2e_frac": 0.9412},
            "kernels": [{"kernel": "jacobi5_f32", "frac": 0.9351, "avg_us": 21.932, "bound": "hbm"}], "cpu_baseline": {"value": 1.0}}
    detail = {"kernels": [krow, dict(krow, kernel="affine_f32", total_us=1.1)], "streams_per_lane": 2,
              "baselines": {"batch_sync_graphs_e2e": {"jobs_per_s": 193000.0, "host_us_per_job": _fake_arm(1, "host")["host_us_per_job"]}},
              "device_gaps": {"how": "...", "config1": {"set_e2e": gaps, "batch_sync_graphs_e2e": dict(gaps, gap_mean_us=22.1), "mutex_queue_e2e": gaps}},
              "pipeline_roofline": {"e2e_bound_by": "link", "e2e_bound_jobs_per_s": 380868.2, "e2e_frac": 0.5703},
              "workloads": {f"config{c}": dict(side) for c in (0, 2, 3, 4, 5, 6)},
              "cpu_baseline": {"value": 9943.12, "unit": "jobs/s", "cores": 1, "kind": "oracle",
                               "sample": "99431 jobs of the workload (first 2048 job inputs, repeated) in 10.0 s, single thread, oracle/*.c -O2",
                               "all_cores": {"value": 43460.0, "cores": 16, "sample": "s" * 40}},
              "side_mismatches": 0}
    detail["workloads"]["config3"]["kernels"] = [{"kernel": "gemm_bias_gelu_bf16", "frac": 0.7123, "avg_us": 15.01, "bound": "tensor"}]
    clocks = {"sm_mhz": 1965.0, "sm_max_mhz": 1965.0, "reasons": ["sw_power_cap"], "samples": 12}
    line = bench.compact_line(wl, 1, 20, 5, 10000, 24.8, 402503.2, 46.0, 217224.4, _fake_arm(402503.2, "device"), _fake_arm(217224.4, "host"),
                              clocks, detail, "/x/bench_detail.json", pk)
    s = json.dumps(line, separators=(",", ":"))
    back = json.loads(s)
    for k in bench.REQUIRED_KEYS:
        assert k in back, k
    assert len(s) < 2048, len(s)
    assert back["e2e"]["value"] == 217224.4 and back["e2e"]["h2d_bytes_per_step"] == 1310720000 and back["value"] == 402503.2
    assert back["roofline"]["kernel"] == "block_sum_f32" and back["roofline"]["frac"] == 0.0054 and back["roofline"]["traffic"] == 12345.0
    assert back["cpu_baseline"]["kind"] == "oracle" and back["cpu_baseline"]["cores"] == 1
    hm = back["headline_metrics"]
    assert hm["set_over_batch_sync_e2e"] == round(217224.4 / 193000.0, 3)
    assert hm["sched_overhead_frac"] == {"set": 0.0312, "batch_sync": 0.0312} and hm["gap_between_jobs_us"]["batch_sync"] == 22.1
    assert back["kernel_rooflines"]["jacobi5_f32"]["frac"] == 0.9351 and back["kernel_rooflines"]["gemm_bias_gelu_bf16"]["frac"] == 0.7123
    side_line = back["workloads_e2e_frac_vsbatch"]
    assert set(side_line) == {"config0", "config2", "config3", "config4", "config5", "config6"} and side_line["config2"] == [812.3, 0.9412, 1.031]
    assert back["detail"] == "bench_detail.json"
    # side workloads that failed put a short error each on the line: it stays under 2 KB
    detail_err = dict(detail, workloads={f"config{c}": {"error": "e" * 300} for c in (0, 2, 3, 4, 5, 6)})
    line_err = bench.compact_line(wl, 1, 20, 5, 10000, 24.8, 402503.2, 46.0, 217224.4, _fake_arm(402503.2, "device"), _fake_arm(217224.4, "host"),
                                  clocks, detail_err, "/x/bench_detail.json", pk)
    assert len(json.dumps(line_err, separators=(",", ":"))) < 2048
    assert line_err["workloads_e2e_frac_vsbatch"]["config5"].startswith("error: ")
    # world > 1: no side passes ran, the line is still complete
    line2 = bench.compact_line(wl, 8, 20, 5, 10000, 24.8, 3.2e6, 46.0, 1.7e6, _fake_arm(402503.2, "device"), _fake_arm(217224.4, "host"),
                               clocks, {}, None, pk)
    assert line2["n_gpus"] == 8 and line2["e2e"]["h2d_bytes_per_step"] == 8 * 1310720000 and line2["roofline"] is None


def test_merge_gap_stats_weights_by_jobs():
    a = {"jobs": 100, "gaps": 90, "gap_mean_us": 10.0, "gap_p50_us": 9.0, "gap_p99_us": 30.0, "gap_max_us": 50.0, "job_mean_us": 20.0,
         "span_us": 1000.0, "stream_busy_frac": 0.5, "busy_union_us": 900.0, "idle_frac": 0.1, "overhead_frac": 0.2}
    b = dict(a, jobs=300, gaps=290, gap_mean_us=20.0, gap_p99_us=40.0, gap_max_us=45.0, overhead_frac=0.4)
    m = bench.merge_gap_stats([a, b])
    assert m["jobs"] == 400 and m["gaps"] == 380 and m["gap_mean_us"] == 17.5 and m["gap_p99_us"] == 40.0 and m["gap_max_us"] == 50.0
    assert m["overhead_frac"] == 0.35 and m["span_us"] == 2000.0 and m["busy_union_us"] == 1800.0
