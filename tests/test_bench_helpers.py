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
