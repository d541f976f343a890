"""The gap reduction of libsettrace (include/set_trace.h) on hand-built timelines whose gaps, busy time and idle
fraction are known by construction.  No GPU and no CUPTI call: set_trace_reduce is host-only."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def trace(libset):
    from paper_2606_05495_b200 import trace as t
    t.load()
    return t


def test_trace_library_exports_every_declared_symbol(trace):
    text = open(os.path.join(ROOT, "include", "set_trace.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = sorted(set(re.findall(r"\b(set_trace_[a-z0-9_]+)\s*\(", text)))
    assert declared == ["set_trace_error", "set_trace_reduce", "set_trace_start", "set_trace_stop"]
    for name in declared:
        assert hasattr(trace.load(), name)
    assert C.sizeof(trace.GapSummary) == 40 and C.sizeof(trace.TraceStats) == 8 * 8 + 5 * 8 + 4 * 40 and C.sizeof(trace.TraceRec) == 32


def test_one_stream_two_jobs(trace):
    K, S, M, Z = trace.KIND_KERNEL, trace.KIND_SIGNAL, trace.KIND_MEMCPY, trace.KIND_MEMSET
    us = 1000
    # job 7: H2D [0,10] K [12,14] K [15,16] D2H [20,30] signal [31,32];  job 8 starts 5 us later with a memset
    recs = [(1, 7, M, 0, 10 * us), (1, 7, K, 12 * us, 14 * us), (1, 7, K, 15 * us, 16 * us), (1, 7, M, 20 * us, 30 * us),
            (1, 7, S, 31 * us, 32 * us),
            (1, 8, Z, 37 * us, 38 * us), (1, 8, M, 38 * us, 48 * us), (1, 8, K, 50 * us, 52 * us), (1, 8, K, 55 * us, 56 * us)]
    st = trace.reduce(reversed(recs))                       # order of arrival must not matter
    assert (st["kernels"], st["signal_kernels"], st["memcpys"], st["memsets"], st["streams"]) == (5, 1, 3, 1, 1)
    assert st["wall_us"] == 56.0
    assert st["busy_us"] == pytest.approx(10 + 2 + 1 + 10 + 1 + 1 + 10 + 2 + 1)
    assert st["idle_frac"] == pytest.approx(1 - 38 / 56, abs=1e-4)
    assert st["kernel_mean_us"] == pytest.approx((2 + 1 + 2 + 1) / 4)
    kk = st["kernel_kernel"]                                # K->K with nothing between: 14->15 and 52->55
    assert (kk["count"], kk["mean_us"], kk["max_us"]) == (2, 2.0, 3.0)
    assert st["inter_job"] == {"count": 1, "mean_us": 5.0, "p50_us": 5.0, "p99_us": 5.0, "max_us": 5.0}
    intra = st["intra_job"]                                 # 2,1,4,1 in job 7; 0,2,3 in job 8
    assert intra["count"] == 7 and intra["mean_us"] == pytest.approx(13 / 7, abs=1e-3) and intra["max_us"] == 4.0
    assert st["any_op"]["count"] == 8


def test_streams_are_separate_and_overlap_counts_once(trace):
    K = trace.KIND_KERNEL
    # stream 1: [0,10] [20,30]; stream 2: [5,25]  -> union [0,30] is fully busy, yet stream 1 has a 10 us gap
    st = trace.reduce([(1, 1, K, 0, 10_000), (1, 2, K, 20_000, 30_000), (2, 3, K, 5_000, 25_000)])
    assert st["streams"] == 2 and st["busy_us"] == 30.0 and st["idle_frac"] == 0.0 and st["sum_op_us"] == 40.0
    assert st["kernel_kernel"]["count"] == 0               # the two kernels of stream 1 belong to different jobs
    assert st["inter_job"]["count"] == 1 and st["inter_job"]["mean_us"] == 10.0 and st["intra_job"]["count"] == 0


def test_overlapping_ops_on_one_stream_give_zero_gap_and_empty_input(trace):
    K, M = trace.KIND_KERNEL, trace.KIND_MEMCPY
    st = trace.reduce([(1, 1, M, 0, 10_000), (1, 1, K, 8_000, 12_000)])
    assert st["any_op"]["max_us"] == 0.0 and st["busy_us"] == 12.0
    st = trace.reduce([])
    assert st["kernels"] == 0 and st["wall_us"] == 0.0


def test_percentiles(trace):
    K = trace.KIND_KERNEL
    recs, t = [], 0
    for i in range(101):                                    # gaps 0,1,...,99 us between 1 us kernels
        recs.append((3, 9, K, t, t + 1000))               # one job: kernel->kernel gaps are counted inside a job only
        t += 1000 + i * 1000
    kk = trace.reduce(recs)["kernel_kernel"]
    assert kk["count"] == 100 and kk["p50_us"] == 50.0 and kk["p99_us"] == 98.0 and kk["max_us"] == 99.0 and kk["mean_us"] == 49.5


def test_jobs_are_grouped_by_launch_not_by_cupti_stream_id(trace):
    """CUPTI labels the parallel branches of a job graph with stream ids of their own (round 1 saw 200 'streams' on an
    8-stream context): jobs are rebuilt from the correlation id, the work stream is the id most of a job's kernels ran
    under, and a PDL overlap shows as a NEGATIVE kernel-to-kernel gap."""
    K, S, M, Z = trace.KIND_KERNEL, trace.KIND_SIGNAL, trace.KIND_MEMCPY, trace.KIND_MEMSET
    us = 1000
    recs = [  # job 1 on work stream 7: memset on an internal id 901 beside the H2D on 7; kernels on 7; second D2H leaf on 902
        (901, 1, Z, 0, 1 * us), (7, 1, M, 0, 10 * us), (7, 1, K, 11 * us, 14 * us), (7, 1, K, 13 * us, 16 * us), (7, 1, K, 18 * us, 19 * us),
        (7, 1, M, 20 * us, 30 * us), (902, 1, M, 20 * us, 22 * us), (7, 1, S, 31 * us, 32 * us),
        # job 2 on the same work stream, 4 us after job 1's last op; its memset again on another internal id
        (903, 2, Z, 36 * us, 37 * us), (7, 2, M, 36 * us, 46 * us), (7, 2, K, 47 * us, 49 * us), (7, 2, S, 50 * us, 51 * us),
        # job 3 on work stream 8, overlapping both
        (8, 3, M, 5 * us, 15 * us), (8, 3, K, 16 * us, 40 * us), (8, 3, S, 41 * us, 42 * us)]
    st = trace.reduce(recs)
    assert st["jobs"] == 3 and st["streams"] == 2                      # not 5
    kk = st["kernel_kernel"]                                           # job 1: 13 - 14 = -1 (PDL overlap), 18 - 16 = +2
    assert kk["count"] == 2 and st["kernel_kernel_overlapped"] == 1 and kk["mean_us"] == 0.5 and kk["max_us"] == 2.0
    assert st["inter_job"] == {"count": 1, "mean_us": 4.0, "p50_us": 4.0, "p99_us": 4.0, "max_us": 4.0}    # 36 - 32 on work stream 7
    # intra-job gaps never count a parallel branch as idle time: job 1 has 1 (10->11), 2 (16->18), 1, 1 and zeros
    assert st["intra_job"]["max_us"] == 2.0
