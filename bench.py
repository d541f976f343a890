#!/usr/bin/env python
"""bench.py -- jobs/s of the SET hot path on B200 (BASELINE.json metric).  The LAST line of stdout is one compact JSON
object (< 2 KB: the contract keys plus roofline, cpu_baseline, e2e, headline_metrics and one scalar per side workload);
everything else -- per-arm statistics, per-kernel tables, baselines, gaps, sweeps -- goes to a detail file (--out, default
bench_detail.json beside this script) and, as progress lines, to stderr.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--suite headline|default|all] [--sweep]
                    [--impl reference] [--out FILE]

A *step* is one pass of the whole hot path over one batch of synthetic input: every job of the workload
(BASELINE.json:configs[C], default C = 1: 10,000 jobs of the short-lived-kernel pipeline, 8 streams, 32 in
flight) goes through set_submit -> SET dispatch -> graph launch (H2D, stage kernels, D2H) -> callback, then
set_drain.  `value` is measured with the jobs' inputs/outputs already resident in HBM (SET_IO_DEVICE: the copy
nodes are D2D); `e2e` is the same call sequence with pinned HOST buffers, so every job's H2D and D2H copies run
inside the timed region.  Everything that computes runs inside libset.so; this file only marshals pointers.

Under torchrun (N > 1) every rank drives its own GPU with its own scheduler instance over its own jobs (weak
scaling, no data-path collective -- SURVEY.md §8(e)); time = max over ranks, value = all ranks' jobs / time.
"""
from __future__ import annotations

import argparse
import ctypes as C
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

L2_FLUSH_BYTES = 512 << 20  # > 126 MB L2


def log(*a):
    print(*a, file=sys.stderr, flush=True)


# ------------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled every 100 ms while a timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._pump, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for ln in self.proc.stdout:
            self.lines.append((time.perf_counter(), ln.strip()))

    def stop(self):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except subprocess.TimeoutExpired:
                self.proc.kill()

    def summary(self, windows):
        """Median SM clock over the samples that fall inside any (t0, t1) window of timed work."""
        sm, smax, reasons = [], 0.0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for t, ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                clk, mx = float(f[0]), float(f[1])
            except ValueError:
                continue
            smax = max(smax, mx)
            if any(a <= t <= b for a, b in windows):
                sm.append(clk)
                for n, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
        if not sm:  # region shorter than the sampling period: fall back to every sample taken
            for t, ln in self.lines:
                try:
                    sm.append(float(ln.split(",")[0]))
                except ValueError:
                    pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax or None, "reasons": sorted(reasons),
                "samples": len(sm)}


# ------------------------------------------------------------------------------------------------ job sets
class JobSet:
    """Pointers of one workload's jobs: ctypes arrays ready for set_submit_batch."""

    def __init__(self, n):
        self.n = n
        self.ins = (C.c_void_p * n)()
        self.outs = (C.c_void_p * n)()
        self.dims = None
        self.keep = []          # owners of the memory
        self.in_bytes = 0       # per step, summed over jobs
        self.out_bytes = 0
        self.out_views = []     # (job index, host view or device tensor) for spot checks
        self.pool_inputs = []   # distinct input images (numpy), index = job % len


_INPUTS = {}  # (config, params, variant, first job id, count) -> list of input images: generated once, reused by every arm


def job_inputs(wl, job_ids, npool):
    key = (wl.config, tuple(wl.params), wl.variant, job_ids[0] if len(job_ids) else 0, npool)
    if key not in _INPUTS:
        _INPUTS[key] = [wl.make_input(job_ids[k]) for k in range(npool)]
    return _INPUTS[key]


def build_jobs(setlib, ctx, wl, job_ids, io_device: bool, pool: int, out_ring: int):
    """Place the jobs' inputs in pinned host memory (or HBM) and give every job an output slot.
    pool     : number of DISTINCT input images generated (job k uses image k mod pool); 0 = all distinct.
    out_ring : number of output slots (job k writes slot k mod out_ring); 0 = one per job.  A ring is only used
               where one-slot-per-job does not fit (config 2: 512 x 64 MiB); it is >= in-flight + queued jobs."""
    import torch
    from paper_2606_05495_b200.workloads import PinnedArena
    n = len(job_ids)
    js = JobSet(n)
    npool = n if pool == 0 else min(pool, n)
    nring = n if out_ring == 0 else min(out_ring, n)
    dims = [wl.dims(j) for j in job_ids]
    if wl.config in (4, 5, 6):
        js.dims = (C.c_uint32 * (4 * n))(*[v for d in dims for v in d])
    images = job_inputs(wl, job_ids, npool)
    js.pool_inputs = images
    pool_dims = dims[:npool]
    in_sz = [wl.in_bytes(d) for d in pool_dims]
    # config 4: the job's frame size is that of its pool image
    if wl.config in (4, 5, 6):
        for k in range(n):
            d = pool_dims[k % npool]
            for i in range(4):
                js.dims[4 * k + i] = d[i]
        dims = [pool_dims[k % npool] for k in range(n)]
    out_sz = [wl.out_bytes(d) for d in dims]
    ring_sz = [max(out_sz[k] for k in range(r, n, nring)) for r in range(nring)]
    al = 256
    tot_in = sum((s + al - 1) // al * al for s in in_sz) + al
    tot_out = sum((s + al - 1) // al * al for s in ring_sz) + al
    if io_device:
        dev_in = torch.empty(tot_in, dtype=torch.uint8, device="cuda")
        dev_out = torch.zeros(tot_out, dtype=torch.uint8, device="cuda")
        js.keep += [dev_in, dev_out]
        base_in, base_out = dev_in.data_ptr(), dev_out.data_ptr()
        stage = torch.empty(max(in_sz), dtype=torch.uint8).pin_memory()
    else:
        arena = PinnedArena(ctx, tot_in + tot_out)
        js.keep.append(arena)
        base_in, base_out = arena.ptr, arena.ptr + tot_in
    in_ptr, off = [], 0
    for k in range(npool):
        a = base_in + off
        a = (a + al - 1) // al * al
        off = a - base_in
        if io_device:
            stage[:in_sz[k]] = torch.from_numpy(images[k])
            dev_in[off:off + in_sz[k]].copy_(stage[:in_sz[k]])
            torch.cuda.synchronize()
        else:
            arena.view[off:off + in_sz[k]] = images[k]
        in_ptr.append(a)
        off += in_sz[k]
    out_ptr, off = [], 0
    for r in range(nring):
        a = (base_out + off + al - 1) // al * al
        off = a - base_out
        out_ptr.append((a, off))
        off += ring_sz[r]
    for k in range(n):
        js.ins[k] = in_ptr[k % npool]
        js.outs[k] = out_ptr[k % nring][0]
    js.in_bytes = sum(in_sz[k % npool] for k in range(n))
    js.out_bytes = sum(out_sz)

    def read_out(k):
        o = out_ptr[k % nring][1]
        if io_device:
            return dev_out[o:o + out_sz[k]].cpu().numpy()
        return np.array(arena.view[tot_in + o:tot_in + o + out_sz[k]], copy=True)

    js.read_out = read_out
    js.dims_list = dims
    js.npool, js.nring = npool, nring
    return js


# ------------------------------------------------------------------------------------------------ one timed arm
MODES = {"set": 0, "plain_streams": 1, "batch_sync_graphs": 2, "single_graph": 3, "mutex_queue": 4}


# graph-shape options of every arm (SET and the in-run baselines share the job graph): --sm-copy / --pdl
OPTS = {"sm_copy_max_bytes": 0, "pdl": True, "num_dispatchers": 0, "submitters": 1, "streams_per_lane": 0, "completion_fence": 0,
        "completion_thread": 0, "bind_at_launch": 0}


def run_arm(setlib, wl, job_ids, mode: str, io_device: bool, steps: int, warmup: int, pool: int, out_ring: int,
            verify: int = 0, ctx_kw=None, flush=None, clock_windows=None, trace=None, opts=None):
    """W untimed + K timed steps of (submit every job, drain).  Returns a dict with per-step ms (CUDA events on
    torch's current stream, recorded around the host-synchronous submit..drain region), wall ms and library stats."""
    import torch
    o = dict(OPTS, **(opts or {}))
    ctx = setlib.Context(wl.num_streams, wl.max_inflight, mode=MODES[mode], io=setlib.IO_DEVICE if io_device else setlib.IO_HOST,
                         sm_copy_max_bytes=o["sm_copy_max_bytes"], timestamps=bool(o.get("timestamps")),
                         streams_per_lane=o["streams_per_lane"], completion_fence=o["completion_fence"], completion_thread=o["completion_thread"], bind_at_launch=o["bind_at_launch"],
                         **dict({"num_dispatchers": o["num_dispatchers"]}, **(ctx_kw or {})))
    try:
        ctx.register_builtin(wl.config, wl.variant, list(wl.params), pdl=o["pdl"])
        js = build_jobs(setlib, ctx, wl, job_ids, io_device, pool, out_ring)
        n = js.n

        # SET takes submissions from several caller threads (Algorithm 1 claims jobs with an atomic); the
        # baseline models are single-caller by definition
        nsub = max(1, min(int(o["submitters"]), n)) if mode == "set" else 1
        pool_ex = None
        if nsub > 1:
            from concurrent.futures import ThreadPoolExecutor
            pool_ex = ThreadPoolExecutor(nsub)
            cuts = [n * t // nsub for t in range(nsub + 1)]

            def step():
                futs = [pool_ex.submit(ctx.submit_batch_slice, js.ins, js.outs, js.dims, cuts[t], cuts[t + 1]) for t in range(nsub)]
                for f in futs:
                    f.result()
                ctx.drain()
        else:
            def step():
                ctx.submit_batch(js.ins, js.outs, js.dims)
                ctx.drain()

        for _ in range(warmup):
            step()
        torch.cuda.synchronize()
        ctx.reset_stats()
        if trace is not None:
            # gap pass: one step under CUPTI activity tracing; never used for a throughput number
            trace.start()
            step()
            torch.cuda.synchronize()
            g = trace.stop()
            js.keep.clear()
            return {"mode": mode, "io": "device" if io_device else "host", "jobs": n, "gaps": g}
        ev_ms, wall_ms, per_step_gaps, st_sum = [], [], [], None
        for _ in range(steps):
            if flush is not None:
                flush.add_(1)  # rewrite a buffer larger than L2 between timed steps
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0 = time.perf_counter()
            e0.record()
            step()
            e1.record()
            e1.synchronize()
            t1 = time.perf_counter()
            ev_ms.append(e0.elapsed_time(e1))
            wall_ms.append((t1 - t0) * 1e3)
            if clock_windows is not None:
                clock_windows.append((t0, t1))
            if o.get("timestamps"):
                # one reduction per step: the span of a step's stamps must not include the pause between steps
                g = ctx.gap_stats()
                g["overhead_frac"] = max(0.0, 1.0 - g["busy_union_us"] / (ev_ms[-1] * 1e3))
                per_step_gaps.append(g)
                stp = ctx.stats()
                st_sum = stp if st_sum is None else {k: (max(st_sum[k], v) if k in ("max_inflight_seen", "cuda_streams") else st_sum[k] + v) for k, v in stp.items()}
                ctx.reset_stats()
        st = st_sum if st_sum is not None else ctx.stats()
        gap_stats = merge_gap_stats(per_step_gaps) if per_step_gaps else None
        bad = 0
        if verify:
            from checker import compare, oracle_out          # the oracle is only touched for this spot check
            picks = sorted(set(np.linspace(0, n - 1, verify).astype(int).tolist()))
            # with an output ring only the last writer of a slot is still there
            picks = [k for k in picks if k + js.nring >= n] or [n - 1]
            for k in picks:
                try:
                    compare(wl, js.read_out(k), oracle_out(wl, js.pool_inputs[k % js.npool], js.dims_list[k]))
                except AssertionError as e:
                    bad += 1
                    log(f"  MISMATCH {wl.name} job {k}: {str(e)[:200]}")
        ms = float(np.sum(ev_ms)) / steps
        out = {"mode": mode, "io": "device" if io_device else "host", "jobs": n, "ms_per_step": ms,
               "wall_ms_per_step": float(np.sum(wall_ms)) / steps, "jobs_per_s": n / (ms * 1e-3),
               "step_ms": [round(x, 4) for x in ev_ms], "h2d_bytes": 0 if io_device else js.in_bytes,
               "d2h_bytes": 0 if io_device else js.out_bytes, "in_bytes": js.in_bytes, "out_bytes": js.out_bytes,
               "kernel_launches": st["kernel_nodes"] + st["copy_nodes"] + st["signal_nodes"], "verified": len(picks) if verify else 0, "mismatches": bad,
               "stats": st}
        if gap_stats is not None:
            out["device_gaps"] = gap_stats
        jobs_total = max(1, st["submitted"])
        out["host_us_per_job"] = {k: st["ns_" + k] / jobs_total / 1e3 for k in ("submit", "bind", "launch", "callback", "sync")}
        js.keep.clear()
        return out
    finally:
        if "pool_ex" in locals() and pool_ex is not None:
            pool_ex.shutdown()
        ctx.close()


def merge_gap_stats(per_step):
    """Job-weighted mean of the per-step device-stamp statistics (p99 / max: the worst step's)."""
    out = {}
    w = [g["jobs"] for g in per_step]
    tot = max(1, sum(w))
    for k in per_step[0]:
        if k in ("jobs", "gaps"):
            out[k] = int(sum(g[k] for g in per_step))
        elif k in ("gap_p99_us", "gap_max_us"):
            out[k] = round(max(g[k] for g in per_step), 4)
        elif k in ("span_us", "busy_union_us", "idle_gaps"):
            out[k] = round(sum(g[k] for g in per_step), 3)
        else:
            out[k] = round(sum(g[k] * n for g, n in zip(per_step, w)) / tot, 4)
    return out


def time_stages(setlib, wl, dims=None, iters=50):
    """Average device time of every stage kernel launched alone, back to back (set_time_stage: CUDA events on the
    launching stream).  Operands are L2-resident when the job is smaller than L2 -- as they are in the pipeline."""
    with setlib.Context(1, 1) as ctx:
        ctx.register_builtin(wl.config, wl.variant, list(wl.params))
        if wl.config == 5:
            # the SSSP kernels follow indices found in the slot's buffers: run one job first so that they hold a valid graph
            from paper_2606_05495_b200.workloads import PinnedArena
            img, d = wl.make_input(0), wl.dims(0)
            arena = PinnedArena(ctx, img.size + wl.out_bytes(d) + 1024)
            a_in, v_in = arena.take(img.size)
            v_in[:] = img
            a_out, _ = arena.take(wl.out_bytes(d))
            ctx.submit(0, a_in, a_out, d)
            ctx.drain()
            v_in = None
            arena.free()
        out = []
        for s in range(ctx.num_stages):
            try:
                out.append(ctx.time_stage(s, dims, warmup=5, iters=iters))
            except setlib.SetError:      # a loop's control kernel cannot run outside its WHILE node
                out.append(float("nan"))
        return out


_FLOOR = {}


def launch_floor_us(setlib):
    """Duration of a kernel node that does nothing (the debug delay stage with a 0 ns wait), timed like the stages: what
    one node of a job graph costs on this GPU whatever its work.  SURVEY.md 8(d): the latency-class kernels of configs
    0, 1 and 4 are judged against this floor rather than against the HBM roofline."""
    if "us" not in _FLOOR:
        with setlib.Context(1, 1) as ctx:
            ctx.register_builtin(0, setlib.VARIANT_SPIN, [64])
            _FLOOR["us"] = round(ctx.time_stage(ctx.num_stages - 1, (1, 1, 1, 0), warmup=5, iters=50), 3)
    return _FLOOR["us"]


def link_bandwidth():
    """H2D and D2H bandwidth of this box, both directions at once (pinned memory, two streams), GB/s."""
    import torch
    n = 256 << 20
    h_in, h_out = torch.empty(n, dtype=torch.uint8).pin_memory(), torch.empty(n, dtype=torch.uint8).pin_memory()
    d_in, d_out = torch.empty(n, dtype=torch.uint8, device="cuda"), torch.zeros(n, dtype=torch.uint8, device="cuda")
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    res = {}
    for name, both in (("simplex", False), ("duplex", True)):
        best_h2d = best_d2h = 0.0
        for _ in range(4):
            torch.cuda.synchronize()
            a0, a1, b0, b1 = (torch.cuda.Event(enable_timing=True) for _ in range(4))
            with torch.cuda.stream(s1):
                a0.record()
                d_in.copy_(h_in, non_blocking=True)
                a1.record()
            if not both:
                torch.cuda.synchronize()
            with torch.cuda.stream(s2):
                b0.record()
                h_out.copy_(d_out, non_blocking=True)
                b1.record()
            torch.cuda.synchronize()
            best_h2d = max(best_h2d, n / (a0.elapsed_time(a1) * 1e-3) / 1e9)
            best_d2h = max(best_d2h, n / (b0.elapsed_time(b1) * 1e-3) / 1e9)
        res[name] = {"h2d_gbs": best_h2d, "d2h_gbs": best_d2h}
    return res


# ------------------------------------------------------------------------------------------------ rooflines
def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "bf16_tflops": d["bf16_tflops"], "bf16_tflops_sustained": d.get("bf16_tflops_sustained"),
                "source": "measured (MEASURED_PEAKS.json)"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback (B200_PROFILING.md)"}


def stage_algorithmic(wl, dims):
    """Per stage: (kernel name, bound, algorithmic bytes or flops per launch) -- DESIGN.md "Kernels"."""
    c, p = wl.config, wl.params
    if c == 0:
        n = p[0]
        return [("scan_i32", "hbm", 8 * n), ("hist_mod64", "hbm", 4 * n + 256)]
    if c == 1:
        n = p[0]
        return [("affine_f32", "hbm", 8 * n), ("add_bias_f32", "hbm", 12 * n), ("relu_f32", "hbm", 8 * n),
                ("square_f32", "hbm", 8 * n), ("block_sum_f32", "hbm", 4 * n + 4)]
    if c == 2:
        h, w, sweeps = p
        return [("jacobi5_f32", "hbm", 8 * h * w)] * sweeps
    if c == 3:
        m, n, k = p
        return [("gemm_bias_gelu_bf16", "tensor", 2 * m * n * k)]
    if c == 4:
        px = dims[0] * dims[1]
        return [("rgb2gray_u8", "hbm", 4 * px), ("blur3x3_u8", "hbm", 2 * px), ("hist256_u8", "hbm", px + 1024)]
    if c == 5 and wl.variant == 1:  # one kernel runs the job: reads the image once per round at most; latency-class
        e = p[0] * wl.extra.get("mean_deg", 8)  # image (header, row_ptr, col, w) read + distances written
        return [("sssp_solo", "hbm", 16 + 4 * (p[0] + 1) + 8 * e + 4 * p[0] + 16)]
    if c == 5:  # timed alone the relaxation sees an empty frontier: it scans the V flags and stops (latency-class)
        v, unroll = p[0], (p[2] if len(p) > 2 else 4)
        return [("sssp_init", "hbm", 12 * v)] + [("sssp_relax", "hbm", 4 * v)] * unroll + [("sssp_control", "hbm", 16)]
    if c == 6:
        px = dims[0] * dims[1]
        return [("rgb2gray_u8", "hbm", 4 * px), ("sobel3x3_u8", "hbm", 2 * px), ("mean3x3_u8", "hbm", 2 * px), ("threshold_u8", "hbm", 2 * px),
                ("blend_u8", "hbm", 3 * px)]
    raise ValueError(c)


def kernel_rooflines(setlib, wl, pk, dims=None):
    us = time_stages(setlib, wl, dims)
    alg = stage_algorithmic(wl, dims or (1, 1, 1, 1))
    rows = []
    for (name, bound, work), t in zip(alg, us):
        if t != t:  # not timed (NaN)
            continue
        if bound == "hbm":
            ach, peak, unit = work / (t * 1e-6) / 1e9, pk["hbm_gbs"], "GB/s"
        else:
            ach, peak, unit = work / (t * 1e-6) / 1e12, pk["bf16_tflops"], "TFLOP/s"
        rows.append({"kernel": name, "bound": bound, "avg_us": round(t, 3), "algorithmic": work, "achieved": round(ach, 2),
                     "peak": peak, "unit": unit, "frac": round(ach / peak, 4)})
    # merge identical stages (the 10 Jacobi sweeps)
    merged = {}
    for r in rows:
        m = merged.setdefault(r["kernel"], dict(r, launches_per_job=0, total_us=0.0))
        m["launches_per_job"] += 1
        m["total_us"] += r["avg_us"]
    out = []
    for m in merged.values():
        m["avg_us"] = round(m["total_us"] / m["launches_per_job"], 3)
        if m["bound"] == "hbm":
            m["achieved"] = round(m["algorithmic"] / (m["avg_us"] * 1e-6) / 1e9, 2)
        else:
            m["achieved"] = round(m["algorithmic"] / (m["avg_us"] * 1e-6) / 1e12, 2)
        m["frac"] = round(m["achieved"] / m["peak"], 4)
        m["traffic"] = NCU_TRAFFIC.get("set_k_" + m["kernel"], {}).get(wl_key(wl))
        m["launch_floor_us"] = launch_floor_us(setlib)
        out.append(m)
    return out


def wl_key(wl):
    return f"config{wl.config}"


def _load_traffic():
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` captures
    (profiles/ncu_traffic.json, written from the .ncu-rep files; the file names the capture it came from)."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as f:
            return json.load(f).get("kernels", {})
    except Exception:
        return {}


NCU_TRAFFIC = _load_traffic()


def pipeline_roofline(wl, in_bytes_job, out_bytes_job, link, pk, dims):
    """north_star: slowest of host-link bytes / measured H2D,D2H bandwidth (full duplex), HBM bytes / HBM bandwidth,
    flops / tensor peak, per job.  Returns the three times (us) and the bound in jobs/s for e2e and device-resident IO."""
    alg = stage_algorithmic(wl, dims)
    hbm_bytes = sum(w for _, b, w in alg if b == "hbm")
    flops = sum(w for _, b, w in alg if b == "tensor")
    if wl.config == 3:
        m, n, k = wl.params
        hbm_bytes = 2 * m * k + 2 * k * n + 4 * n + 2 * m * n
    t_link = max(in_bytes_job / (link["duplex"]["h2d_gbs"] * 1e3), out_bytes_job / (link["duplex"]["d2h_gbs"] * 1e3))
    t_hbm_k = hbm_bytes / (pk["hbm_gbs"] * 1e3)
    t_hbm_copy = 2 * (in_bytes_job + out_bytes_job) / (pk["hbm_gbs"] * 1e3)   # D2D copy nodes of the device-resident arm
    t_flop = flops / (pk["bf16_tflops_sustained"] * 1e6) if flops else 0.0
    t_e2e = max(t_link, t_hbm_k + (in_bytes_job + out_bytes_job) / (pk["hbm_gbs"] * 1e3), t_flop)
    t_dev = max(t_hbm_k + t_hbm_copy, t_flop)
    return {"t_link_us": round(t_link, 3), "t_hbm_us": round(t_hbm_k, 3), "t_flop_us": round(t_flop, 3),
            "e2e_bound_jobs_per_s": round(1e6 / t_e2e, 1), "device_bound_jobs_per_s": round(1e6 / t_dev, 1),
            "e2e_bound_by": "link" if t_e2e == t_link else ("tensor" if t_e2e == t_flop else "hbm")}


# ------------------------------------------------------------------------------------------------ CPU oracle arm
def oracle_pass(wl, images, dims_list, budget_s: float):
    """Time the oracle, as it stands, single-threaded, over the given job images until `budget_s` of CPU work is done
    or every job has been processed once.  Returns (jobs done, seconds)."""
    from checker import oracle_out
    done, t0 = 0, time.perf_counter()
    for img, d in zip(images, dims_list):
        oracle_out(wl, img, d)
        done += 1
        if time.perf_counter() - t0 > budget_s:
            break
    return done, time.perf_counter() - t0


def cpu_baseline(wl, job_ids, budget_s=12.0, passes=100000, all_cores_s=4.0):
    """The oracle, as it stands, timed on this box's host cores over a bounded sample of the workload's jobs."""
    cap = {0: 256, 1: 2048, 2: 2, 3: 1, 4: 24, 5: 64, 6: 24}[wl.config]      # distinct inputs prepared for the sample
    n = min(len(job_ids), cap)
    if wl.config == 3 and budget_s < 60:
        return cpu_baseline_config3_sampled(wl, job_ids, budget_s)
    images = job_inputs(wl, job_ids, n)
    dims = [wl.dims(j) for j in job_ids[:n]]
    total, secs = 0, 0.0
    for _ in range(passes):
        d, s = oracle_pass(wl, images, dims, budget_s - secs)
        total += d
        secs += s
        if secs >= budget_s:
            break
    out = {"value": round(total / secs, 2), "unit": "jobs/s", "cores": 1, "kind": "oracle",
           "sample": f"{total} jobs of the workload (first {n} job inputs, repeated) in {secs:.1f} s, single thread, oracle/*.c -O2"}
    # the same oracle, job-parallel over the box's cores (jobs are independent; ctypes releases the GIL inside the C call)
    try:
        from concurrent.futures import ThreadPoolExecutor
        cores = len(os.sched_getaffinity(0))
        if cores > 1 and all_cores_s > 0:
            chunks = [(images[i::cores], dims[i::cores]) for i in range(cores)]
            def worker(c, budget=all_cores_s):
                n_done, t_used = 0, 0.0
                while t_used < budget and c[0]:
                    d, t = oracle_pass(wl, c[0], c[1], budget - t_used)
                    n_done, t_used = n_done + d, t_used + t
                return n_done

            t0 = time.perf_counter()
            with ThreadPoolExecutor(cores) as ex:
                done = sum(ex.map(worker, chunks))
            dt = time.perf_counter() - t0
            out["all_cores"] = {"value": round(done / dt, 2), "cores": cores, "sample": f"{done} jobs in {dt:.1f} s, one thread per core"}
    except Exception as e:
        out["all_cores"] = {"error": str(e)[:120]}
    return out




def cpu_baseline_config3_sampled(wl, job_ids, budget_s):
    """Config 3: one full 2048^3 job takes the naive-loop oracle minutes, so the bounded sample is a set of output entries
    of one job computed one by one (oracle_config3_sampled, the same arithmetic per entry) and the per-job figure is
    extrapolated from the entry rate -- labelled as such (SURVEY.md 8(d) "Oracle timing")."""
    import oracle
    m, n, k = wl.params
    img = job_inputs(wl, job_ids, 1)[0]
    a = img[:2 * m * k].view(np.uint16).reshape(m, k)
    b = img[2 * m * k:2 * m * k + 2 * k * n].view(np.uint16).reshape(k, n)
    bias = img[2 * m * k + 2 * k * n:].view(np.float32)
    per, done, t0 = 4096, 0, time.perf_counter()
    while time.perf_counter() - t0 < budget_s:
        r = np.arange(done, done + per, dtype=np.int64)
        oracle.config3_sampled(a, b, bias, (r * 7919) % m, (r * 104729) % n)
        done += per
    secs = time.perf_counter() - t0
    return {"value": round(done / secs / (m * n), 6), "unit": "jobs/s", "cores": 1, "kind": "oracle", "extrapolated": True,
            "sample": f"{done} output entries of one job ({m}x{n}x{k}) in {secs:.1f} s, single thread; per-job rate = entry rate / {m * n}"}
# ------------------------------------------------------------------------------------------------ main
# distinct-input pool / output ring per config (0 = one per job).  Rings are >= b*(q+1) outstanding jobs.
LAYOUT = {0: (0, 0), 1: (0, 0), 2: (16, 32), 3: (8, 64), 4: (96, 128), 5: (64, 0), 6: (96, 128)}
GAP_JOBS = {0: 256, 1: 2000, 2: 64, 3: 200, 4: 512, 5: 256, 6: 512}  # jobs traced per arm in the CUPTI pass (records stay in host memory)
SIDE_STEPS, SIDE_WARMUP = 2, 2                                       # side workloads and secondary arms: fixed, small


def gap_pass(setlib, wl, ids, all_configs: bool, warmup: int):
    """Kernel-level gaps and device idle fraction from CUPTI activity records (include/set_trace.h), for SET and for the
    batch-synchronous-graph baseline on the same jobs.  Runs after every timed arm: tracing slows the launch path, so no
    throughput figure comes from here."""
    out = {"how": "one step per arm under CUPTI activity tracing (kernel, memcpy, memset records), after all timed arms; records are "
                  "grouped into jobs by the correlation id of their cudaGraphLaunch and jobs into work streams by the stream of the job's "
                  "first stage kernel; kernel->kernel gaps are signed (negative = PDL overlap); idle_frac = 1 - |union of activity| / wall"}
    try:
        from paper_2606_05495_b200 import trace
        trace.load()
    except Exception as e:
        return {"unavailable": str(e)[:200]}
    todo = [(wl, ids)]
    if all_configs:
        todo += [(workload_for(c), None) for c in range(5) if c != wl.config]
    for w, job_ids in todo:
        job_ids = list(range(w.jobs)) if job_ids is None else job_ids
        job_ids = job_ids[:GAP_JOBS[w.config]]
        p, r = LAYOUT[w.config]
        res = {"jobs": len(job_ids)}
        for mode in ("set", "batch_sync_graphs"):
            key = f"{mode}_e2e"
            try:
                g = run_arm(setlib, w, job_ids, mode, False, 1, max(1, min(warmup, 2)), p, r, trace=trace)["gaps"]
                res[key] = g
                log(f"[bench]   cupti config{w.config} {key:28s} kernel->kernel mean {g['kernel_kernel']['mean_us']:.2f} us "
                    f"p99 {g['kernel_kernel']['p99_us']:.2f}  inter-job mean {g['inter_job']['mean_us']:.2f} us  idle {g['idle_frac']:.3f}")
            except Exception as e:
                res[key] = {"error": str(e)[:200]}
                log(f"[bench]   cupti config{w.config} {key} failed: {e}")
        out[f"config{w.config}"] = res
    return out


SWEEP_B = (1, 2, 4, 8, 16, 32, 64, 128, 256, 512, 1024, 2048, 4096)


def batch_sweep(setlib, wl, ids, flush):
    """SURVEY.md 8(f)2 / PAPER.md:274-288 (Fig. 5-6): for b = max_inflight from 1 to 4096 and the three models the paper
    draws (SET, batching, queue) -- throughput, the scheduling-overhead fraction (1 - |union of job intervals| / T, reading
    S12, from the device stamps) and the mean device-side gap between consecutive jobs of a stream.  End to end, pinned host
    buffers, streams fixed at the workload's S (b < S: b streams)."""
    import copy
    out = {"workload": wl.name, "jobs": min(len(ids), 8192), "b": {},
           "how": "3 timed steps per point with set_config.timestamps=1 (two stamp nodes per job); overhead_frac = 1 - busy_union / step time"}
    job_ids = ids[:out["jobs"]]
    p, r = LAYOUT[wl.config]
    for b in SWEEP_B:
        w = copy.copy(wl)
        w.max_inflight, w.num_streams = b, min(b, wl.num_streams)
        row = {}
        for mode in ("set", "batch_sync_graphs", "mutex_queue"):
            try:
                res = run_arm(setlib, w, job_ids, mode, False, 3, 2, p, max(r, 0), verify=0, flush=flush, opts={"timestamps": True})
                g = res["device_gaps"]
                row[mode] = {"jobs_per_s": round(res["jobs_per_s"], 1), "overhead_frac": round(g["overhead_frac"], 4),
                             "gap_mean_us": round(g["gap_mean_us"], 2), "host_us_per_job": round(sum(res["host_us_per_job"][k] for k in ("submit", "launch", "callback")), 3)}
            except Exception as e:
                row[mode] = {"error": str(e)[:120]}
        if all("jobs_per_s" in v for v in row.values()):
            row["set_over_batch"] = round(row["set"]["jobs_per_s"] / row["batch_sync_graphs"]["jobs_per_s"], 3)
            row["set_over_queue"] = round(row["set"]["jobs_per_s"] / row["mutex_queue"]["jobs_per_s"], 3)
        out["b"][str(b)] = row
        log(f"[bench]   sweep b={b:5d} S={w.num_streams}: {row}")
    return out


def device_gap_arms(setlib, w, job_ids, modes, flush, steps=3):
    """Gaps between consecutive jobs of a stream and the overhead fraction from the GPU's own clock (set_config.timestamps,
    set_get_gap_stats): two one-thread stamp nodes per job graph, no profiler attached, full speed, end to end."""
    p, r = LAYOUT[w.config]
    res = {"jobs_per_step": len(job_ids)}
    for mode in modes:
        key = f"{mode}_e2e"
        try:
            a = run_arm(setlib, w, job_ids, mode, False, steps, 2, p, r, verify=0, flush=flush, opts={"timestamps": True})
            res[key] = dict(a["device_gaps"], jobs_per_s=round(a["jobs_per_s"], 1),
                            host_us_per_job={k: round(v, 3) for k, v in a["host_us_per_job"].items()})
            g = res[key]
            log(f"[bench]   stamps config{w.config} {key:24s} inter-job gap mean {g['gap_mean_us']:.2f} us p99 {g['gap_p99_us']:.2f}  job chain "
                f"{g['job_mean_us']:.2f} us  overhead frac {g['overhead_frac']:.4f}  {g['jobs_per_s']:.0f} jobs/s")
        except Exception as e:
            res[key] = {"error": str(e)[:200]}
            log(f"[bench]   stamps config{w.config} {key} failed: {e}")
    return res


def workload_for(config, jobs_override=None):
    from paper_2606_05495_b200.workloads import baseline_workload
    wl = baseline_workload(config)
    if jobs_override:
        wl.jobs = jobs_override
    return wl


def mean_dims(wl, job_ids):
    if wl.config not in (4, 6):
        return (1, 1, 1, 1)
    return (1280, 720, 1, 1)


def reference_main(args, rank, world):
    """--impl reference: the CPU oracle, as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return 0
    from oracle import build as ob
    ob.build()
    wl = workload_for(args.config, args.jobs)
    ids = list(range(wl.jobs))
    per_step_budget = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    n = min(len(ids), 4096 if wl.config == 1 else 64)
    images = [wl.make_input(j) for j in ids[:n]]
    dims = [wl.dims(j) for j in ids[:n]]
    for _ in range(args.warmup):
        oracle_pass(wl, images[:max(1, n // 8)], dims, per_step_budget / 4)
    tot, secs = 0, 0.0
    for _ in range(args.steps):
        d, s = oracle_pass(wl, images, dims, per_step_budget)
        tot += d
        secs += s
    v = tot / secs
    line = {"impl": "reference", "metric": "jobs/s", "value": round(v, 3), "unit": "jobs/s", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": round(secs / args.steps * 1e3, 3), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": wl.dtype, "data": "synthetic",
            "config": {"workload": wl.name, "jobs_per_step_sampled": tot // max(1, args.steps)},
            "cpu_baseline": {"value": round(v, 3), "unit": "jobs/s", "cores": 1, "kind": "oracle",
                             "sample": f"each step = up to {n} jobs of the workload or {per_step_budget:.0f} s, single thread"},
            "e2e": {"value": round(v, 3), "unit": "jobs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------ the compact line
REQUIRED_KEYS = ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
                 "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline")


def _r(x, nd=1):
    return None if x is None else round(float(x), nd)


def compact_line(wl, world, steps, warmup, n_jobs, ms_dev, value, ms_e2e, e2e_value, dev_arm, e2e_arm, clocks, detail, detail_path, pk):
    """The one stdout line (driver contract + tier additions), built from the measured arms and the detail dict.  Pure host
    arithmetic: tests/test_bench_helpers.py feeds it fake arms and checks the keys and the size bound."""
    kr = detail.get("kernels") or []
    dom = max(kr, key=lambda r: r.get("total_us", 0)) if kr else None
    roof = None
    if dom:
        roof = {"bound": dom["bound"], "achieved": dom["achieved"], "peak": dom["peak"], "unit": dom["unit"], "frac": dom["frac"],
                "traffic": dom.get("traffic"), "kernel": dom["kernel"], "avg_us": dom["avg_us"], "peak_source": pk["source"].split(" ")[0],
                "floor_us": dom.get("launch_floor_us")}  # floor_us: an empty kernel node; avg_us near it = latency-class kernel
    line = {"metric": "jobs/s", "value": _r(value), "unit": "jobs/s", "n_gpus": world, "steps": steps, "warmup": warmup,
            "ms_per_step": _r(ms_dev, 4), "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": wl.dtype,
            "data": "synthetic",
            "config": {"workload": wl.name, "jobs_per_step_per_gpu": n_jobs, "num_streams": wl.num_streams, "max_inflight": wl.max_inflight,
                       "streams_per_lane": detail.get("streams_per_lane"), "io": "value: HBM-resident; e2e: pinned host",
                       "l2": f"{L2_FLUSH_BYTES >> 20} MiB flush/step; {dev_arm['in_bytes'] / 1e6:.0f} MB inputs/step"},
            "clocks": clocks,
            "e2e": {"value": _r(e2e_value), "unit": "jobs/s", "h2d_bytes_per_step": int(e2e_arm["h2d_bytes"] * world),
                    "d2h_bytes_per_step": int(e2e_arm["d2h_bytes"] * world), "ms_per_step": _r(ms_e2e, 4)},
            "gpu_launches": int(dev_arm["kernel_launches"] * world),
            "mismatches": int(dev_arm["mismatches"] + e2e_arm["mismatches"] + detail.get("side_mismatches", 0)),
            "roofline": roof, "cpu_baseline": None}
    cb = detail.get("cpu_baseline")
    if cb:  # the line carries the contract's five fields; the job-parallel figure stays in the detail file
        line["cpu_baseline"] = {"value": cb["value"], "unit": cb["unit"], "cores": cb["cores"], "kind": cb["kind"], "sample": cb["sample"][:90]}
    # BASELINE.json:metric in one object, e2e first: jobs/s; gap between jobs of a stream; scheduling overhead vs batched graphs
    base = detail.get("baselines", {})
    dg = detail.get("device_gaps", {}).get(f"config{wl.config}", {})

    def pick(key, field, nd=3):
        v = dg.get(key, {})
        return _r(v.get(field), nd) if isinstance(v, dict) and field in v else None

    bs = base.get("batch_sync_graphs_e2e", {}).get("jobs_per_s")
    hm = {"batch_sync_e2e_jobs_per_s": _r(bs),  # SET's own is e2e.value
          "set_over_batch_sync_e2e": _r(e2e_value / bs, 3) if bs else None,
          # per CUDA stream: start(next job) - end(previous job); device-wide: intervals with no job in progress anywhere
          "gap_between_jobs_us": {"set": pick("set_e2e", "gap_mean_us", 2), "batch_sync": pick("batch_sync_graphs_e2e", "gap_mean_us", 2),
                                  "set_p99": pick("set_e2e", "gap_p99_us", 2), "batch_sync_p99": pick("batch_sync_graphs_e2e", "gap_p99_us", 2)},
          "idle_gaps_n_meanus": {"set": [pick("set_e2e", "idle_gaps", 0), pick("set_e2e", "idle_gap_mean_us", 2)],
                                            "batch_sync": [pick("batch_sync_graphs_e2e", "idle_gaps", 0), pick("batch_sync_graphs_e2e", "idle_gap_mean_us", 2)]},
          "sched_overhead_frac": {"set": pick("set_e2e", "overhead_frac", 4), "batch_sync": pick("batch_sync_graphs_e2e", "overhead_frac", 4)},
          "host_us_per_job": {"set": _r(sum(e2e_arm["host_us_per_job"][k] for k in ("submit", "launch", "callback")), 3),
                              "batch_sync": _r(sum(base["batch_sync_graphs_e2e"]["host_us_per_job"][k] for k in ("submit", "launch")), 3)
                              if "batch_sync_graphs_e2e" in base else None}}
    cg = detail.get("gaps_cupti", {}).get(f"config{wl.config}", {})

    def kk(key):
        v = cg.get(key, {})
        return _r(v["kernel_kernel"]["mean_us"], 2) if isinstance(v, dict) and "kernel_kernel" in v else None

    # stage kernel -> next stage kernel of a job, signed (negative = the PDL edge overlapped them), from CUPTI records of a traced step
    hm["inter_kernel_gap_us"] = {"set": kk("set_e2e"), "batch_sync": kk("batch_sync_graphs_e2e")}
    pr = detail.get("pipeline_roofline")
    if pr:
        hm["pipeline_roofline"] = {"bound_by": pr["e2e_bound_by"], "e2e_bound_jobs_per_s": pr["e2e_bound_jobs_per_s"], "e2e_frac": pr["e2e_frac"]}
    line["headline_metrics"] = hm
    side = {}
    for k, v in (detail.get("workloads") or {}).items():
        side[k] = [v.get("e2e"), (v.get("pipeline_roofline") or {}).get("e2e_frac"), v.get("speedup_vs_batch_sync_e2e")] \
            if "error" not in v else "error: " + v["error"][:24]  # the full text is in the detail file
    if side:
        line["workloads_e2e_frac_vsbatch"] = side  # per config: [e2e jobs/s, fraction of its pipeline roofline, SET / batch-sync]
    kroofs = {}
    for k, v in (detail.get("workloads") or {}).items():
        for row in v.get("kernels", []) if isinstance(v, dict) else []:
            if row["kernel"] in ("jacobi5_f32", "gemm_bias_gelu_bf16"):
                kroofs[row["kernel"]] = {"frac": row["frac"], "avg_us": row["avg_us"], "bound": row["bound"]}
    if kroofs:
        line["kernel_rooflines"] = kroofs
    line["detail"] = os.path.basename(detail_path) if detail_path else None
    return line


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json:configs index of the headline workload")
    ap.add_argument("--jobs", type=int, default=None, help="override the job count (debugging only)")
    ap.add_argument("--suite", default="default", choices=["headline", "default", "all"],
                    help="headline: the headline workload, its batch-sync baseline, rooflines, CPU oracle; default: + the other four "
                         "configs (2 steps each) and the device-stamp gap pass; all: + completion modes, graph variants, every "
                         "baseline model, per-config CPU oracle timing and the CUPTI gap pass (N=1 only)")
    ap.add_argument("--impl", default="set", choices=["set", "reference"])
    ap.add_argument("--no-baselines", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-gaps", action="store_true", help="skip the gap passes")
    ap.add_argument("--sm-copy", type=int, default=0, help="set_config.sm_copy_max_bytes: 0 = library default, -1 = copy engines only")
    ap.add_argument("--submitters", type=int, default=1, help="caller threads that submit a step's jobs to SET (baselines: always 1)")
    ap.add_argument("--dispatchers", type=int, default=0, help="set_config.num_dispatchers (0 = library default, 1)")
    ap.add_argument("--lanes", type=int, default=0, help="set_config.streams_per_lane (0 = library default)")
    ap.add_argument("--fence", type=int, default=0, help="set_config.completion_fence: 0 default, 1 system fence, 2 none")
    ap.add_argument("--pdl", type=int, default=1, help="1: programmatic-dependent-launch edges between kernel nodes (default), 0: plain edges")
    ap.add_argument("--sweep", action="store_true", help="also sweep the batch size b = 1..4096 (PAPER.md Fig. 5-6) on the headline workload")
    ap.add_argument("--out", default=os.path.join(ROOT, "bench_detail.json"), help="detail file (everything that is not on the stdout line)")
    args = ap.parse_args()
    OPTS["sm_copy_max_bytes"], OPTS["pdl"], OPTS["num_dispatchers"] = args.sm_copy, bool(args.pdl), args.dispatchers
    OPTS["submitters"], OPTS["streams_per_lane"], OPTS["completion_fence"] = args.submitters, args.lanes, args.fence

    from paper_2606_05495_b200 import multi
    if args.impl == "reference":
        rank, _, world = multi.env_rank()
        return reference_main(args, rank, world)

    import torch
    rank, local_rank, world = multi.init_process_group()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    from paper_2606_05495_b200 import build as lib_build
    if rank == 0:
        lib_build.build()
    multi.barrier(dev)
    import paper_2606_05495_b200 as setlib
    setlib.load()

    t_start = time.perf_counter()
    steps, warmup = args.steps, max(args.warmup, 0)
    pk = peaks()
    flush = torch.zeros(L2_FLUSH_BYTES // 4, dtype=torch.int32, device=dev)
    sampler = ClockSampler(local_rank)
    sampler.start()
    windows = []

    wl = workload_for(args.config, args.jobs)
    ids = list(multi.shard_jobs(wl.jobs, rank, world, "weak"))
    log(f"[bench] rank {rank}/{world} headline {wl.name}: {len(ids)} jobs/step, {steps} steps, {warmup} warm-up, suite {args.suite}")

    def arm(w, job_ids, mode, io_device, k=steps, wu=warmup, verify=4, win=None, **kw):
        p, r = LAYOUT[w.config]
        multi.barrier(dev)
        torch.cuda.synchronize()
        res = run_arm(setlib, w, job_ids, mode, io_device, k, wu, p, r, verify=verify, flush=flush, clock_windows=win, **kw)
        torch.cuda.synchronize()
        multi.barrier(dev)
        log(f"[bench]   {w.config} {mode:18s} {'device' if io_device else 'host  '} {res['jobs_per_s']:12.1f} jobs/s "
            f"{res['ms_per_step']:9.3f} ms/step  host us/job { {k_: round(v, 3) for k_, v in res['host_us_per_job'].items()} }  mismatches {res['mismatches']}")
        return res

    def brief(r):
        return {"jobs_per_s": round(r["jobs_per_s"], 1), "ms_per_step": round(r["ms_per_step"], 3), "mismatches": r["mismatches"],
                "host_us_per_job": {k: round(v, 3) for k, v in r["host_us_per_job"].items()}}

    # ---- the headline arms first: whatever happens later, these numbers exist
    e2e_arm = arm(wl, ids, "set", False, win=windows)
    dev_arm = arm(wl, ids, "set", True, win=windows)
    ms_dev, units = multi.aggregate(dev_arm["ms_per_step"], dev_arm["jobs"], dev)
    ms_e2e, _ = multi.aggregate(e2e_arm["ms_per_step"], e2e_arm["jobs"], dev)
    value, e2e_value = units / (ms_dev * 1e-3), units / (ms_e2e * 1e-3)

    detail = {"argv": sys.argv[1:], "suite": args.suite, "peaks": pk}
    detail["streams_per_lane"] = e2e_arm["stats"].get("cuda_streams", 0) // max(1, wl.num_streams)
    detail["set_e2e"], detail["set_device"] = dict(brief(e2e_arm), stats=e2e_arm["stats"], step_ms=e2e_arm["step_ms"]), dict(brief(dev_arm), stats=dev_arm["stats"], step_ms=dev_arm["step_ms"])
    side_bad = 0
    if world == 1:
        link = link_bandwidth()
        detail["link_gbs"] = link
        d = mean_dims(wl, ids)
        in_job, out_job = e2e_arm["in_bytes"] / e2e_arm["jobs"], e2e_arm["out_bytes"] / e2e_arm["jobs"]
        pr = pipeline_roofline(wl, in_job, out_job, link, pk, d)
        pr["e2e_frac"] = round(e2e_value / pr["e2e_bound_jobs_per_s"], 4)
        pr["device_frac"] = round(value / pr["device_bound_jobs_per_s"], 4)
        detail["pipeline_roofline"] = pr
        detail["kernels"] = kernel_rooflines(setlib, wl, pk, d if wl.config in (4, 6) else None)
        ks = min(steps, 10)
        if not args.no_baselines:
            base = {}
            modes = ("batch_sync_graphs",) if args.suite != "all" else ("batch_sync_graphs", "plain_streams", "single_graph", "mutex_queue")
            for mode in modes:
                for io_device in (False, True):
                    base[f"{mode}_{'device' if io_device else 'e2e'}"] = brief(arm(wl, ids, mode, io_device, ks, min(warmup, 3), verify=2))
            detail["baselines"] = base
            detail["speedup_vs_batch_sync_graphs"] = {"e2e": round(e2e_value / base["batch_sync_graphs_e2e"]["jobs_per_s"], 3),
                                                      "device": round(value / base["batch_sync_graphs_device"]["jobs_per_s"], 3)}
        if not args.no_gaps:
            gm = ("set", "batch_sync_graphs") if args.suite == "headline" else ("set", "batch_sync_graphs", "mutex_queue")
            detail["device_gaps"] = {"how": "set_config.timestamps=1: %globaltimer at graph start (root node) and end (signal / last node); gap = "
                                            "start(next job on the CUDA stream) - end(previous); overhead_frac = 1 - |union of job intervals| / step time "
                                            "(PAPER.md:81-90, :253, reading S12), per step; e2e arms",
                                     f"config{wl.config}": device_gap_arms(setlib, wl, ids, gm, flush)}
        if args.suite == "all" and not args.no_baselines:
            cm = {}
            for name, cb in (("hostfunc_notify_stream", 1), ("hostfunc_work_stream", 2), ("graph_host_node", 4)):
                cm[name + "_e2e"] = brief(arm(wl, ids, "set", False, ks, min(warmup, 3), verify=2, ctx_kw={"callback_mode": cb}))
            for name, f in (("flag_poll_system_fence", 1), ("flag_poll_no_fence", 2)):
                cm[name + "_e2e"] = brief(arm(wl, ids, "set", False, ks, min(warmup, 3), verify=2, opts={"completion_fence": f}))
            detail["completion_modes"] = cm
            gv = {}
            for name, o in (("ce_copies_plain_edges", {"sm_copy_max_bytes": -1, "pdl": False}), ("ce_copies_pdl", {"sm_copy_max_bytes": -1, "pdl": True}),
                            ("sm_copies_plain_edges", {"sm_copy_max_bytes": 262144, "pdl": False}), ("sm_copies_pdl", {"sm_copy_max_bytes": 262144, "pdl": True})):
                for io_device in (False, True):
                    gv[f"{name}_{'device' if io_device else 'e2e'}"] = brief(arm(wl, ids, "set", io_device, ks, min(warmup, 3), verify=2, opts=o))
            detail["graph_variants"] = gv
            lv = {}
            for lanes in (1, 2, 4):
                for mode in ("set", "batch_sync_graphs"):
                    lv[f"{mode}_lanes{lanes}_e2e"] = brief(arm(wl, ids, mode, False, ks, min(warmup, 3), verify=2, opts={"streams_per_lane": lanes}))
            detail["streams_per_lane_variants"] = lv
        if args.suite in ("default", "all"):
            others = {}
            for c in SIDE_CONFIGS:
                if c == wl.config:
                    continue
                w2 = workload_for(c)
                ids2 = list(range(w2.jobs))
                try:
                    a_e2e = arm(w2, ids2, "set", False, SIDE_STEPS, SIDE_WARMUP, verify=2)
                    b_e2e = arm(w2, ids2, "batch_sync_graphs", False, SIDE_STEPS, SIDE_WARMUP, verify=0)
                    a_dev = arm(w2, ids2, "set", True, SIDE_STEPS, SIDE_WARMUP, verify=2)
                    d2 = mean_dims(w2, ids2)
                    pr2 = pipeline_roofline(w2, a_e2e["in_bytes"] / a_e2e["jobs"], a_e2e["out_bytes"] / a_e2e["jobs"], link, pk, d2)
                    row = {"workload": w2.name, "e2e": round(a_e2e["jobs_per_s"], 1), "value": round(a_dev["jobs_per_s"], 1),
                           "batch_sync_graphs_e2e": round(b_e2e["jobs_per_s"], 1),
                           "speedup_vs_batch_sync_e2e": round(a_e2e["jobs_per_s"] / b_e2e["jobs_per_s"], 3),
                           "host_us_per_job": {k: round(v, 3) for k, v in a_e2e["host_us_per_job"].items()},
                           "mismatches": a_dev["mismatches"] + a_e2e["mismatches"],
                           "pipeline_roofline": dict(pr2, e2e_frac=round(a_e2e["jobs_per_s"] / pr2["e2e_bound_jobs_per_s"], 4)),
                           "kernels": kernel_rooflines(setlib, w2, pk, d2 if c in (4, 6) else None)}
                    side_bad += row["mismatches"]
                    if args.suite == "all" and not args.no_baselines:
                        b_dev = arm(w2, ids2, "batch_sync_graphs", True, SIDE_STEPS, SIDE_WARMUP, verify=0)
                        row["batch_sync_graphs_device"] = round(b_dev["jobs_per_s"], 1)
                        row["speedup_vs_batch_sync_device"] = round(a_dev["jobs_per_s"] / b_dev["jobs_per_s"], 3)
                    if not args.no_cpu:
                        # SURVEY.md 8(d) "Oracle timing": every config, bounded; config 0 is where a CPU core may out-run the PCIe round trip
                        row["cpu_baseline"] = cpu_baseline(w2, ids2, budget_s=3.0 if args.suite == "default" else 10.0,
                                                           all_cores_s=0.0 if args.suite == "default" else 3.0)
                        row["gpu_e2e_over_one_cpu_core"] = round(row["e2e"] / row["cpu_baseline"]["value"], 2) if row["cpu_baseline"]["value"] else None
                    if args.suite == "all" and not args.no_gaps:
                        detail["device_gaps"][f"config{c}"] = device_gap_arms(setlib, w2, ids2[:{0: 256, 1: 10000, 2: 64, 3: 200, 4: 1024}.get(c, 256)],
                                                                              ("set", "batch_sync_graphs"), flush, steps=2)
                    others[f"config{c}"] = row
                except Exception as e:  # a failing side workload must not hide the headline number
                    others[f"config{c}"] = {"error": str(e)[:300]}
                    log(f"[bench] config {c} failed: {e}")
                _INPUTS.clear()  # the side workloads' inputs are large (config 2: 1 GB): keep only what is in use
            detail["workloads"] = others
            # config 5, variant 1: the whole SSSP job as ONE kernel of one block instead of the WHILE-node pipeline;
            # detail file only -- the stdout line keeps the WHILE-node pipeline, which is what SURVEY.md 8(f)4 names
            if wl.config != 5:
                try:
                    import dataclasses
                    w5 = dataclasses.replace(workload_for(5), variant=1, kernels_per_job=1)
                    ids5 = list(range(w5.jobs))
                    # the copy-in (16 + 4 (V + 1) + 8 E bytes, capacity 508 KB) as an SM copy: the copy engines get through about
                    # 90 K copies of this size a second whatever the stream count; device-resident: one CUDA stream per slot
                    vo = {"sm_copy_max_bytes": 1 << 20}
                    v_e2e = arm(w5, ids5, "set", False, SIDE_STEPS, SIDE_WARMUP, verify=2, opts=vo)
                    v_bat = arm(w5, ids5, "batch_sync_graphs", False, SIDE_STEPS, SIDE_WARMUP, verify=0, opts=vo)
                    v_dev = arm(w5, ids5, "set", True, SIDE_STEPS, SIDE_WARMUP, verify=2, opts=dict(vo, streams_per_lane=4))
                    v_ce = arm(w5, ids5, "set", False, SIDE_STEPS, SIDE_WARMUP, verify=0)
                    bound = (others.get("config5") or {}).get("pipeline_roofline", {}).get("e2e_bound_jobs_per_s")
                    detail["variants"] = {"config5_single_kernel": {
                        "options": "sm_copy_max_bytes = 1 MiB (SM copy-in); device-resident arm: streams_per_lane = 4",
                        "e2e_with_default_options_copy_engine_in": round(v_ce["jobs_per_s"], 1),
                        "e2e": round(v_e2e["jobs_per_s"], 1), "value": round(v_dev["jobs_per_s"], 1), "batch_sync_graphs_e2e": round(v_bat["jobs_per_s"], 1),
                        "speedup_vs_batch_sync_e2e": round(v_e2e["jobs_per_s"] / v_bat["jobs_per_s"], 3),
                        "e2e_frac_of_link_bound": round(v_e2e["jobs_per_s"] / bound, 4) if bound else None,
                        "mismatches": v_e2e["mismatches"] + v_dev["mismatches"],
                        "kernels": kernel_rooflines(setlib, w5, pk, None)}}
                    side_bad += detail["variants"]["config5_single_kernel"]["mismatches"]
                except Exception as e:
                    detail["variants"] = {"config5_single_kernel": {"error": str(e)[:300]}}
                    log(f"[bench] config 5 variant 1 failed: {e}")
                _INPUTS.clear()
        if args.sweep:
            detail["batch_sweep"] = batch_sweep(setlib, wl, ids, flush)
    detail["side_mismatches"] = side_bad
    sampler.stop()
    clocks = sampler.summary(windows)
    if world == 1 and args.suite != "headline" and not args.no_gaps:
        # kernel-level gaps need the profiler's activity records: after every timed arm, the headline workload only unless --suite all
        detail["gaps_cupti"] = gap_pass(setlib, wl, ids, args.suite == "all", warmup)
    if rank == 0 and world == 1 and not args.no_cpu:
        detail["cpu_baseline"] = cpu_baseline(wl, ids)
    detail["wall_s"] = round(time.perf_counter() - t_start, 1)

    if rank == 0:
        line = compact_line(wl, world, steps, warmup, len(ids), ms_dev, value, ms_e2e, e2e_value, dev_arm, e2e_arm, clocks, detail, args.out, pk)
        detail["line"] = line
        try:
            with open(args.out, "w") as f:
                json.dump(detail, f, indent=1)
            log(f"[bench] detail written to {args.out} ({detail['wall_s']} s)")
        except OSError as e:
            log(f"[bench] could not write {args.out}: {e}")
        s = json.dumps(line, separators=(",", ":"))
        print(s, flush=True)
    multi.barrier(dev)
    return 0


SIDE_CONFIGS = (0, 1, 2, 3, 4, 5, 6)  # BASELINE.json:configs[0..4] and the two paper workloads of SURVEY.md 8(f)4

if __name__ == "__main__":
    sys.exit(main())
