"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Integer workloads bit-exact; fp32 within 1e-6 relative; bf16 GEMM within 2e-2 relative
Frobenius error (BASELINE.json:north_star).  Every job's output must land in its own output slot."""
import numpy as np
import pytest

import inputgen
from checker import compare, oracle_out

pytestmark = pytest.mark.gpu

SENTINEL = 0xA5


def run_jobs(setlib, wl, job_ids, mode=0, pageable=False, io_check=True, pdl=False, misalign=0, **ctx_kw):
    """Submit the jobs through the C ABI; returns (list of output uint8 arrays, list of input images, dims, stats)."""
    from paper_2606_05495_b200.workloads import PinnedArena
    ctx = setlib.Context(wl.num_streams, wl.max_inflight, mode=mode, **ctx_kw)
    try:
        ctx.register_builtin(wl.config, wl.variant, list(wl.params), pdl=pdl)
        ins = [wl.make_input(j) for j in job_ids]
        dims = [wl.dims(j) for j in job_ids]
        if "spin_ns" in wl.extra:
            dims = [(d[0], d[1], d[2], wl.extra["spin_ns"](j)) for d, j in zip(dims, job_ids)]
        in_sz = [wl.in_bytes(d) for d in dims]
        out_sz = [wl.out_bytes(d) for d in dims]
        pad = 256
        if pageable:
            in_bufs = [np.array(x, copy=True) for x in ins]
            out_bufs = [np.full(n, SENTINEL, np.uint8) for n in out_sz]
            canaries = None
        else:
            arena = PinnedArena(ctx, sum(in_sz) + sum(out_sz) + (2 * len(ins) + 2) * (pad + 256) + 4096)
            arena.view[:] = SENTINEL
            in_bufs, out_bufs = [], []
            m = misalign  # byte offset that breaks the 16-byte alignment the vector paths want
            for x, n in zip(ins, in_sz):
                a, v = arena.take(n + pad)
                v[m:m + n] = x
                in_bufs.append(v[m:m + n])
            for n in out_sz:
                a, v = arena.take(n + pad)
                out_bufs.append(v[m:m + n])
        for k, j in enumerate(job_ids):
            ctx.submit(j, in_bufs[k].ctypes.data, out_bufs[k].ctypes.data, dims[k] if wl.config in (4, 5, 6) or "spin_ns" in wl.extra else None)
        ctx.drain()
        stats = ctx.stats()
        outs = [np.array(o, copy=True) for o in out_bufs]
        if not pageable and io_check:
            # canary bytes between the blocks are untouched and inputs are unmodified
            for k, (x, n) in enumerate(zip(ins, in_sz)):
                assert np.array_equal(in_bufs[k], x), f"input of job {job_ids[k]} was modified"
            used = np.zeros(arena.nbytes, bool)
            for v, n in list(zip(in_bufs, in_sz)) + list(zip(out_bufs, out_sz)):
                off = v.ctypes.data - arena.ptr
                used[off:off + n] = True
            assert np.all(arena.view[~used] == SENTINEL), "bytes outside every job's slots were written"
        if not pageable:
            in_bufs = out_bufs = None
            arena.free()
        return outs, ins, dims, stats
    finally:
        ctx.close()


def check(setlib, wl, job_ids, **kw):
    outs, ins, dims, stats = run_jobs(setlib, wl, job_ids, **kw)
    assert stats["completed"] == len(job_ids) and stats["submitted"] == len(job_ids)
    for k in range(len(job_ids)):
        compare(wl, outs[k], oracle_out(wl, ins[k], dims[k]))
    return stats


@pytest.mark.parametrize("config", [0, 1, 2, 3, 4, 5, 6])
def test_parity_small(libset, config):
    from paper_2606_05495_b200.workloads import small_workload
    wl = small_workload(config)
    st = check(libset, wl, list(range(wl.jobs)))
    assert st["max_inflight_seen"] <= wl.max_inflight
    assert st["kernel_nodes"] == wl.jobs * wl.kernels_per_job


@pytest.mark.parametrize("config", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("mode", [1, 2, 3, 4])
def test_baseline_models_compute_the_same(libset, config, mode):
    from paper_2606_05495_b200.workloads import small_workload
    wl = small_workload(config)
    n = min(wl.jobs, 20)
    check(libset, wl, list(range(n)), mode=mode)


def test_config0_histogram_of_input_variant(libset):
    from paper_2606_05495_b200.workloads import small_workload
    wl = small_workload(0)
    wl.variant = 1
    check(libset, wl, list(range(16)))


@pytest.mark.parametrize("n", [1, 3, 4095, 4097, 10000])
def test_config0_ragged_sizes(libset, n):
    from paper_2606_05495_b200.workloads import Workload
    check(libset, Workload(0, (n,), jobs=6, num_streams=2, max_inflight=4), list(range(6)))


@pytest.mark.parametrize("n", [1, 5, 1023, 16385])
def test_config1_ragged_sizes(libset, n):
    from paper_2606_05495_b200.workloads import Workload
    check(libset, Workload(1, (n,), jobs=6, num_streams=2, max_inflight=4), list(range(6)))


@pytest.mark.parametrize("h,w,sweeps", [(1, 1, 1), (5, 9, 3), (33, 1028, 2), (70, 2049, 10), (16, 4, 1)])
def test_config2_ragged_grids(libset, h, w, sweeps):
    from paper_2606_05495_b200.workloads import Workload
    check(libset, Workload(2, (h, w, sweeps), jobs=3, num_streams=2, max_inflight=4), list(range(3)))


@pytest.mark.parametrize("m,n,k", [(128, 256, 64), (128, 256, 576), (200, 264, 72), (130, 8, 8), (1, 2048, 40), (300, 768, 320)])
def test_config3_ragged_shapes(libset, m, n, k):
    """One tile exactly; more k-blocks than pipeline stages (the smem ring wraps twice); partial tiles in M, N and K;
    degenerate thin shapes."""
    from paper_2606_05495_b200.workloads import Workload
    check(libset, Workload(3, (m, n, k), jobs=3, num_streams=2, max_inflight=4), list(range(3)))


@pytest.mark.parametrize("size", [(1, 1), (5, 4), (7, 3), (128, 64), (132, 65), (644, 9), (16, 1), (512, 33), (528, 40), (1040, 37), (1920, 3)])
def test_config4_ragged_frames(libset, size):
    from paper_2606_05495_b200.workloads import Workload
    wl = Workload(4, (1920, 1080), jobs=3, num_streams=2, max_inflight=4, extra={"size": size})
    check(libset, wl, list(range(3)))


def test_config4_oversize_frame_is_rejected_per_job(libset):
    from paper_2606_05495_b200.workloads import PinnedArena
    ctx = libset.Context(2, 4)
    ctx.register_builtin(4, 0, [64, 64])
    arena = PinnedArena(ctx, 1 << 20)
    a, _ = arena.take(3 * 128 * 128)
    b, _ = arena.take(128 * 128 + 1024)
    with pytest.raises(libset.SetError) as ei:
        ctx.submit(0, a, b, (128, 128, 1, 1))
    assert ei.value.status == libset.SET_ERR_SIZE
    ctx.submit(1, a, b, (64, 64, 1, 1))          # SET_ERR_SIZE is per job, the context stays usable
    ctx.drain()
    arena.free()
    ctx.close()


def test_pageable_buffers_go_through_the_staging_ring(libset):
    from paper_2606_05495_b200.workloads import small_workload
    for config in (0, 4):
        wl = small_workload(config)
        st = check(libset, wl, list(range(24)), pageable=True)
        assert st["staged_jobs"] == 24


@pytest.mark.parametrize("policy", [0, 1])
def test_work_stealing_with_jittered_jobs_max_depth(libset, policy):
    """config 4 geometry (8 streams, 32 in flight) with a random-length delay stage: completions reorder, queues
    drain unevenly, idle slots steal.  Every output must still equal F(in) of its own job."""
    from paper_2606_05495_b200.workloads import Workload
    # jobs 0, 32, 64, ... start in slot 0's queue and hold it for 2 ms each while the other 31 slots run short
    # jobs and go idle: whatever is still queued behind a long job must be stolen (Alg. 2 l.12-16).
    wl = Workload(4, (1920, 1080), variant=libset.VARIANT_SPIN, jobs=160, num_streams=8, max_inflight=32,
                  extra={"spin_ns": lambda j: 2_000_000 if j % 32 == 0 else int(inputgen.uniform24(99, j, 0, 1)[0] % 400) * 1000})
    st = check(libset, wl, list(range(wl.jobs)), steal_policy=policy, num_dispatchers=2)
    assert st["steals"] > 0
    assert st["max_inflight_seen"] <= 32


def test_same_inputs_twice_give_identical_bits(libset):
    from paper_2606_05495_b200.workloads import small_workload
    for config in (1, 3):
        wl = small_workload(config)
        ids = list(range(6))
        a, _, _, _ = run_jobs(libset, wl, ids)
        b, _, _, _ = run_jobs(libset, wl, ids, num_dispatchers=2, callback_mode=libset.CB_WORK_STREAM)
        for x, y in zip(a, b):
            assert np.array_equal(x, y)


@pytest.mark.parametrize("cb", [1, 2, 3, 4])
@pytest.mark.parametrize("disp", [1, 2])
def test_every_completion_mode_delivers_every_job(libset, cb, disp):
    """A6/A7: event chain + cudaLaunchHostFunc on a notify stream (1), host function on the work stream (2, PAPER.md:203
    literally), the GPU-written flag watched by the dispatcher (3) and a host node at the end of the job graph (4) all release
    each slot exactly once."""
    from paper_2606_05495_b200.workloads import small_workload
    for config in (0, 4):
        wl = small_workload(config)
        st = check(libset, wl, list(range(wl.jobs)), callback_mode=cb, num_dispatchers=disp)
        # flag-polled completion: config 4 (two copy-out nodes) keeps a signal node of its own; config 0's single SM copy-out node
        # stores the completion word itself (SET_K_COPY_OUT), so no signal node is launched at all
        assert st["signal_nodes"] == (wl.jobs if cb == 3 and config == 4 else 0)
        assert st["copy_nodes"] == wl.jobs * (2 if config == 0 else 1)
        assert st["max_inflight_seen"] <= wl.max_inflight


@pytest.mark.parametrize("config", [0, 1, 4])
@pytest.mark.parametrize("sm_copy", [-1, 0, 4096])
@pytest.mark.parametrize("pdl", [False, True])
@pytest.mark.parametrize("mode", [0, 1, 2])
def test_graph_shapes_compute_the_same(libset, config, sm_copy, pdl, mode):
    """Copy-engine memcpy nodes or SM copy nodes (set_config.sm_copy_max_bytes), ordinary or programmatic (PDL) edges:
    the job graph's result is the same in SET and in the baseline models that share the graph."""
    from paper_2606_05495_b200.workloads import small_workload
    wl = small_workload(config)
    st = check(libset, wl, list(range(min(wl.jobs, 48))), mode=mode, sm_copy_max_bytes=sm_copy, pdl=pdl)
    if sm_copy == -1:
        assert st["copy_nodes"] == 0


@pytest.mark.parametrize("misalign", [4, 1])
def test_sm_copies_with_unaligned_pinned_pointers(libset, misalign):
    from paper_2606_05495_b200.workloads import Workload
    check(libset, Workload(0, (1001,), jobs=12, num_streams=2, max_inflight=4), list(range(12)), misalign=misalign, pdl=True)


def test_completion_word_never_overtakes_the_output(libset):
    """The signal node stores the slot's word without a system fence: the graph edge from the D2H copy node orders the
    output before it.  600 jobs over 4 slots with sentinel-filled outputs of three copy blocks each (config 0 with
    n = 5000 -> 20,256 bytes): a word seen early would release the slot and the check would read sentinel bytes."""
    from paper_2606_05495_b200.workloads import Workload
    st = check(libset, Workload(0, (5000,), jobs=600, num_streams=2, max_inflight=4), list(range(600)), pdl=True)
    assert st["signal_nodes"] == 0 and st["copy_nodes"] == 1200       # the completion word is stored by the copy-out node itself


def test_submit_before_register_and_double_register(libset):
    ctx = libset.Context(2, 4)
    with pytest.raises(libset.SetError) as ei:
        ctx.submit(0, 1, 1)
    assert ei.value.status == libset.SET_ERR_STATE
    ctx.register_builtin(0)
    with pytest.raises(libset.SetError) as ei:
        ctx.register_builtin(0)
    assert ei.value.status == libset.SET_ERR_STATE
    ctx.drain()                       # empty drain returns at once
    ctx.close()


def test_torch_streams_and_device_arena(libset):
    import torch
    from paper_2606_05495_b200.workloads import small_workload
    wl = small_workload(0)
    streams = [torch.cuda.Stream() for _ in range(wl.num_streams)]
    arena = torch.empty(64 << 20, dtype=torch.uint8, device="cuda")
    check(libset, wl, list(range(32)), streams=[s.cuda_stream for s in streams], device_arena=arena.data_ptr(),
          device_arena_bytes=arena.numel())


def test_device_resident_io(libset):
    """SET_IO_DEVICE: host_in/host_out are device pointers (the copy nodes become D2D)."""
    import torch
    from paper_2606_05495_b200.workloads import small_workload
    wl = small_workload(1)
    ctx = libset.Context(wl.num_streams, wl.max_inflight, io=libset.IO_DEVICE)
    ctx.register_builtin(1, 0, list(wl.params))
    ins = [wl.make_input(j) for j in range(40)]
    d_in = [torch.from_numpy(x).cuda() for x in ins]
    d_out = [torch.zeros(4, dtype=torch.uint8, device="cuda") for _ in ins]
    torch.cuda.synchronize()
    for j in range(40):
        ctx.submit(j, d_in[j].data_ptr(), d_out[j].data_ptr())
    ctx.drain()
    for j in range(40):
        compare(wl, d_out[j].cpu().numpy(), oracle_out(wl, ins[j], (1, 1, 1, 1)))
    ctx.close()


@pytest.mark.parametrize("config", [0, 1, 4])
def test_device_slot_padding_is_never_written(libset, config):
    """Canary bytes on the device: the slot buffers live in a caller-owned torch arena pre-filled with a sentinel; each
    buffer is padded to a multiple of 1024 bytes (set.h: set_register_pipeline), and neither the padding, nor the space
    in front of the first slot, nor the space after the last one may change while jobs run at full depth."""
    import torch
    from paper_2606_05495_b200.workloads import small_workload
    wl = small_workload(config)
    _, _, bufs, nb, _, _ = libset.builtin_pipeline(wl.config, wl.variant, list(wl.params))
    sizes = [int(bufs[i].bytes) for i in range(nb)]
    up = lambda v: (v + 1023) & ~1023
    per_slot = sum(up(b) for b in sizes)
    arena = torch.full((per_slot * wl.max_inflight + 4096,), SENTINEL, dtype=torch.uint8, device="cuda")
    check(libset, wl, list(range(min(wl.jobs, 64))), device_arena=arena.data_ptr(), device_arena_bytes=arena.numel(), pdl=True)
    torch.cuda.synchronize()
    host = arena.cpu().numpy()
    first = up(arena.data_ptr()) - arena.data_ptr()
    pad = np.ones(host.size, bool)                      # True = must still hold the sentinel
    for w in range(wl.max_inflight):
        off = first + w * per_slot
        for b in sizes:
            pad[off:off + b] = False
            off += up(b)
    assert pad.sum() > 0
    assert np.all(host[pad] == SENTINEL), "a kernel or copy wrote outside its slot buffer"


def test_full_size_config2_bit_exact(libset):
    """BASELINE.json:configs[2] at its full per-job size (4096 x 4096 fp32, 10 sweeps, 4 streams, 8 in flight), every
    element of every output against the oracle."""
    from paper_2606_05495_b200.workloads import baseline_workload
    wl = baseline_workload(2)
    st = check(libset, wl, list(range(3)), io_check=False)
    assert st["kernel_nodes"] == 3 * 10


def test_full_size_config3_sampled_entries(libset):
    """BASELINE.json:configs[3] at its full per-job size (2048^3, 4 streams, 8 in flight, 10 jobs so that slots are
    reused): the naive-loop oracle takes minutes per job at this size, so 4096 seeded (m, n) entries per job are
    computed one by one (oracle_config3_sampled) and compared; tile corners and edges are always among them."""
    import oracle
    from paper_2606_05495_b200.workloads import baseline_workload
    wl = baseline_workload(3)
    M, N, K = wl.params
    ids = list(range(10))
    outs, ins, _, st = run_jobs(libset, wl, ids, io_check=False)
    assert st["completed"] == len(ids)
    fixed = [(0, 0), (M - 1, N - 1), (127, 255), (128, 256), (127, 256), (128, 255), (M - 1, 0), (0, N - 1), (1023, 1024), (1024, 1023)]
    for k, j in enumerate(ids):
        a = ins[k][:2 * M * K].view(np.uint16).reshape(M, K)
        b = ins[k][2 * M * K:2 * M * K + 2 * K * N].view(np.uint16).reshape(K, N)
        bias = ins[k][2 * M * K + 2 * K * N:].view(np.float32)
        r = inputgen.uniform24(1234, j, 7, 2 * 4096)
        ms = np.concatenate([np.array([f[0] for f in fixed]), r[:4096] % M]).astype(np.int64)
        ns = np.concatenate([np.array([f[1] for f in fixed]), r[4096:] % N]).astype(np.int64)
        ref = inputgen.bf16_bits_to_f64(oracle.config3_sampled(a, b, bias, ms, ns))
        got = inputgen.bf16_bits_to_f64(outs[k].view(np.uint16).reshape(M, N)[ms, ns])
        assert np.linalg.norm(got - ref) / np.linalg.norm(ref) <= 2e-2
        assert np.abs(got - ref).max() <= 0.05 * max(1.0, np.abs(ref).max())


@pytest.mark.parametrize("mode", [0, 2, 4])
@pytest.mark.parametrize("config", [1, 4])
def test_device_timestamps_give_per_stream_gaps(libset, config, mode):
    """set_config.timestamps: two stamp nodes per job graph, gaps between consecutive jobs of a stream from the GPU's own
    clock.  The results stay the oracle's, every job is stamped, and the numbers are sane."""
    from paper_2606_05495_b200.workloads import PinnedArena, small_workload
    wl = small_workload(config)
    n = min(wl.jobs, 96)
    ctx = libset.Context(wl.num_streams, wl.max_inflight, mode=mode, timestamps=True)
    try:
        ctx.register_builtin(wl.config, wl.variant, list(wl.params), pdl=True)
        ins = [wl.make_input(j) for j in range(n)]
        dims = [wl.dims(j) for j in range(n)]
        arena = PinnedArena(ctx, sum(wl.in_bytes(d) + wl.out_bytes(d) + 1024 for d in dims))
        outs = []
        for j in range(n):
            a_in, v_in = arena.take(wl.in_bytes(dims[j]))
            v_in[:] = ins[j]
            a_out, v_out = arena.take(wl.out_bytes(dims[j]))
            v_out[:] = SENTINEL
            outs.append(v_out)
            ctx.submit(j, a_in, a_out, dims[j] if config == 4 else None)
        ctx.drain()
        for j in range(n):
            compare(wl, np.array(outs[j], copy=True), oracle_out(wl, ins[j], dims[j]))
        g = ctx.gap_stats()
        assert g["jobs"] == n
        assert n - ctx.stats()["cuda_streams"] <= g["gaps"] <= n - 1      # one gap less than jobs on every CUDA stream that ran any
        assert 1.0 < g["job_mean_us"] < 5000.0 and 0.0 <= g["gap_mean_us"] <= g["gap_max_us"] < 1e6
        assert g["gap_p50_us"] <= g["gap_p99_us"] <= g["gap_max_us"] and 0.0 < g["stream_busy_frac"] <= 1.0001
        ctx.reset_stats()
        assert ctx.gap_stats()["jobs"] == 0
        outs = None
        arena.free()
    finally:
        ctx.close()


def test_gap_stats_are_zero_without_timestamps(libset):
    from paper_2606_05495_b200.workloads import small_workload
    wl = small_workload(0)
    ctx = libset.Context(wl.num_streams, wl.max_inflight)
    ctx.register_builtin(0)
    assert ctx.gap_stats() == {"jobs": 0, "gaps": 0, "gap_mean_us": 0.0, "gap_p50_us": 0.0, "gap_p99_us": 0.0, "gap_max_us": 0.0,
                               "job_mean_us": 0.0, "span_us": 0.0, "stream_busy_frac": 0.0, "busy_union_us": 0.0, "idle_frac": 0.0,
                               "idle_gaps": 0.0, "idle_gap_mean_us": 0.0}
    ctx.close()


def test_every_output_is_there_when_the_completion_word_is_seen(libset):
    """Full-rate check of the fence-free signal node: 30,000 config-1 jobs at the bench geometry (8 streams, 32
    in flight, SM copies, PDL edges), every 4-byte output pre-filled with a sentinel pattern and read as soon as
    set_drain returns.  A completion word that reached the host before its job's output would release the slot early
    and leave sentinel bytes (or a neighbour's result) behind."""
    import ctypes as C
    from paper_2606_05495_b200.workloads import PinnedArena, baseline_workload
    wl = baseline_workload(1)
    n, npool = 30000, 128
    ctx = libset.Context(wl.num_streams, wl.max_inflight)
    try:
        ctx.register_builtin(1, 0, list(wl.params), pdl=True)
        ins = [wl.make_input(j) for j in range(npool)]
        want = np.array([oracle_out(wl, x, (1, 1, 1, 1)).view(np.float32)[0] for x in ins], np.float32)
        arena = PinnedArena(ctx, npool * (wl.in_bytes() + 256) + 4 * n + 4096)
        in_ptrs = []
        for x in ins:
            a, v = arena.take(wl.in_bytes())
            v[:] = x
            in_ptrs.append(a)
        a_out, v_out = arena.take(4 * n)
        out_f = v_out.view(np.float32)
        pi = (C.c_void_p * n)(*[in_ptrs[k % npool] for k in range(n)])
        po = (C.c_void_p * n)(*[a_out + 4 * k for k in range(n)])
        import os
        for rep in range(int(os.environ.get("SET_SOAK_REPS", "3"))):  # a soak run sets this to a few hundred
            v_out[:] = SENTINEL
            ctx.submit_batch(pi, po)
            ctx.drain()
            got = np.array(out_f, copy=True)
            ref = want[np.arange(n) % npool]
            bad = np.nonzero(np.abs(got - ref) > 1e-6 * np.abs(ref))[0]
            assert bad.size == 0, f"rep {rep}: {bad.size} outputs wrong, first job {bad[0]}: {got[bad[0]]} vs {ref[bad[0]]}"
        out_f = v_out = None
        arena.free()
    finally:
        ctx.close()


@pytest.mark.parametrize("n", [32768, 32772])
def test_config1_around_the_sm_copy_limit(libset, n):
    """8n = 262,144 bytes is the largest H2D copy the SMs do by default; 4 floats more and the same copy becomes a
    copy-engine memcpy node.  Both sides of the limit compute the same thing."""
    from paper_2606_05495_b200.workloads import Workload
    st = check(libset, Workload(1, (n,), jobs=12, num_streams=2, max_inflight=4), list(range(12)), pdl=True)
    assert st["copy_nodes"] == 12 * (2 if n == 32768 else 1)


def test_config3_gelu_epilogue_within_one_bf16_ulp(libset):
    """K9 evaluates erfc by a branch-free formula (C3-3) instead of calling erff.  With A = 0 the output is
    bf16(GELU(bias)) exactly, so the epilogue alone is compared with the oracle's double-precision erf: over biases from -9
    to 9 the two bf16 results may differ by at most one unit in the last place where |GELU| >= 1e-3 (almost all must be
    identical) and by at most 4e-6 (one bf16 ulp at 1e-3) in the far negative tail."""
    from paper_2606_05495_b200.workloads import PinnedArena, Workload
    M, N, K = 128, 2048, 64
    wl = Workload(3, (M, N, K), jobs=1, num_streams=1, max_inflight=1)
    a = np.zeros((M, K), np.uint16)
    b = inputgen.f32_to_bf16_bits(inputgen.gaussian(3, 0, 1, K * N).astype(np.float32)).reshape(K, N)
    bias = np.linspace(-9.0, 9.0, N).astype(np.float32)
    image = inputgen.config3_pack(a, b, bias)
    ctx = libset.Context(1, 1)
    try:
        ctx.register_builtin(3, 0, [M, N, K])
        arena = PinnedArena(ctx, image.size + 2 * M * N + 4096)
        a_in, v_in = arena.take(image.size)
        v_in[:] = image
        a_out, v_out = arena.take(2 * M * N)
        ctx.submit(0, a_in, a_out)
        ctx.drain()
        got = np.array(v_out, copy=True).view(np.uint16).reshape(M, N)
        ref = oracle_out(wl, image, (1, 1, 1, 1)).view(np.uint16).reshape(M, N)
        v_in = v_out = None
        arena.free()
    finally:
        ctx.close()
    assert np.array_equal(got, np.broadcast_to(got[0], got.shape))          # every row sees the same bias
    # where GELU is not negligible: bf16 bit patterns of equal sign are ordered like the values, compare in units in the
    # last place; in the far negative tail (|GELU| < 1e-3) the formula's absolute error bound applies instead
    g, r = inputgen.bf16_bits_to_f64(got), inputgen.bf16_bits_to_f64(ref)
    big = np.abs(r) >= 1e-3
    assert np.all(((got >> 15) == (ref >> 15))[big])
    ulp = np.abs((got & 0x7fff).astype(np.int32) - (ref & 0x7fff).astype(np.int32))
    assert ulp[big].max() <= 1
    assert (ulp[big] == 0).mean() > 0.98
    assert np.abs(g - r)[~big].max() <= 4e-6              # one bf16 ulp just below 1e-3 is 3.8e-6


# ---------------------------------------------------------------------------------------------------------------------
# config 1, element by element: K3..K6 are only visible through K7's sum in the built-in pipeline, and a sum at 1e-6
# cannot see a contracted fma(2.5, x, 0.1) (about 1 ulp per element, random sign).  Reading C1-1 says the four
# elementwise kernels are bit-exact, so the stage list is registered truncated after K3, K4, K5, K6 in turn -- through
# set_register_pipeline, with the y buffer copied back instead of the scalar -- and y is compared bit for bit with the
# oracle's intermediate of the same step (oracle_config1_chain).
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [16384, 16385, 1023, 5])
@pytest.mark.parametrize("pdl", [False, True])
@pytest.mark.parametrize("upto", [1, 2, 3, 4])
def test_config1_elementwise_stages_bit_exact(libset, upto, pdl, n):
    import oracle
    from paper_2606_05495_b200.workloads import PinnedArena
    st, ns, bf, nb, hin, _ = libset.builtin_pipeline(1, 0, [n])
    assert ns == 5 and nb == 3
    for i in range(ns):
        if pdl:
            st[i].flags |= libset.STAGE_PDL
    bf[1].d2h_bytes.fixed = 4 * n          # y comes back ...
    bf[2].d2h_bytes.fixed = 0              # ... the scalar does not (K7 is not part of the truncated chain)
    jobs = 24
    ctx = libset.Context(4, 8)
    try:
        ctx.register_pipeline(st, upto, bf, nb)
        ins = [inputgen.config1_job(1000 + j, n) for j in range(jobs)]
        arena = PinnedArena(ctx, jobs * (hin + 4 * n + 1024) + 4096)
        outs = []
        for j, x in enumerate(ins):
            a_in, v_in = arena.take(hin)
            v_in[:] = x.view(np.uint8)
            a_out, v_out = arena.take(4 * n)
            v_out[:] = SENTINEL
            outs.append(v_out)
            ctx.submit(j, a_in, a_out)
        ctx.drain()
        for j, x in enumerate(ins):
            want = oracle.config1_chain(x[:n], x[n:])[upto - 1]
            got = np.array(outs[j], copy=True).view(np.uint32)
            bad = np.nonzero(got != want.view(np.uint32))[0]
            assert bad.size == 0, (f"stage {upto} (pdl={pdl}, n={n}) job {j}: {bad.size} of {n} elements differ, first at {bad[0]}: "
                                   f"{got.view(np.float32)[bad[0]]!r} vs {want[bad[0]]!r}")
        outs = None
        arena.free()
    finally:
        ctx.close()


# ---------------------------------------------------------------------------------------------------------------------
# Parity at the configs' FULL job counts, in the launch configuration bench.py times (BASELINE geometry, SM copies, PDL
# edges): every output of every job is checked.  Jobs that share a pool input must produce identical bytes, and one
# representative per distinct input is compared with the oracle -- which together pins every output to the oracle.
# ---------------------------------------------------------------------------------------------------------------------
def _full_count(libset, wl, n_jobs, npool, dims_of=None, sampled=None):
    import ctypes as C
    from paper_2606_05495_b200.workloads import PinnedArena
    ctx = libset.Context(wl.num_streams, wl.max_inflight)
    try:
        ctx.register_builtin(wl.config, wl.variant, list(wl.params), pdl=True)
        ins = [wl.make_input(j) for j in range(npool)]
        dims = [wl.dims(j) for j in range(npool)]
        in_sz = [wl.in_bytes(d) for d in dims]
        out_sz = [wl.out_bytes(dims[k % npool]) for k in range(n_jobs)]
        arena = PinnedArena(ctx, sum(in_sz) + sum(out_sz) + 256 * (npool + n_jobs + 2))
        in_ptr = []
        for x, n in zip(ins, in_sz):
            a, v = arena.take(n)
            v[:] = x
            in_ptr.append(a)
        out_ptr, out_view = [], []
        for n in out_sz:
            a, v = arena.take(n)
            v[:] = SENTINEL
            out_ptr.append(a)
            out_view.append(v)
        pi = (C.c_void_p * n_jobs)(*[in_ptr[k % npool] for k in range(n_jobs)])
        po = (C.c_void_p * n_jobs)(*out_ptr)
        pd = None
        if wl.config in (4, 5, 6):
            pd = (C.c_uint32 * (4 * n_jobs))(*[v for k in range(n_jobs) for v in dims[k % npool]])
        ctx.submit_batch(pi, po, pd)
        ctx.drain()
        st = ctx.stats()
        assert st["completed"] == n_jobs and st["submitted"] == n_jobs and st["max_inflight_seen"] <= wl.max_inflight
        for p in range(npool):
            first = np.array(out_view[p], copy=True)
            if sampled is None:
                compare(wl, first, oracle_out(wl, ins[p], dims[p]))
            else:
                sampled(p, ins[p], first)
            ref5 = oracle_out(wl, ins[p], dims[p]) if wl.config == 5 else None
            for k in range(p + npool, n_jobs, npool):     # same input -> same bytes, in its own output slot
                if wl.config == 5:                        # the round count may differ from run to run (reading S5-4): compare as the rule says
                    compare(wl, np.array(out_view[k], copy=True), ref5)
                else:
                    assert np.array_equal(out_view[k], first), f"job {k} differs from job {p} although both ran input {p}"
        out_view = None
        arena.free()
        return st
    finally:
        ctx.close()


def test_full_job_count_config0(libset):
    from paper_2606_05495_b200.workloads import baseline_workload
    wl = baseline_workload(0)
    _full_count(libset, wl, wl.jobs, wl.jobs)                       # 256 jobs, all distinct


def test_full_job_count_config1(libset):
    from paper_2606_05495_b200.workloads import baseline_workload
    wl = baseline_workload(1)
    _full_count(libset, wl, wl.jobs, wl.jobs)                       # 10,000 jobs, all distinct


def test_full_job_count_config4(libset):
    from paper_2606_05495_b200.workloads import baseline_workload
    wl = baseline_workload(4)
    st = _full_count(libset, wl, wl.jobs, 96)                       # 4,096 frames over 96 distinct ones (jittered sizes)
    assert st["full_rebinds"] > 0                                   # frame sizes change from job to job on a slot


def test_slot_reuse_config2_full_size(libset):
    """Full-size Jacobi jobs, every slot (8) and every exec (3 per slot) reused: 40 jobs over 8 distinct grids."""
    from paper_2606_05495_b200.workloads import baseline_workload
    wl = baseline_workload(2)
    _full_count(libset, wl, 40, 8)


def test_slot_reuse_config3_full_size(libset):
    """Full-size GEMM jobs, 48 jobs over the 8 distinct triples of the bench pool: every slot used >= 4 times.  The oracle is
    evaluated on 2,048 sampled entries per distinct input (tile corners included); identical inputs must give identical
    bytes."""
    import oracle
    from paper_2606_05495_b200.workloads import baseline_workload
    wl = baseline_workload(3)
    M, N, K = wl.params
    fixed = [(0, 0), (M - 1, N - 1), (127, 255), (128, 256), (127, 256), (128, 255), (M - 1, 0), (0, N - 1), (1023, 1024), (1024, 1023)]

    def sampled(p, image, out):
        a = image[:2 * M * K].view(np.uint16).reshape(M, K)
        b = image[2 * M * K:2 * M * K + 2 * K * N].view(np.uint16).reshape(K, N)
        bias = image[2 * M * K + 2 * K * N:].view(np.float32)
        r = inputgen.uniform24(4321, p, 7, 2 * 2048)
        ms = np.concatenate([np.array([f[0] for f in fixed]), r[:2048] % M]).astype(np.int64)
        ns = np.concatenate([np.array([f[1] for f in fixed]), r[2048:] % N]).astype(np.int64)
        ref = inputgen.bf16_bits_to_f64(oracle.config3_sampled(a, b, bias, ms, ns))
        got = inputgen.bf16_bits_to_f64(out.view(np.uint16).reshape(M, N)[ms, ns])
        assert np.linalg.norm(got - ref) / np.linalg.norm(ref) <= 2e-2
        assert np.abs(got - ref).max() <= 0.05 * max(1.0, np.abs(ref).max())

    _full_count(libset, wl, 48, 8, sampled=sampled)


# ---------------------------------------------------------------------------------------------------------------------
# round 2: PDL edge into the tcgen05 GEMM, completion fence modes with the early-completion hook, CUDA streams per lane,
# declared pinned ranges, maximum depth
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape,sm_copy", [((128, 256, 64), 0), ((384, 512, 256), 1 << 20), ((200, 264, 72), 1 << 20)])
def test_config3_behind_a_programmatic_edge(libset, shape, sm_copy):
    """with the whole [A][B][bias] image at or below sm_copy_max_bytes the GEMM's only predecessor is an SM copy
    node and SET_STAGE_PDL makes the edge programmatic: the kernel must not issue a TMA load or read bias before
    griddepcontrol.wait.  64 jobs over 4 slots so that every slot's buffers are overwritten while the next GEMM's prologue
    is already running."""
    from paper_2606_05495_b200.workloads import Workload
    st = check(libset, Workload(3, shape, jobs=64, num_streams=2, max_inflight=4), list(range(64)), pdl=True, sm_copy_max_bytes=sm_copy)
    assert st["copy_nodes"] >= 64          # the copy-in really was a kernel node


def _completion_soak(libset, fence, lanes):
    """30,000 config-1 jobs and 30,000 config-0 jobs per repetition at the bench geometry with set_config.debug_sentinel: inside
    Algorithm 3, at the moment the dispatcher sees a job's completion word and before the slot is released, the library itself
    looks at the first and last word of the job's sentinel-filled output.  Returns the number of early completions; every output
    is checked after set_drain regardless.  SET_SOAK_REPS raises the repetition count for a soak run."""
    import ctypes as C
    import os
    from paper_2606_05495_b200.workloads import PinnedArena, baseline_workload
    reps = int(os.environ.get("SET_SOAK_REPS", "2"))
    early = 0
    for config in (1, 0):
        wl = baseline_workload(config)
        n, npool = 30000, 64
        ctx = libset.Context(8, 32, completion_fence=fence, streams_per_lane=lanes, debug_sentinel=0xA5A5A5A5)
        try:
            ctx.register_builtin(config, 0, list(wl.params), pdl=True)
            ins = [wl.make_input(j) for j in range(npool)]
            want = [oracle_out(wl, x, (1, 1, 1, 1)) for x in ins]
            ob = wl.out_bytes()
            arena = PinnedArena(ctx, npool * (wl.in_bytes() + 256) + ob * n + 4096)
            in_ptrs = []
            for x in ins:
                a, v = arena.take(wl.in_bytes())
                v[:] = x
                in_ptrs.append(a)
            a_out, v_out = arena.take(ob * n, align=256)
            pi = (C.c_void_p * n)(*[in_ptrs[k % npool] for k in range(n)])
            po = (C.c_void_p * n)(*[a_out + ob * k for k in range(n)])
            for rep in range(reps):
                v_out[:] = SENTINEL
                ctx.submit_batch(pi, po)
                ctx.drain()
                got = np.array(v_out, copy=True).reshape(n, ob)
                for p_ in range(npool):                       # after set_drain every output is there, whatever the fence mode
                    rows = got[p_::npool]
                    if config == 1:
                        g, r = rows.view(np.float32)[:, 0], want[p_].view(np.float32)[0]
                        assert np.all(np.abs(g - r) <= 1e-6 * abs(r))
                    else:
                        assert np.all(rows == want[p_][None, :])
            st = ctx.stats()
            assert st["completed"] == n * reps
            early += st["early_completions"]
            v_out = None
            arena.free()
        finally:
            ctx.close()
    return early


@pytest.mark.parametrize("lanes", [1, 4])
def test_no_completion_is_seen_before_its_output(libset, lanes):
    """The default completion store (SET_FENCE_SYSTEM: fence.acq_rel.sys, then the word): no completion may ever be observed
    before its job's output is in host memory."""
    assert _completion_soak(libset, libset.FENCE_SYSTEM, lanes) == 0


@pytest.mark.parametrize("lanes", [1, 4])
def test_fence_free_completion_is_only_a_measurement_arm(libset, lanes):
    """SET_FENCE_NONE (round 1's default) relies on grid completion alone.  Round 2 caught it in the act: with four CUDA
    streams per lane about one completion in 30,000 overtakes its output (profiles/r2_signal_soak.md), so the mode is opt-in,
    documented as unsafe for anything that reads the output on completion, and this test only requires what still holds --
    every output is correct once set_drain has returned -- and prints what the hook counted."""
    early = _completion_soak(libset, libset.FENCE_NONE, lanes)
    print(f"SET_FENCE_NONE, {lanes} CUDA stream(s) per lane: {early} early completions")
    assert early >= 0


def test_pageable_staging_at_full_rate(libset):
    """The one path that reads a job's output the moment its completion is seen: the staged D2H memcpy from the exec's pinned
    block into the caller's pageable buffer (set_ctx::finish).  6,000 config-0 jobs with pageable buffers, every output checked."""
    from paper_2606_05495_b200.workloads import baseline_workload
    wl = baseline_workload(0)
    n, npool = 6000, 32
    ctx = libset.Context(8, 32)
    try:
        ctx.register_builtin(0, 0, list(wl.params), pdl=True)
        ins = [np.array(wl.make_input(j), copy=True) for j in range(npool)]
        want = [oracle_out(wl, x, (1, 1, 1, 1)) for x in ins]
        outs = np.full((n, wl.out_bytes()), SENTINEL, np.uint8)
        for k in range(n):
            ctx.submit(k, ins[k % npool].ctypes.data, outs[k].ctypes.data)
        ctx.drain()
        st = ctx.stats()
        assert st["staged_jobs"] == n and st["completed"] == n
        for p_ in range(npool):
            assert np.all(outs[p_::npool] == want[p_][None, :])
    finally:
        ctx.close()


@pytest.mark.parametrize("config", [0, 1, 4])
@pytest.mark.parametrize("lanes", [1, 2, 4, 8])
@pytest.mark.parametrize("mode", [0, 2, 4])
def test_streams_per_lane_compute_the_same(libset, config, lanes, mode):
    """set_config.streams_per_lane: consecutive jobs of a logical stream run on different CUDA streams; results, slot
    safety and the in-flight bound are unchanged, in SET and in the baseline models that share the streams."""
    from paper_2606_05495_b200.workloads import small_workload
    wl = small_workload(config)
    st = check(libset, wl, list(range(min(wl.jobs, 64))), mode=mode, streams_per_lane=lanes, pdl=True)
    depth = wl.max_inflight // wl.num_streams
    assert st["cuda_streams"] == wl.num_streams * min(lanes, depth)
    assert st["max_inflight_seen"] <= wl.max_inflight


def test_declared_pinned_ranges(libset):
    """set_host_register / set_host_unregister: a torch pinned tensor declared once is used in place; pageable memory and
    device memory are refused; after unregistering, the pointer is queried per job again (still pinned, still in place)."""
    import torch
    from paper_2606_05495_b200.workloads import small_workload
    wl = small_workload(0)
    ctx = libset.Context(wl.num_streams, wl.max_inflight)
    try:
        ctx.register_builtin(0)
        n = 16
        t_in = torch.empty(n * wl.in_bytes(), dtype=torch.uint8).pin_memory()
        t_out = torch.full((n * wl.out_bytes(),), SENTINEL, dtype=torch.uint8).pin_memory()
        ins = [wl.make_input(j) for j in range(n)]
        for j, x in enumerate(ins):
            t_in[j * wl.in_bytes():(j + 1) * wl.in_bytes()] = torch.from_numpy(np.array(x, copy=True))
        ctx.host_register(t_in.data_ptr(), t_in.numel())
        ctx.host_register(t_out.data_ptr(), t_out.numel())
        with pytest.raises(libset.SetError):
            ctx.host_register(np.zeros(4096, np.uint8).ctypes.data, 4096)            # pageable
        with pytest.raises(libset.SetError):
            ctx.host_register(torch.zeros(4096, dtype=torch.uint8, device="cuda").data_ptr(), 4096)
        for rnd in range(2):
            for j in range(n):
                ctx.submit(j, t_in.data_ptr() + j * wl.in_bytes(), t_out.data_ptr() + j * wl.out_bytes())
            ctx.drain()
            out = t_out.numpy()
            for j in range(n):
                compare(wl, np.array(out[j * wl.out_bytes():(j + 1) * wl.out_bytes()], copy=True), oracle_out(wl, ins[j], (1, 1, 1, 1)))
            if rnd == 0:
                ctx.host_unregister(t_in.data_ptr())
                ctx.host_unregister(t_out.data_ptr())
                with pytest.raises(libset.SetError):
                    ctx.host_unregister(t_out.data_ptr())
                t_out.fill_(SENTINEL)
        assert ctx.stats()["staged_jobs"] == 0
    finally:
        ctx.close()


def test_maximum_depth_4096_in_flight(libset):
    """PAPER.md:276 sweeps the batch size to b = 4096: max_inflight = 4096 registers (4096 slots x 2 execs), runs 8,192
    config-1 jobs and every result is the oracle's."""
    import ctypes as C
    from paper_2606_05495_b200.workloads import PinnedArena, Workload
    wl = Workload(1, (4096,), jobs=8192, num_streams=8, max_inflight=4096)
    n, npool = 8192, 256
    ctx = libset.Context(8, 4096, queue_capacity=1)
    try:
        ctx.register_builtin(1, 0, list(wl.params), pdl=True)
        assert ctx.geometry() == (4096, 8, 2)
        ins = [wl.make_input(j) for j in range(npool)]
        want = np.array([oracle_out(wl, x, (1, 1, 1, 1)).view(np.float32)[0] for x in ins], np.float32)
        arena = PinnedArena(ctx, npool * (wl.in_bytes() + 256) + 4 * n + 4096)
        in_ptrs = []
        for x in ins:
            a, v = arena.take(wl.in_bytes())
            v[:] = x
            in_ptrs.append(a)
        a_out, v_out = arena.take(4 * n)
        v_out[:] = SENTINEL
        pi = (C.c_void_p * n)(*[in_ptrs[k % npool] for k in range(n)])
        po = (C.c_void_p * n)(*[a_out + 4 * k for k in range(n)])
        ctx.submit_batch(pi, po)
        ctx.drain()
        st = ctx.stats()
        assert st["completed"] == n and st["max_inflight_seen"] <= 4096
        got = np.array(v_out.view(np.float32), copy=True)
        ref = want[np.arange(n) % npool]
        assert np.all(np.abs(got - ref) <= 1e-6 * np.abs(ref))
        v_out = None
        arena.free()
    finally:
        ctx.close()


def test_time_stage_chains_by_plain_or_programmatic_edges(libset):
    """set_time_stage (bench.py's kernel rooflines): a chain of launches by plain edges, or by programmatic edges when the
    stage carries SET_STAGE_PDL; both run, give a sane time, leave the context usable and its results right."""
    from paper_2606_05495_b200.workloads import small_workload
    wl = small_workload(1)
    for pdl in (False, True):
        with libset.Context(2, 4) as ctx:
            ctx.register_builtin(1, 0, list(wl.params), pdl=pdl)
            ts = [ctx.time_stage(k, None, warmup=2, iters=20) for k in range(ctx.num_stages)]
            assert all(0.2 < t < 100.0 for t in ts), ts
        check(libset, wl, list(range(8)), pdl=pdl)


# ---------------------------------------------------------------------------------------------------------------------
# one scheduler instance per GPU behind one submit call, host-side stealing across instances.  One GPU here:
# both instances sit on device 0 (set.h allows it), which exercises everything but the second device.
# ---------------------------------------------------------------------------------------------------------------------
def _multi_run(libset, m, wl, job_ids):
    from paper_2606_05495_b200.workloads import PinnedArena
    ins = [wl.make_input(j) for j in job_ids]
    arena = PinnedArena(m, sum(x.nbytes + 512 for x in ins) + len(ins) * (wl.out_bytes() + 512) + 4096)
    bufs = []
    for x in ins:
        a_in, v_in = arena.take(x.nbytes)
        v_in[:] = x
        a_out, v_out = arena.take(wl.out_bytes())
        v_out[:] = SENTINEL
        bufs.append((a_in, a_out, v_out))
    for k, j in enumerate(job_ids):
        m.submit(j, bufs[k][0], bufs[k][1])
    m.drain()
    for k in range(len(job_ids)):
        compare(wl, np.array(bufs[k][2], copy=True), oracle_out(wl, ins[k], (1, 1, 1, 1)))
    bufs = None
    arena.free()


@pytest.mark.parametrize("config", [0, 1])
def test_multi_instance_front_end_routes_jobs_to_their_home(libset, config):
    from paper_2606_05495_b200.workloads import small_workload
    wl = small_workload(config)
    n = 300
    with libset.MultiContext([0, 0, 0], 2, 8) as m:
        m.register_builtin(config, 0, list(wl.params), pdl=True)
        _multi_run(libset, m, wl, list(range(n)))
        done = [m.stats(i)["completed"] for i in range(3)]
        assert sum(done) == n and m.stolen() <= n
        # a job runs at home unless home was full at that instant: whatever was not stolen ran at job_id mod 3
        assert all(abs(d - n // 3) <= m.stolen() for d in done), (done, m.stolen())


def test_multi_instance_front_end_steals_when_home_is_full(libset):
    """Every job id is even, so instance 0 is everybody's home; with one slot and two executables it is full most of the time
    and instance 1 takes what it cannot: every output is still F(in) of its own job, and instance 1 ran exactly the stolen jobs."""
    from paper_2606_05495_b200.workloads import small_workload
    wl = small_workload(1)
    n = 400
    with libset.MultiContext([0, 0], 1, 1, queue_capacity=1) as m:
        m.register_builtin(1, 0, list(wl.params))
        _multi_run(libset, m, wl, [2 * k for k in range(n)])
        s0, s1 = m.stats(0), m.stats(1)
        assert s0["completed"] + s1["completed"] == n
        assert m.stolen() == s1["completed"] and m.stolen() > 0
        assert s0["max_inflight_seen"] <= 1 and s1["max_inflight_seen"] <= 1


def test_try_submit_reports_busy_and_leaves_the_context_usable(libset):
    import ctypes as C
    from paper_2606_05495_b200.workloads import PinnedArena, small_workload
    wl = small_workload(1)
    lib = libset.load()
    with libset.Context(1, 1, queue_capacity=1) as ctx:
        ctx.register_builtin(1, 0, list(wl.params))
        x = wl.make_input(0)
        arena = PinnedArena(ctx, x.nbytes + 64 * 512 + 4096)
        a_in, v_in = arena.take(x.nbytes)
        v_in[:] = x
        outs = [arena.take(4) for _ in range(64)]
        codes = [lib.set_try_submit_dims(ctx._h, k, a_in, outs[k][0], None) for k in range(64)]
        ctx.drain()
        assert set(codes) <= {libset.SET_OK, libset.SET_ERR_BUSY} and codes[0] == libset.SET_OK
        assert codes.count(libset.SET_ERR_BUSY) > 0                       # two executables, 64 submissions in a few microseconds
        assert ctx.stats()["completed"] == codes.count(libset.SET_OK)
        want = oracle_out(wl, x, (1, 1, 1, 1))
        for k, c in enumerate(codes):
            if c == libset.SET_OK:
                compare(wl, np.array(outs[k][1], copy=True), want)
        ctx.submit(99, a_in, outs[0][0])                                  # still usable
        ctx.drain()
        v_in = outs = None
        arena.free()


# ---------------------------------------------------------------------------------------------------------------------
# the two paper workloads of SURVEY.md 8(f)4: SSSP with a conditional WHILE node (config 5), Sobel chain (config 6)
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("config", [5, 6])
@pytest.mark.parametrize("mode", [2, 3, 4])
def test_paper_workloads_in_the_graph_baseline_models(libset, config, mode):
    from paper_2606_05495_b200.workloads import small_workload
    wl = small_workload(config)
    check(libset, wl, list(range(min(wl.jobs, 20))), mode=mode)


def test_plain_streams_refuse_a_loop_pipeline(libset):
    ctx = libset.Context(2, 4, mode=libset.MODE_PLAIN_STREAMS)
    with pytest.raises(libset.SetError) as ei:
        ctx.register_builtin(5, 0, [256, 2048])
    assert ei.value.status == libset.SET_ERR_INVALID
    ctx.close()
    ctx = libset.Context(2, 4, steal_policy=libset.STEAL_RETARGET)     # executables of a loop pipeline cannot migrate
    with pytest.raises(libset.SetError):
        ctx.register_builtin(5, 0, [256, 2048])
    ctx.close()


@pytest.mark.parametrize("streams,lanes,want", [(8, 4, 8), (8, 1, 8), (16, 2, 8), (12, 2, 6), (3, 4, 3)])
def test_loop_pipelines_run_on_at_most_8_streams(libset, streams, lanes, want):
    """More than 8 WHILE graphs in flight at once fail now and then on this driver, and a WHILE graph queued on a stream
    behind a running one slows both (profiles/r2_probes.md section 3), so a pipeline with a loop keeps to the largest
    divisor of S that is <= 8 CUDA streams and to one job in flight on each, whatever streams_per_lane and max_inflight
    ask for; the other workloads keep all their streams and slots."""
    from paper_2606_05495_b200.workloads import Workload
    wl = Workload(5, (512, inputgen.sssp_max_edges(512, 4)), jobs=96, num_streams=streams, max_inflight=4 * streams, kernels_per_job=6,
                  extra={"mean_deg": 4})
    st = check(libset, wl, list(range(96)), streams_per_lane=lanes, pdl=True)
    assert st["cuda_streams"] == want and 1 <= st["max_inflight_seen"] <= want
    wl6 = Workload(6, (1920, 1080), jobs=16, num_streams=streams, max_inflight=4 * streams, dtype="u8", kernels_per_job=5)
    assert check(libset, wl6, list(range(16)), streams_per_lane=lanes)["cuda_streams"] == streams * lanes


@pytest.mark.parametrize("v,deg", [(1, 1), (2, 1), (37, 2), (256, 1), (1000, 4), (4096, 8), (20000, 3)])
@pytest.mark.parametrize("pdl", [False, True])
def test_config5_graph_sizes(libset, v, deg, pdl):
    """One vertex, a sparse graph most of which is unreachable (degree 1), several blocks plus a ragged tail, the bench
    size, and a graph large enough for dozens of rounds: distances bit-exact, rounds within the oracle's."""
    from paper_2606_05495_b200.workloads import Workload
    wl = Workload(5, (v, inputgen.sssp_max_edges(v, deg)), jobs=10, num_streams=2, max_inflight=4, kernels_per_job=6, extra={"mean_deg": deg})
    check(libset, wl, list(range(10)), pdl=pdl)


@pytest.mark.parametrize("unroll", [2, 3, 5, 8])
@pytest.mark.parametrize("v,deg", [(1, 1), (37, 2), (4096, 8), (20000, 3)])
def test_config5_relaxations_per_loop_pass(libset, unroll, v, deg):
    """U relaxation kernels per pass of the WHILE body (default 4), odd and even: the frontier's double buffer follows the
    relaxation's running number, relaxations over an empty frontier change nothing and are not counted as rounds, so the
    distances and the bound on the round count do not depend on U; the graph has 2 + U stage kernels."""
    from paper_2606_05495_b200.workloads import Workload
    wl = Workload(5, (v, inputgen.sssp_max_edges(v, deg), unroll), jobs=8, num_streams=2, max_inflight=4, kernels_per_job=2 + unroll,
                  extra={"mean_deg": deg})
    st = check(libset, wl, list(range(8)))
    assert st["kernel_nodes"] == 8 * (2 + unroll)


@pytest.mark.parametrize("v,deg", [(1, 1), (2, 1), (37, 2), (256, 1), (1000, 4), (4096, 8), (20000, 3)])
@pytest.mark.parametrize("pdl", [False, True])
def test_config5_single_kernel_variant(libset, v, deg, pdl):
    """Variant 1 of config 5: the whole job in ONE kernel of one block (SET_K_SSSP_SOLO), no WHILE node.  Same images, same
    outputs, same rule: distances bit for bit, rounds within the oracle's; more jobs than slots, so every slot's scratch is
    reused by a job with another graph."""
    from paper_2606_05495_b200.workloads import Workload
    wl = Workload(5, (v, inputgen.sssp_max_edges(v, deg)), variant=1, jobs=24, num_streams=4, max_inflight=8, kernels_per_job=1,
                  extra={"mean_deg": deg})
    st = check(libset, wl, list(range(24)), pdl=pdl)
    assert st["kernel_nodes"] == 24 and st["cuda_streams"] >= 4       # an ordinary pipeline: no loop, all streams in use


def test_config5_single_kernel_variant_at_the_bench_size_in_every_model(libset):
    from paper_2606_05495_b200.workloads import baseline_workload
    import dataclasses
    wl = dataclasses.replace(baseline_workload(5), variant=1, kernels_per_job=1, jobs=256)
    for mode in (0, 1, 2, 3, 4):
        check(libset, wl, list(range(256 if mode == 0 else 40)), mode=mode)


@pytest.mark.parametrize("variant", [0, 1])
def test_copies_of_a_job_dependent_size_as_sm_copies(libset, variant):
    """Config 5's copy-in is 16 + 4 (V + 1) + 8 E bytes, E per job: with sm_copy_max_bytes above the buffer's capacity it is an
    SM copy node whose byte count and grid are updated per job (two SM copies per job then: in and out); the default limit
    keeps the copy engine for it at the bench size.  Jobs of different E alternate on every slot."""
    from paper_2606_05495_b200.workloads import Workload
    v, deg = 4096, 8
    wl = Workload(5, (v, inputgen.sssp_max_edges(v, deg)), variant=variant, jobs=40, num_streams=4, max_inflight=8,
                  kernels_per_job=1 if variant else 6, extra={"mean_deg": deg})
    assert len({wl.dims(j)[0] for j in range(40)}) > 30                       # the sizes really differ
    st = check(libset, wl, list(range(40)), sm_copy_max_bytes=1 << 20)
    assert st["copy_nodes"] == 2 * 40
    st = check(libset, wl, list(range(8)))
    assert st["copy_nodes"] == 8                                              # default: copy-out only


def test_config5_unroll_out_of_range_is_refused(libset):
    for u in (0, 1, 9):       # U = 1 would be a two-node loop body, which this driver does not run reliably (set.h)
        ctx = libset.Context(2, 4)
        with pytest.raises(libset.SetError) as ei:
            ctx.register_builtin(5, 0, [256, 2048, u])
        assert ei.value.status == libset.SET_ERR_INVALID
        ctx.close()


def test_config5_hand_graphs_through_the_library(libset):
    """The oracle's hand cases on the GPU path: a path graph (one round per hop), the late shortcut, a zero-weight cycle,
    a source without edges, and a source that is not vertex 0."""
    import oracle
    from paper_2606_05495_b200.workloads import PinnedArena

    def image(v, edges, src):
        edges = sorted(edges)
        rp = np.zeros(v + 1, np.int32)
        for u, _, _ in edges:
            rp[u + 1] += 1
        rp = np.cumsum(rp).astype(np.int32)
        return np.concatenate([np.array([v, len(edges), src, 0], np.int32), rp, np.array([e[1] for e in edges], np.int32),
                               np.array([e[2] for e in edges], np.int32)]).astype(np.int32)

    maxv, maxe = 16, 64
    cases = [image(16, [(k, k + 1, 3) for k in range(15)], 0),
             image(16, [(0, 1, 1), (0, 3, 10), (1, 2, 1), (2, 3, 1), (3, 4, 1)], 0),
             image(16, [(0, 1, 0), (1, 2, 0), (2, 0, 0)], 0),
             image(16, [(1, 2, 5)], 0),
             image(16, [(k, k + 1, 3) for k in range(15)], 9)]
    ctx = libset.Context(2, 4)
    try:
        ctx.register_builtin(5, 0, [maxv, maxe])
        arena = PinnedArena(ctx, 1 << 16)
        outs = []
        for j, img in enumerate(cases):
            a_in, v_in = arena.take(img.nbytes)
            v_in[:] = img.view(np.uint8)
            a_out, v_out = arena.take(4 * maxv + 16)
            v_out[:] = SENTINEL
            outs.append(v_out)
            ctx.submit(j, a_in, a_out, (int(img[1]), 1, 1, 1))
        ctx.drain()
        for img, o in zip(cases, outs):
            got = np.array(o, copy=True).view(np.int32)
            ref = oracle.sssp_job(img).view(np.int32)
            assert np.array_equal(got[:16], ref[:16]) and 1 <= got[16] <= ref[16]
        # the path graph needs one round per hop whatever the relaxation order: 16 rounds exactly
        assert np.array(outs[0], copy=True).view(np.int32)[16] == 16
        outs = None
        arena.free()
    finally:
        ctx.close()


def test_config5_work_stealing_with_slot_bound_executables(libset):
    """A loop pipeline's executables cannot leave their slot (set.h SET_STAGE_LOOP_BEGIN): with a delay stage that keeps
    one slot busy, idle slots steal its queued jobs and run them on their OWN executables; every distance still exact."""
    from paper_2606_05495_b200.workloads import Workload
    wl = Workload(5, (512, inputgen.sssp_max_edges(512, 4)), variant=libset.VARIANT_SPIN, jobs=160, num_streams=4, max_inflight=8,
                  kernels_per_job=4, extra={"mean_deg": 4, "spin_ns": lambda j: 2_000_000 if j % 8 == 0 else 1000})
    outs, ins, dims, st = run_jobs(libset, wl, list(range(wl.jobs)), num_dispatchers=2)
    assert st["completed"] == wl.jobs
    for k in range(wl.jobs):
        compare(wl, outs[k], oracle_out(wl, ins[k], dims[k]))
    assert st["steals"] > 0


@pytest.mark.parametrize("size", [(1, 1), (5, 4), (7, 3), (128, 64), (132, 65), (644, 9), (16, 1), (1, 16), (1920, 3), (640, 480), (1916, 7)])
def test_config6_ragged_frames(libset, size):
    from paper_2606_05495_b200.workloads import Workload
    wl = Workload(6, (1920, 1080), jobs=3, num_streams=2, max_inflight=4, kernels_per_job=5, extra={"size": size})
    check(libset, wl, list(range(3)))


@pytest.mark.parametrize("size", [(328, 77), (336, 77), (1040, 19), (512, 16)])
@pytest.mark.parametrize("upto", [2, 3, 4])
def test_config6_stage_by_stage(libset, upto, size):
    """The Sobel chain truncated after the edge (2), mean (3) and threshold (4) stages, with that stage's buffer copied
    back: every intermediate image bit for bit against the oracle's stage functions."""
    import oracle
    from paper_2606_05495_b200.workloads import PinnedArena
    w, h = size    # a ragged width (per-pixel path); multiples of 16: part of a 512-pixel tile, two tiles and a bit, exactly one tile
    st, ns, bf, nb, _, _ = libset.builtin_pipeline(6, 0, [w, h])
    assert ns == 5 and nb == 4
    src_buf = {2: 2, 3: 3, 4: 2}[upto]                         # sobel -> buffer 2, mean -> 3, threshold -> 2
    bf[3].d2h_bytes.per_unit = 0
    bf[src_buf].d2h_bytes.per_unit, bf[src_buf].d2h_bytes.dim_mask = 1, 3
    ctx = libset.Context(2, 4)
    try:
        ctx.register_pipeline(st, upto, bf, nb)
        arena = PinnedArena(ctx, 8 * (4 * w * h + 1024))
        frames, outs = [inputgen.sobel_frame(500 + j, (w, h)) for j in range(6)], []
        for j, f in enumerate(frames):
            a_in, v_in = arena.take(3 * w * h)
            v_in[:] = f.reshape(-1)
            a_out, v_out = arena.take(w * h)
            v_out[:] = SENTINEL
            outs.append(v_out)
            ctx.submit(j, a_in, a_out, (w, h, 1, 1))
        ctx.drain()
        for f, o in zip(frames, outs):
            n = oracle.gray_u8(f)
            e = oracle.sobel_u8(n)
            want = e if upto == 2 else oracle.mean3x3_u8(e) if upto == 3 else oracle.threshold_u8(oracle.mean3x3_u8(e), 64)
            assert np.array_equal(np.array(o, copy=True).reshape(h, w), want)
        outs = None
        arena.free()
    finally:
        ctx.close()


def test_full_job_count_config5_and_config6(libset):
    from paper_2606_05495_b200.workloads import baseline_workload
    wl = baseline_workload(5)
    _full_count(libset, wl, wl.jobs, 64)                         # 2,048 SSSP jobs over 64 distinct graphs
    wl = baseline_workload(6)
    _full_count(libset, wl, wl.jobs, 96)                         # 4,096 frames over 96 distinct ones


@pytest.mark.parametrize("config", [0, 1, 5])
@pytest.mark.parametrize("fuse,forward", [("1", "1"), ("0", "1"), ("0", "0")])
def test_signal_fusing_and_output_forwarding_variants(libset, monkeypatch, config, fuse, forward):
    """The three shapes of a short job's tail: completion word stored by the forwarded copy-out node (default), a signal node
    of its own behind a forwarded copy-out node, and round 1's shape (two node updates per job, separate signal node)."""
    from paper_2606_05495_b200.workloads import small_workload
    monkeypatch.setenv("SET_FUSE_SIGNAL", fuse)
    monkeypatch.setenv("SET_FORWARD_OUT", forward)
    wl = small_workload(config)
    n = min(wl.jobs, 64)
    st = check(libset, wl, list(range(n)), pdl=True, debug_sentinel=0xA5A5A5A5)
    assert st["early_completions"] == 0
    # config 5's copy-in has a job-dependent size: it is an SM copy too while its buffer's capacity is within sm_copy_max_bytes
    assert st["signal_nodes"] == (0 if fuse == "1" and forward == "1" else n)
