"""set_sssp_noalloc (include/set.h): the entry point that allocates nothing -- one SSSP job as one kernel launch, its
scratch in the library's file-scope static __device__ array.  Checked against the EXISTING path (builtin config 5 through
a set_ctx: WHILE-node job graph, per-slot scratch from cudaMalloc) under the rule the config-5 parity tests use: the
distances bit for bit, the round count within [1, the oracle's synchronous count] (reading S5-4).

Named test_zz_* so that pytest collects it last: the suite runs with `pytest -x`, and a failure here must not hide
another test.  Passes alone in a fresh process and after the other tests (it shares nothing with them but the library)."""
import numpy as np
import pytest

import inputgen
from checker import compare, oracle_out


def _library_path_outputs(setlib, v, deg, job_ids):
    """out images of the jobs through the existing path: set_ctx + builtin pipeline 5."""
    from paper_2606_05495_b200.workloads import PinnedArena, Workload
    wl = Workload(5, (v, inputgen.sssp_max_edges(v, deg)), jobs=len(job_ids), num_streams=2, max_inflight=4, kernels_per_job=6,
                  extra={"mean_deg": deg})
    ctx = setlib.Context(wl.num_streams, wl.max_inflight)
    try:
        ctx.register_builtin(5, 0, list(wl.params))
        ins = [wl.make_input(j) for j in job_ids]
        dims = [wl.dims(j) for j in job_ids]
        arena = PinnedArena(ctx, sum(x.nbytes + 512 for x in ins) + len(ins) * (wl.out_bytes() + 512) + 4096)
        bufs = []
        for x in ins:
            a_in, v_in = arena.take(x.nbytes)
            v_in[:] = x
            a_out, v_out = arena.take(wl.out_bytes())
            bufs.append((a_in, a_out, v_out))
        for k, j in enumerate(job_ids):
            ctx.submit(j, bufs[k][0], bufs[k][1], dims[k])
        ctx.drain()
        outs = [np.array(b[2][:wl.out_bytes()], copy=True) for b in bufs]
        bufs = None
        arena.free()
        return wl, ins, dims, outs
    finally:
        ctx.close()


@pytest.mark.gpu
def test_sssp_noalloc_matches_the_library_path_on_two_calls_in_a_row(libset):
    import torch
    dev = torch.device("cuda:0")
    # the second graph is smaller than the first: the static scratch still holds the first call's flags beyond its V
    cases = [(4096, 8, 3), (1000, 4, 5), (4096, 8, 7), (37, 2, 1)]
    want = []
    for v, deg, job in cases:
        wl, ins, dims, outs = _library_path_outputs(libset, v, deg, [job])
        compare(wl, outs[0], oracle_out(wl, ins[0], dims[0]))     # the existing path is right to begin with
        want.append((wl, ins[0], dims[0], outs[0]))

    stream = torch.cuda.Stream(device=dev)
    imgs = [torch.from_numpy(np.array(w[1], copy=True).view(np.int32)).to(dev) for w in want]
    outs = [torch.full((c[0] + 4,), -559038737, dtype=torch.int32, device=dev) for c in cases]
    libset.sssp_noalloc(0, 0, 0)                                  # per-device set-up only: launches nothing
    libset.sssp_noalloc(imgs[0].data_ptr(), outs[0].data_ptr(), cases[0][0], stream.cuda_stream)  # warm: the kernel's module is loaded
    torch.cuda.synchronize()
    for o in outs:
        o.fill_(-559038737)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info(dev)[0]
    for k, c in enumerate(cases):                                 # calls in a row on one stream, nothing in between
        libset.sssp_noalloc(imgs[k].data_ptr(), outs[k].data_ptr(), c[0], stream.cuda_stream)
    stream.synchronize()
    assert torch.cuda.mem_get_info(dev)[0] == free_before, "the no-alloc entry point changed the device's free memory"
    for k, (wl, img, dims, lib_out) in enumerate(want):
        got = outs[k].cpu().numpy()
        ref = lib_out.view(np.int32)
        assert np.array_equal(got[:-4], ref[:-4]), f"case {k}: distances differ from the library path"
        assert got[-4] >= 1 and ref[-4] >= 1 and not got[-3:].any()
        compare(wl, got.view(np.uint8), oracle_out(wl, img, dims))  # same rule as the config-5 parity tests, round count included


@pytest.mark.gpu
def test_sssp_noalloc_clamps_to_the_callers_vertex_count_and_handles_a_lone_vertex(libset):
    import torch
    dev = torch.device("cuda:0")
    img = np.array([1, 0, 0, 0, 0, 0], np.int32)                  # V = 1, E = 0, src = 0, row_ptr = [0, 0]
    d_img = torch.from_numpy(img).to(dev)
    d_out = torch.full((5,), 77, dtype=torch.int32, device=dev)
    libset.sssp_noalloc(d_img.data_ptr(), d_out.data_ptr(), 1)
    torch.cuda.synchronize()
    assert d_out.cpu().tolist() == [0, 1, 0, 0, 0]                # dist[src] = 0; one round had a frontier


def test_sssp_noalloc_rejects_sizes_beyond_the_static_scratch(libset):
    """Checked before any CUDA call, so this runs without a GPU too."""
    with pytest.raises(libset.SetError) as ei:
        libset.sssp_noalloc(0, 0, libset.NOALLOC_MAX_VERTICES + 1)
    assert ei.value.status == libset.SET_ERR_SIZE
    assert "16384" in str(ei.value) and "16385" in str(ei.value)
