"""paper_2606_05495_b200 -- thin Python binding of libset (include/set.h).

Argument marshalling only: every step of the hot path (scheduling, graph updates, launches, stage kernels)
runs inside the C-ABI library.  The binding fails loudly if the CUDA extension is missing: there is no CPU
fallback and nothing here imports `oracle/`.

    import paper_2606_05495_b200 as setlib
    ctx = setlib.Context(num_streams=4, max_inflight=8)
    ctx.register_builtin(0)                       # BASELINE.json:configs[0]
    ctx.submit(job_id, host_in_ptr, host_out_ptr) # plain integer addresses (e.g. tensor.data_ptr())
    ctx.drain()
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libset.so")

SET_OK, SET_ERR_INVALID, SET_ERR_CUDA, SET_ERR_NOMEM, SET_ERR_STATE, SET_ERR_SIZE, SET_ERR_BUSY = 0, -1, -2, -3, -4, -5, -6
SET_MAX_STAGES, SET_MAX_BUFFERS, SET_MAX_ARGS, SET_MAX_DIMS = 16, 8, 12, 4
MODE_SET, MODE_PLAIN_STREAMS, MODE_BATCH_SYNC, MODE_SINGLE_GRAPH, MODE_MUTEX_QUEUE = 0, 1, 2, 3, 4
IO_HOST, IO_DEVICE = 0, 1
STEAL_SWAP, STEAL_RETARGET = 0, 1
CB_DEFAULT, CB_NOTIFY_STREAM, CB_WORK_STREAM, CB_FLAG_POLL, CB_HOST_NODE = 0, 1, 2, 3, 4
ARG_BUFFER, ARG_IMM32, ARG_IMM64, ARG_DIM, ARG_TMAP2D, ARG_COND = 0, 1, 2, 3, 4, 5
STAGE_LOOP_BEGIN, STAGE_LOOP_END = 2, 4
STAGE_PDL = 1
FENCE_DEFAULT, FENCE_SYSTEM, FENCE_NONE = 0, 1, 2
K_COPY = 15
BUF_ZERO = 1
VARIANT_SPIN = 0x100

_STATUS_NAMES = {0: "SET_OK", -1: "SET_ERR_INVALID", -2: "SET_ERR_CUDA", -3: "SET_ERR_NOMEM", -4: "SET_ERR_STATE",
                 -5: "SET_ERR_SIZE", -6: "SET_ERR_BUSY"}


class SetError(RuntimeError):
    def __init__(self, status: int, what: str, detail: str = ""):
        self.status = status
        super().__init__(f"{what}: {_STATUS_NAMES.get(status, status)}" + (f" -- {detail}" if detail else ""))


class SizeExpr(C.Structure):
    _fields_ = [("fixed", C.c_uint64), ("per_unit", C.c_uint64), ("dim_mask", C.c_uint32), ("reserved", C.c_uint32)]


class GridRule(C.Structure):
    _fields_ = [("count", SizeExpr), ("divisor", C.c_uint32), ("reserved", C.c_uint32)]


class Tmap2D(C.Structure):
    _fields_ = [("elem_bytes", C.c_uint32), ("swizzle", C.c_uint32), ("inner", C.c_uint64), ("outer", C.c_uint64),
                ("pitch_bytes", C.c_uint64), ("box_inner", C.c_uint32), ("box_outer", C.c_uint32)]


class ArgDesc(C.Structure):
    _fields_ = [("kind", C.c_int32), ("index", C.c_int32), ("offset", SizeExpr), ("imm", C.c_uint64), ("tmap", Tmap2D)]


class StageDesc(C.Structure):
    _fields_ = [("func", C.c_void_p), ("grid", GridRule * 3), ("block", C.c_uint32 * 3), ("smem_bytes", C.c_uint32),
                ("flags", C.c_uint32), ("num_args", C.c_int32), ("reserved", C.c_int32), ("args", ArgDesc * SET_MAX_ARGS)]


class BufferDesc(C.Structure):
    _fields_ = [("bytes", C.c_uint64), ("flags", C.c_uint32), ("reserved", C.c_uint32), ("h2d_bytes", SizeExpr),
                ("h2d_host_off", SizeExpr), ("h2d_dev_off", SizeExpr), ("d2h_bytes", SizeExpr), ("d2h_host_off", SizeExpr),
                ("d2h_dev_off", SizeExpr), ("zero_off", SizeExpr), ("zero_bytes", SizeExpr)]


class Config(C.Structure):
    _fields_ = [("struct_bytes", C.c_uint32), ("num_streams", C.c_int32), ("max_inflight", C.c_int32), ("mode", C.c_int32),
                ("io", C.c_int32), ("queue_capacity", C.c_int32), ("num_dispatchers", C.c_int32), ("steal_policy", C.c_int32),
                ("callback_mode", C.c_int32), ("device", C.c_int32), ("spin_us", C.c_int32), ("sm_copy_max_bytes", C.c_int32),
                ("timestamps", C.c_int32), ("completion_fence", C.c_int32), ("streams", C.POINTER(C.c_void_p)), ("device_arena", C.c_void_p), ("device_arena_bytes", C.c_uint64),
                ("streams_per_lane", C.c_int32), ("completion_thread", C.c_int32), ("bind_at_launch", C.c_int32), ("debug_sentinel", C.c_uint32)]


class Stats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in
                ("submitted", "completed", "launched", "steals", "full_rebinds", "host_rebinds", "staged_jobs", "submit_stalls",
                 "dispatcher_sleeps", "kernel_nodes", "ns_submit", "ns_bind", "ns_launch", "ns_callback", "ns_sync",
                 "max_inflight_seen", "signal_nodes", "copy_nodes", "early_completions", "cuda_streams")]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_ if n != "reserved"}


class GapStats(C.Structure):
    _fields_ = [("jobs", C.c_uint64), ("gaps", C.c_uint64), ("gap_mean_us", C.c_double), ("gap_p50_us", C.c_double),
                ("gap_p99_us", C.c_double), ("gap_max_us", C.c_double), ("job_mean_us", C.c_double), ("span_us", C.c_double),
                ("stream_busy_frac", C.c_double), ("busy_union_us", C.c_double), ("idle_frac", C.c_double),
                ("idle_gaps", C.c_double), ("idle_gap_mean_us", C.c_double)]

    def as_dict(self):
        return {n: (int(getattr(self, n)) if n in ("jobs", "gaps") else round(float(getattr(self, n)), 4)) for n, _ in self._fields_}


# every symbol include/set.h declares -- tests/test_abi.py checks the list against the header
EXPORTS = ["set_create", "set_create_ex", "set_register_pipeline", "set_submit", "set_submit_dims", "set_submit_batch",
           "set_drain", "set_destroy", "set_host_alloc", "set_host_free", "set_host_register", "set_host_unregister", "set_get_stats", "set_reset_stats", "set_get_gap_stats",
           "set_last_error", "set_get_geometry", "set_time_stage", "set_builtin_kernel", "set_builtin_pipeline",
           "set_selftest_find_order", "set_selftest_ring", "set_selftest_scheduler", "set_sssp_noalloc", "set_noalloc_last_error",
           "set_try_submit_dims", "set_multi_create", "set_multi_register_pipeline", "set_multi_submit_dims", "set_multi_drain",
           "set_multi_instance", "set_multi_stolen", "set_multi_destroy"]

_lib = None


def load():
    """dlopen libset.so and declare the prototypes.  Raises if the extension has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2606_05495_b200.build` (nvcc, sm_100a). "
                          "There is no CPU fallback.")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64, u64 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint64
    lib.set_create.argtypes = [C.c_int, C.c_int, C.POINTER(vp)]
    lib.set_create_ex.argtypes = [C.POINTER(Config), C.POINTER(vp)]
    lib.set_register_pipeline.argtypes = [vp, C.POINTER(StageDesc), C.c_int, C.POINTER(BufferDesc), C.c_int]
    lib.set_submit.argtypes = [vp, u64, vp, vp]
    lib.set_submit_dims.argtypes = [vp, u64, vp, vp, C.POINTER(C.c_uint32)]
    lib.set_submit_batch.argtypes = [vp, i64, u64, C.POINTER(u64), C.POINTER(vp), C.POINTER(vp), C.POINTER(C.c_uint32)]
    lib.set_drain.argtypes = [vp]
    lib.set_destroy.argtypes = [vp]
    lib.set_host_alloc.argtypes = [vp, C.c_size_t]
    lib.set_host_alloc.restype = vp
    lib.set_host_free.argtypes = [vp, vp]
    lib.set_host_free.restype = None
    lib.set_host_register.argtypes = [vp, vp, C.c_size_t]
    lib.set_host_unregister.argtypes = [vp, vp]
    lib.set_get_stats.argtypes = [vp, C.POINTER(Stats)]
    lib.set_reset_stats.argtypes = [vp]
    lib.set_get_gap_stats.argtypes = [vp, C.POINTER(GapStats)]
    lib.set_last_error.argtypes = [vp]
    lib.set_last_error.restype = C.c_char_p
    lib.set_get_geometry.argtypes = [vp, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int)]
    lib.set_time_stage.argtypes = [vp, C.c_int, C.POINTER(C.c_uint32), C.c_int, C.c_int, C.POINTER(C.c_float)]
    lib.set_builtin_kernel.argtypes = [C.c_int]
    lib.set_builtin_kernel.restype = vp
    lib.set_builtin_pipeline.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_uint32), C.c_int, C.POINTER(StageDesc), C.POINTER(C.c_int),
                                         C.POINTER(BufferDesc), C.POINTER(C.c_int), C.POINTER(u64), C.POINTER(u64)]
    lib.set_selftest_find_order.argtypes = [C.c_int, C.c_int, u64]
    lib.set_selftest_ring.argtypes = [C.c_int, C.c_int, C.c_int, i64]
    lib.set_selftest_ring.restype = i64
    lib.set_selftest_scheduler.argtypes = [C.c_int] * 5 + [i64, C.c_uint32, C.POINTER(u64)]
    lib.set_selftest_scheduler.restype = i64
    lib.set_try_submit_dims.argtypes = [vp, u64, vp, vp, C.POINTER(C.c_uint32)]
    lib.set_multi_create.argtypes = [C.POINTER(Config), C.c_int, C.POINTER(C.c_int), C.POINTER(vp)]
    lib.set_multi_register_pipeline.argtypes = [vp, C.POINTER(StageDesc), C.c_int, C.POINTER(BufferDesc), C.c_int]
    lib.set_multi_submit_dims.argtypes = [vp, u64, vp, vp, C.POINTER(C.c_uint32)]
    lib.set_multi_drain.argtypes = [vp]
    lib.set_multi_instance.argtypes = [vp, C.c_int]
    lib.set_multi_instance.restype = vp
    lib.set_multi_stolen.argtypes = [vp]
    lib.set_multi_stolen.restype = u64
    lib.set_multi_destroy.argtypes = [vp]
    lib.set_sssp_noalloc.argtypes = [vp, vp, C.c_uint32, vp]
    lib.set_noalloc_last_error.argtypes = []
    lib.set_noalloc_last_error.restype = C.c_char_p
    for name in EXPORTS:
        fn = getattr(lib, name)
        if fn.restype is C.c_int and name not in ("set_selftest_find_order",):
            fn.restype = i32
    _lib = lib
    return lib


def builtin_pipeline(config: int, variant: int = 0, params=None):
    """(stages array, n_stages, bufs array, n_bufs, host_in_bytes, host_out_bytes) for BASELINE.json:configs[config]."""
    lib = load()
    stages = (StageDesc * SET_MAX_STAGES)()
    bufs = (BufferDesc * SET_MAX_BUFFERS)()
    ns, nb = C.c_int(0), C.c_int(0)
    hin, hout = C.c_uint64(0), C.c_uint64(0)
    p = (C.c_uint32 * len(params))(*params) if params else None
    rc = lib.set_builtin_pipeline(config, variant, p, len(params) if params else 0, stages, C.byref(ns), bufs, C.byref(nb),
                                  C.byref(hin), C.byref(hout))
    if rc != SET_OK:
        raise SetError(rc, f"set_builtin_pipeline({config})")
    return stages, ns.value, bufs, nb.value, hin.value, hout.value


class Context:
    """Owner of one set_ctx handle.  All pointers are plain integer addresses."""

    def __init__(self, num_streams: int, max_inflight: int, mode: int = MODE_SET, io: int = IO_HOST, queue_capacity: int = 0,
                 num_dispatchers: int = 0, steal_policy: int = STEAL_SWAP, callback_mode: int = CB_DEFAULT,
                 device: int = -1, spin_us: int = 0, streams=None, device_arena: int = 0, device_arena_bytes: int = 0,
                 sm_copy_max_bytes: int = 0, timestamps: bool = False, completion_fence: int = FENCE_DEFAULT,
                 streams_per_lane: int = 0, debug_sentinel: int = 0, completion_thread: int = 0, bind_at_launch: int = 0):
        self._lib = load()
        self._h = C.c_void_p(None)
        cfg = Config()
        cfg.struct_bytes = C.sizeof(Config)
        cfg.num_streams, cfg.max_inflight, cfg.mode, cfg.io = num_streams, max_inflight, mode, io
        cfg.queue_capacity, cfg.num_dispatchers, cfg.steal_policy = queue_capacity, num_dispatchers, steal_policy
        cfg.callback_mode, cfg.device, cfg.spin_us = callback_mode, device, spin_us
        cfg.sm_copy_max_bytes = sm_copy_max_bytes
        cfg.timestamps = 1 if timestamps else 0
        cfg.completion_fence, cfg.streams_per_lane, cfg.debug_sentinel = completion_fence, streams_per_lane, debug_sentinel
        cfg.completion_thread, cfg.bind_at_launch = completion_thread, bind_at_launch
        self._streams_arr = None
        if streams is not None:
            self._streams_arr = (C.c_void_p * len(streams))(*[int(s) for s in streams])
            cfg.streams = C.cast(self._streams_arr, C.POINTER(C.c_void_p))
        cfg.device_arena = device_arena or None
        cfg.device_arena_bytes = device_arena_bytes
        rc = self._lib.set_create_ex(C.byref(cfg), C.byref(self._h))
        if rc != SET_OK:
            raise SetError(rc, "set_create_ex")
        self.host_in_bytes = self.host_out_bytes = 0
        self.num_stages = 0

    # ---- lifecycle
    def close(self):
        if self._h:
            self._lib.set_destroy(self._h)
            self._h = C.c_void_p(None)

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int, what: str):
        if rc != SET_OK:
            raise SetError(rc, what, self.last_error())

    # ---- the four calls
    def register_pipeline(self, stages, num_stages: int, bufs, num_bufs: int):
        self._check(self._lib.set_register_pipeline(self._h, stages, num_stages, bufs, num_bufs), "set_register_pipeline")
        self.num_stages = num_stages

    def register_builtin(self, config: int, variant: int = 0, params=None, pdl: bool = False):
        st, ns, bf, nb, hin, hout = builtin_pipeline(config, variant, params)
        if pdl:  # programmatic-dependent-launch edges between consecutive kernel nodes (set.h SET_STAGE_PDL)
            for i in range(ns):
                st[i].flags |= STAGE_PDL
        self.register_pipeline(st, ns, bf, nb)
        self.host_in_bytes, self.host_out_bytes = hin, hout
        return hin, hout

    def submit(self, job_id: int, host_in: int, host_out: int, dims=None):
        if dims is None:
            rc = self._lib.set_submit(self._h, job_id, host_in, host_out)
        else:
            d = (C.c_uint32 * 4)(*(list(dims) + [1] * (4 - len(dims))))
            rc = self._lib.set_submit_dims(self._h, job_id, host_in, host_out, d)
        self._check(rc, "set_submit")

    def submit_batch(self, host_ins, host_outs, dims=None, first_id: int = 0):
        """host_ins / host_outs: sequences (or ctypes arrays) of integer addresses; dims: flat sequence of 4*n uint32."""
        n = len(host_ins)
        ins = host_ins if isinstance(host_ins, C.Array) else (C.c_void_p * n)(*host_ins)
        outs = host_outs if isinstance(host_outs, C.Array) else (C.c_void_p * n)(*host_outs)
        d = None
        if dims is not None:
            d = dims if isinstance(dims, C.Array) else (C.c_uint32 * (4 * n))(*dims)
        self._check(self._lib.set_submit_batch(self._h, n, first_id, None, ins, outs, d), "set_submit_batch")

    def submit_batch_slice(self, ins, outs, dims, lo: int, hi: int):
        """Jobs lo..hi-1 of pre-built ctypes arrays (no copies): several caller threads can share one job list --
        set_submit* is thread-safe (set.h), and ctypes releases the GIL for the duration of the call."""
        vp = C.c_void_p
        pi = C.cast(C.byref(ins, lo * C.sizeof(vp)), C.POINTER(vp))
        po = C.cast(C.byref(outs, lo * C.sizeof(vp)), C.POINTER(vp))
        pd = C.cast(C.byref(dims, lo * 16), C.POINTER(C.c_uint32)) if dims is not None else None
        self._check(self._lib.set_submit_batch(self._h, hi - lo, lo, None, pi, po, pd), "set_submit_batch")

    def drain(self):
        self._check(self._lib.set_drain(self._h), "set_drain")

    # ---- extras
    def host_alloc(self, nbytes: int) -> int:
        p = self._lib.set_host_alloc(self._h, nbytes)
        if not p:
            raise SetError(SET_ERR_NOMEM, f"set_host_alloc({nbytes})")
        return int(p)

    def host_free(self, p: int):
        self._lib.set_host_free(self._h, p)

    def host_register(self, p: int, nbytes: int):
        self._check(self._lib.set_host_register(self._h, p, nbytes), "set_host_register")

    def host_unregister(self, p: int):
        self._check(self._lib.set_host_unregister(self._h, p), "set_host_unregister")

    def stats(self) -> dict:
        s = Stats()
        self._check(self._lib.set_get_stats(self._h, C.byref(s)), "set_get_stats")
        return s.as_dict()

    def gap_stats(self) -> dict:
        g = GapStats()
        self._check(self._lib.set_get_gap_stats(self._h, C.byref(g)), "set_get_gap_stats")
        return g.as_dict()

    def reset_stats(self):
        self._lib.set_reset_stats(self._h)

    def last_error(self) -> str:
        if not self._h:
            return ""
        return (self._lib.set_last_error(self._h) or b"").decode()

    def geometry(self):
        a, b, c = C.c_int(0), C.c_int(0), C.c_int(0)
        self._lib.set_get_geometry(self._h, C.byref(a), C.byref(b), C.byref(c))
        return a.value, b.value, c.value

    def time_stage(self, stage: int, dims=None, warmup: int = 3, iters: int = 20) -> float:
        d = (C.c_uint32 * 4)(*(list(dims) + [1] * (4 - len(dims)))) if dims is not None else None
        out = C.c_float(0)
        self._check(self._lib.set_time_stage(self._h, stage, d, warmup, iters, C.byref(out)), "set_time_stage")
        return out.value


class MultiContext:
    """set_multi (include/set.h): one scheduler instance per entry of `devices` behind one submit call; a job's home is
    job_id mod n, an instance with room takes a job whose home is full.  Argument marshalling only."""

    def __init__(self, devices, num_streams: int, max_inflight: int, queue_capacity: int = 0, sm_copy_max_bytes: int = 0,
                 streams_per_lane: int = 0, completion_thread: int = 0):
        self._lib = load()
        self._h = C.c_void_p(None)
        cfg = Config()
        cfg.struct_bytes = C.sizeof(Config)
        cfg.num_streams, cfg.max_inflight, cfg.mode, cfg.io = num_streams, max_inflight, MODE_SET, IO_HOST
        cfg.queue_capacity, cfg.sm_copy_max_bytes, cfg.streams_per_lane, cfg.completion_thread = queue_capacity, sm_copy_max_bytes, streams_per_lane, completion_thread
        self.n = len(devices)
        dev = (C.c_int * self.n)(*[int(d) for d in devices])
        rc = self._lib.set_multi_create(C.byref(cfg), self.n, dev, C.byref(self._h))
        if rc != SET_OK:
            raise SetError(rc, "set_multi_create")

    def _check(self, rc: int, what: str):
        if rc != SET_OK:
            detail = " | ".join(filter(None, ((self._lib.set_last_error(self.instance(i)) or b"").decode() for i in range(self.n))))
            raise SetError(rc, what, detail)

    def instance(self, i: int) -> int:
        return self._lib.set_multi_instance(self._h, i)

    def register_builtin(self, config: int, variant: int = 0, params=None, pdl: bool = False):
        st, ns, bf, nb, hin, hout = builtin_pipeline(config, variant, params)
        if pdl:
            for i in range(ns):
                st[i].flags |= STAGE_PDL
        self._check(self._lib.set_multi_register_pipeline(self._h, st, ns, bf, nb), "set_multi_register_pipeline")
        return hin, hout

    def submit(self, job_id: int, host_in: int, host_out: int, dims=None):
        d = None if dims is None else (C.c_uint32 * 4)(*(list(dims) + [1] * (4 - len(dims))))
        self._check(self._lib.set_multi_submit_dims(self._h, job_id, host_in, host_out, d), "set_multi_submit_dims")

    def drain(self):
        self._check(self._lib.set_multi_drain(self._h), "set_multi_drain")

    def stolen(self) -> int:
        return int(self._lib.set_multi_stolen(self._h))

    def stats(self, i: int) -> dict:
        s = Stats()
        self._check(self._lib.set_get_stats(self.instance(i), C.byref(s)), "set_get_stats")
        return s.as_dict()

    def host_alloc(self, nbytes: int) -> int:
        p = self._lib.set_host_alloc(self.instance(0), nbytes)
        if not p:
            raise SetError(SET_ERR_NOMEM, f"set_host_alloc({nbytes})")
        return p

    def host_free(self, p: int):
        self._lib.set_host_free(self.instance(0), p)

    def close(self):
        if self._h:
            self._lib.set_multi_destroy(self._h)
            self._h = C.c_void_p(None)

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()


NOALLOC_MAX_VERTICES = 16384  # SET_NOALLOC_MAX_VERTICES


def sssp_noalloc(dev_image: int, dev_out: int, num_vertices: int, stream: int = 0) -> None:
    """set_sssp_noalloc (include/set.h): one SSSP job on `stream`, scratch in the library's static device array, no
    allocation.  dev_image / dev_out are DEVICE addresses; asynchronous.  Raises SetError (SET_ERR_SIZE beyond
    NOALLOC_MAX_VERTICES)."""
    lib = load()
    rc = lib.set_sssp_noalloc(dev_image, dev_out, num_vertices, stream or None)
    if rc != SET_OK:
        raise SetError(rc, "set_sssp_noalloc", lib.set_noalloc_last_error().decode())


def selftest_find_order(b: int, w: int, nonempty: int) -> int:
    return load().set_selftest_find_order(b, w, nonempty)


def selftest_ring(capacity: int, producers: int, consumers: int, items_per_producer: int) -> int:
    return load().set_selftest_ring(capacity, producers, consumers, items_per_producer)


def selftest_scheduler(num_streams, max_inflight, queue_capacity, num_dispatchers, submitters, jobs, seed):
    steals = C.c_uint64(0)
    rc = load().set_selftest_scheduler(num_streams, max_inflight, queue_capacity, num_dispatchers, submitters, jobs, seed,
                                       C.byref(steals))
    return rc, steals.value
