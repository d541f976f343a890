"""Thin binding of libsettrace (include/set_trace.h): device-timeline gaps from CUPTI activity records.

Measurement only: nothing on the dispatch path imports this module, and libset.so does not depend on the library.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsettrace.so")

KIND_KERNEL, KIND_SIGNAL, KIND_MEMCPY, KIND_MEMSET = 0, 1, 2, 3


class GapSummary(C.Structure):
    _fields_ = [("count", C.c_uint64), ("mean_us", C.c_double), ("p50_us", C.c_double), ("p99_us", C.c_double),
                ("max_us", C.c_double)]

    def as_dict(self):
        return {"count": int(self.count), "mean_us": round(self.mean_us, 3), "p50_us": round(self.p50_us, 3),
                "p99_us": round(self.p99_us, 3), "max_us": round(self.max_us, 3)}


class TraceStats(C.Structure):
    _fields_ = [("kernels", C.c_uint64), ("signal_kernels", C.c_uint64), ("memcpys", C.c_uint64), ("memsets", C.c_uint64),
                ("streams", C.c_uint64), ("dropped", C.c_uint64), ("jobs", C.c_uint64), ("kernel_kernel_overlapped", C.c_uint64), ("wall_us", C.c_double), ("busy_us", C.c_double),
                ("idle_frac", C.c_double), ("kernel_mean_us", C.c_double), ("sum_op_us", C.c_double),
                ("kernel_kernel", GapSummary), ("intra_job", GapSummary), ("inter_job", GapSummary), ("any_op", GapSummary)]

    def as_dict(self):
        d = {}
        for name, typ in self._fields_:
            v = getattr(self, name)
            d[name] = v.as_dict() if typ is GapSummary else (int(v) if typ is C.c_uint64 else round(float(v), 4))
        return d


class TraceRec(C.Structure):
    _fields_ = [("stream", C.c_uint32), ("job", C.c_uint32), ("kind", C.c_uint32), ("reserved", C.c_uint32),
                ("start_ns", C.c_uint64), ("end_ns", C.c_uint64)]


_lib = None


def load():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2606_05495_b200.build`")
        lib = C.CDLL(LIB_PATH)
        lib.set_trace_start.restype = C.c_int
        lib.set_trace_stop.restype = C.c_int
        lib.set_trace_stop.argtypes = [C.POINTER(TraceStats)]
        lib.set_trace_reduce.restype = C.c_int
        lib.set_trace_reduce.argtypes = [C.POINTER(TraceRec), C.c_uint64, C.POINTER(TraceStats)]
        lib.set_trace_error.restype = C.c_char_p
        _lib = lib
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        raise RuntimeError(f"{what}: {load().set_trace_error().decode()}")


def start() -> None:
    _check(load().set_trace_start(), "set_trace_start")


def stop() -> dict:
    st = TraceStats()
    _check(load().set_trace_stop(C.byref(st)), "set_trace_stop")
    return st.as_dict()


def reduce(records) -> dict:
    """records: iterable of (stream, job, kind, start_ns, end_ns)."""
    records = list(records)
    arr = (TraceRec * max(1, len(records)))()
    for i, (s, j, k, t0, t1) in enumerate(records):
        arr[i] = TraceRec(s, j, k, 0, t0, t1)
    st = TraceStats()
    _check(load().set_trace_reduce(arr, len(records), C.byref(st)), "set_trace_reduce")
    return st.as_dict()
