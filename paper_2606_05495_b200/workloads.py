"""Synthetic workloads of BASELINE.json:configs[0..4]: sizes, scheduler geometry and host-image builders.

Used by tests/ and bench.py to drive the C-ABI library.  Holds no arithmetic of the method and does not import
`oracle/`; inputs come from the shared seeded generator `inputgen`.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass, field

import numpy as np

import inputgen


@dataclass
class Workload:
    config: int
    params: tuple = ()
    variant: int = 0
    # BASELINE.json geometry
    jobs: int = 0
    num_streams: int = 4
    max_inflight: int = 8
    name: str = ""
    dtype: str = ""
    kernels_per_job: int = 0
    extra: dict = field(default_factory=dict)

    # ---- per-job host images
    def dims(self, job_id: int):
        if self.config in (4, 6):
            w, h = inputgen.config4_size(job_id) if "size" not in self.extra else self.extra["size"]
            return (w, h, 1, 1)
        if self.config == 5:  # dims[0] = E of the job's graph (the copy-in size depends on it)
            return (inputgen.sssp_edges(job_id, self.params[0], self.extra.get("mean_deg", 8)), 1, 1, 1)
        return (1, 1, 1, 1)

    def in_bytes(self, dims=None) -> int:
        c, p = self.config, self.params
        if c == 0: return 4 * p[0]
        if c == 1: return 8 * p[0]
        if c == 2: return 4 * p[0] * p[1]
        if c == 3: return 2 * p[0] * p[2] + 2 * p[2] * p[1] + 4 * p[1]
        if c in (4, 6): return 3 * dims[0] * dims[1]
        if c == 5: return 16 + 4 * (p[0] + 1) + 8 * dims[0]
        raise ValueError(c)

    def out_bytes(self, dims=None) -> int:
        c, p = self.config, self.params
        if c == 0: return 4 * p[0] + 256
        if c == 1: return 4
        if c == 2: return 4 * p[0] * p[1]
        if c == 3: return 2 * p[0] * p[1]
        if c == 4: return dims[0] * dims[1] + 1024
        if c == 5: return 4 * p[0] + 16
        if c == 6: return dims[0] * dims[1]
        raise ValueError(c)

    def make_input(self, job_id: int) -> np.ndarray:
        """uint8 byte image of job `job_id`'s host_in."""
        c, p = self.config, self.params
        if c == 0: return inputgen.config0_job(job_id, p[0]).view(np.uint8)
        if c == 1: return inputgen.config1_job(job_id, p[0]).view(np.uint8)
        if c == 2: return inputgen.config2_job(job_id, p[0], p[1]).reshape(-1).view(np.uint8)
        if c == 3: return inputgen.config3_pack(*inputgen.config3_job(job_id, p[0], p[1], p[2]))
        if c == 4:
            d = self.dims(job_id)
            return inputgen.config4_job(job_id, (d[0], d[1])).reshape(-1)
        if c == 5: return inputgen.sssp_job(job_id, p[0], self.extra.get("mean_deg", 8)).view(np.uint8)
        if c == 6:
            d = self.dims(job_id)
            return inputgen.sobel_frame(job_id, (d[0], d[1])).reshape(-1)
        raise ValueError(c)


def baseline_workload(config: int) -> Workload:
    """The workload exactly as BASELINE.json:configs[config] states it."""
    if config == 0:
        return Workload(0, (4096,), jobs=256, num_streams=4, max_inflight=8, name="config0 scan+hist64 (256 x 4096 int32)",
                        dtype="int32", kernels_per_job=2)
    if config == 1:
        return Workload(1, (16384,), jobs=10000, num_streams=8, max_inflight=32,
                        name="config1 short-lived fp32 kernel chain (10000 x 16384 fp32)", dtype="f32", kernels_per_job=5)
    if config == 2:
        return Workload(2, (4096, 4096, 10), jobs=512, num_streams=4, max_inflight=8,
                        name="config2 Jacobi 4096x4096 fp32 x10 sweeps (512 jobs)", dtype="f32", kernels_per_job=10)
    if config == 3:
        return Workload(3, (2048, 2048, 2048), jobs=1000, num_streams=4, max_inflight=8,
                        name="config3 bf16 GEMM 2048^3 + bias + GELU (1000 jobs)", dtype="bf16", kernels_per_job=1)
    if config == 4:
        return Workload(4, (1920, 1080), jobs=4096, num_streams=8, max_inflight=32,
                        name="config4 RGB frames gray->blur->hist256, jittered sizes (4096 jobs)", dtype="u8", kernels_per_job=3)
    if config == 5:  # paper workload 6; SURVEY.md 8(f)4
        return Workload(5, (4096, inputgen.sssp_max_edges(4096, 8)), jobs=2048, num_streams=8, max_inflight=32,
                        name="config5 SSSP frontier Bellman-Ford, 4096 vertices, mean out-degree 8, WHILE node (2048 jobs)", dtype="int32",
                        kernels_per_job=6, extra={"mean_deg": 8})  # graph kernel nodes: init + 4 relaxations + control
    if config == 6:  # paper workload 1; SURVEY.md 8(f)4
        return Workload(6, (1920, 1080), jobs=4096, num_streams=8, max_inflight=32,
                        name="config6 Sobel chain gray->sobel->mean->threshold->blend, jittered sizes (4096 jobs)", dtype="u8", kernels_per_job=5)
    raise ValueError(config)


def small_workload(config: int) -> Workload:
    """Reduced sizes the CPU oracle finishes in seconds; still several tiles plus a ragged tail."""
    if config == 0: return Workload(0, (4096,), jobs=64, num_streams=4, max_inflight=8, dtype="int32", kernels_per_job=2)
    if config == 1: return Workload(1, (16384,), jobs=200, num_streams=8, max_inflight=32, dtype="f32", kernels_per_job=5)
    if config == 2: return Workload(2, (300, 2052, 10), jobs=12, num_streams=4, max_inflight=8, dtype="f32", kernels_per_job=10)
    if config == 3: return Workload(3, (384, 512, 256), jobs=8, num_streams=4, max_inflight=8, dtype="bf16", kernels_per_job=1)
    if config == 4: return Workload(4, (1920, 1080), jobs=48, num_streams=8, max_inflight=32, dtype="u8", kernels_per_job=3)
    if config == 5: return Workload(5, (1000, inputgen.sssp_max_edges(1000, 4)), jobs=48, num_streams=4, max_inflight=8, dtype="int32", kernels_per_job=6, extra={"mean_deg": 4})
    if config == 6: return Workload(6, (1920, 1080), jobs=48, num_streams=8, max_inflight=32, dtype="u8", kernels_per_job=5)
    raise ValueError(config)


class PinnedArena:
    """Pinned host memory from set_host_alloc, carved into numpy views (no torch involved)."""

    def __init__(self, ctx, nbytes: int):
        self.ctx = ctx
        self.nbytes = int(nbytes)
        self.ptr = ctx.host_alloc(self.nbytes)
        self.view = np.ctypeslib.as_array((C.c_uint8 * self.nbytes).from_address(self.ptr))
        self.off = 0

    def take(self, nbytes: int, align: int = 256):
        """(address, uint8 view) of the next `nbytes` block."""
        self.off = (self.off + align - 1) // align * align
        if self.off + nbytes > self.nbytes:
            raise MemoryError("pinned arena exhausted")
        a, v = self.ptr + self.off, self.view[self.off:self.off + nbytes]
        self.off += nbytes
        return a, v

    def free(self):
        if self.ptr:
            self.view = None
            self.ctx.host_free(self.ptr)
            self.ptr = 0
