"""Build libset.so (the C-ABI library) in-tree with nvcc for sm_100a.

    python -m paper_2606_05495_b200.build [--force]

nvcc cross-compiles without a GPU.  The built .so is git-ignored but travels to the GPU box with gpurun.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libset.so")
TRACE_LIB = os.path.join(HERE, "libsettrace.so")  # CUPTI gap tracer (include/set_trace.h): measurement only
BUILD_DIR = os.path.join(HERE, "build")

CUDA_SOURCES = ["kernels/small_kernels.cu", "kernels/stencil_kernels.cu", "kernels/paper_kernels.cu", "kernels/gemm_sm100.cu", "set_builtin.cu", "set_noalloc.cu"]
HOST_SOURCES = ["set_cuda.cpp", "set_selftest.cpp", "set_multi.cpp"]
HEADERS = ["set_core.hpp", "set_ring.hpp", "kernels/kernels.h"]

NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC,-Wall,-Wextra,-pthread", "-I", INCLUDE]
# -fmad=false: no FMA contraction anywhere in the stage kernels (reading C1-1); the GEMM's MMA is
# issued through tcgen05 PTX and is not affected.
DEVICE_FLAGS = ["-fmad=false", "-Xptxas", "-v"]
# the GEMM's epilogue (bias + erf-GELU in fp32, tolerance 2e-2 Frobenius) may contract; the accumulation is tcgen05's
FMA_OK = {"kernels/gemm_sm100.cu"}


def _stale(target: str, deps: list[str]) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(BUILD_DIR, exist_ok=True)
    hdrs = [os.path.join(CSRC, h) for h in HEADERS] + [os.path.join(INCLUDE, "set.h"), os.path.abspath(__file__)]
    objs = []
    for src in CUDA_SOURCES + HOST_SOURCES:
        path = os.path.join(CSRC, src)
        obj = os.path.join(BUILD_DIR, src.replace("/", "_") + ".o")
        objs.append(obj)
        if force or _stale(obj, [path] + hdrs):
            cmd = [NVCC] + ARCH + COMMON + ([f for f in DEVICE_FLAGS if not (f == "-fmad=false" and src in FMA_OK)] if src.endswith(".cu") else ["-x", "cu"]) + ["-c", path, "-o", obj]
            r = subprocess.run(cmd, capture_output=True, text=True)
            if verbose or r.returncode != 0:
                sys.stderr.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
            if r.returncode != 0:
                raise RuntimeError(f"nvcc failed on {src}")
            with open(obj + ".log", "w") as f:
                f.write(r.stdout + r.stderr)
    if force or _stale(LIB, objs):
        cmd = [NVCC] + ARCH + ["-shared", "-o", LIB] + objs + ["-Xcompiler", "-pthread", "-cudart", "static", "-lpthread", "-ldl", "-lrt"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            sys.stderr.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
            raise RuntimeError("link failed")
    build_trace(force)
    return LIB


def build_trace(force: bool = False) -> str:
    """libsettrace.so: host-only C++ against the CUPTI headers; libcupti itself is dlopen'ed at run time."""
    src = os.path.join(CSRC, "set_trace.cpp")
    if force or _stale(TRACE_LIB, [src, os.path.join(INCLUDE, "set_trace.h"), os.path.abspath(__file__)]):
        cuda = os.path.dirname(os.path.dirname(os.path.realpath(NVCC)))
        cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-Wall", "-Wextra", "-I", INCLUDE, "-I", os.path.join(cuda, "include"),
               "-o", TRACE_LIB, src, "-ldl", "-lpthread"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            sys.stderr.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
            raise RuntimeError("building libsettrace.so failed")
    return TRACE_LIB


def build_selftest(sanitizer: str = "thread") -> str:
    """csrc/selftest_main.cpp + set_selftest.cpp (header-only scheduler core, no CUDA) with -fsanitize=<sanitizer>:
    the lock-free ring and Algorithms 1-3 against a simulated device under ThreadSanitizer / AddressSanitizer."""
    os.makedirs(BUILD_DIR, exist_ok=True)
    exe = os.path.join(BUILD_DIR, f"selftest_{sanitizer.replace(',', '_')}")
    srcs = [os.path.join(CSRC, "selftest_main.cpp"), os.path.join(CSRC, "set_selftest.cpp")]
    deps = srcs + [os.path.join(CSRC, h) for h in ("set_core.hpp", "set_ring.hpp")] + [os.path.join(INCLUDE, "set.h")]
    if _stale(exe, deps):
        cmd = ["g++", "-O1", "-g", "-std=c++17", f"-fsanitize={sanitizer}", "-pthread", "-I", INCLUDE, "-o", exe] + srcs
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            sys.stderr.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
            raise RuntimeError("building the sanitizer self test failed")
    return exe


if __name__ == "__main__":
    if "--selftest" in sys.argv:
        print(build_selftest(sys.argv[sys.argv.index("--selftest") + 1]))
    else:
        print(build(force="--force" in sys.argv, verbose=True))
