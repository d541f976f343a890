"""CPU oracle for the five SET workloads -- ctypes front end of oracle/*.c.

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It imports nothing from
paper_2606_05495_b200 and shares no code with the CUDA path.  See oracle.h for what is computed
and which passage / reading each function follows; tests/test_oracle_pins.py pins every function
to closed forms, invariants and brute force.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build as _build

_lib = C.CDLL(_build())
_p = C.c_void_p
_i64 = C.c_int64


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(_p)


_lib.oracle_scan_i32.argtypes = [_p, _i64, _p]
_lib.oracle_hist_mod.argtypes = [_p, _i64, C.c_int32, _p]
_lib.oracle_config0.argtypes = [_p, _i64, C.c_int, _p]
_lib.oracle_config1.argtypes = [_p, _p, _i64, _p]
_lib.oracle_config1.restype = C.c_float
_lib.oracle_config1_chain.argtypes = [_p, _p, _i64, _p, _p, _p, _p]
_lib.oracle_config1_chain.restype = None
_lib.oracle_jacobi5_sweep.argtypes = [_p, _i64, _i64, _p]
_lib.oracle_config2.argtypes = [_p, _i64, _i64, C.c_int, _p, _p]
_lib.oracle_bf16_to_f64.argtypes = [C.c_uint16]
_lib.oracle_bf16_to_f64.restype = C.c_double
_lib.oracle_f64_to_bf16_rne.argtypes = [C.c_double]
_lib.oracle_f64_to_bf16_rne.restype = C.c_uint16
_lib.oracle_gelu_erf.argtypes = [C.c_double]
_lib.oracle_gelu_erf.restype = C.c_double
_lib.oracle_gemm_z_at.argtypes = [_p, _p, _p, _i64, _i64, _i64, _i64]
_lib.oracle_gemm_z_at.restype = C.c_double
_lib.oracle_config3.argtypes = [_p, _p, _p, _i64, _i64, _i64, _p]
_lib.oracle_config3_sampled.argtypes = [_p, _p, _p, _i64, _i64, _p, _p, _i64, _p]
_lib.oracle_gray_u8.argtypes = [_p, _i64, _i64, _p]
_lib.oracle_blur3x3_u8.argtypes = [_p, _i64, _i64, _p]
_lib.oracle_hist256_u8.argtypes = [_p, _i64, _p]
_lib.oracle_config4.argtypes = [_p, _i64, _i64, _p, _p]
_lib.oracle_sssp_frontier_bf.argtypes = [_p, _p, _p, _i64, C.c_int32, _p, _p]
_lib.oracle_sssp_frontier_bf.restype = C.c_int32
_lib.oracle_sssp_job.argtypes = [_p, _p, _p]
_lib.oracle_sssp_job.restype = None
_lib.oracle_sobel_u8.argtypes = [_p, _i64, _i64, _p]
_lib.oracle_mean3x3_u8.argtypes = [_p, _i64, _i64, _p]
_lib.oracle_threshold_u8.argtypes = [_p, _i64, C.c_int32, _p]
_lib.oracle_blend_u8.argtypes = [_p, _p, _i64, _p]
_lib.oracle_sobel_chain.argtypes = [_p, _i64, _i64, _p, _p]


# ------------------------------------------------------------------ config 0
def scan_i32(v: np.ndarray) -> np.ndarray:
    v = np.ascontiguousarray(v, dtype=np.int32)
    out = np.empty_like(v)
    _lib.oracle_scan_i32(_ptr(v), v.size, _ptr(out))
    return out


def hist_mod(s: np.ndarray, bins: int = 64) -> np.ndarray:
    s = np.ascontiguousarray(s, dtype=np.int32)
    out = np.empty(bins, dtype=np.uint32)
    _lib.oracle_hist_mod(_ptr(s), s.size, bins, _ptr(out))
    return out


def config0(v: np.ndarray, hist_of_input: bool = False) -> np.ndarray:
    """Byte image [scan int32[n]][hist uint32[64]] of one config-0 job."""
    v = np.ascontiguousarray(v, dtype=np.int32)
    out = np.empty(v.size * 4 + 256, dtype=np.uint8)
    _lib.oracle_config0(_ptr(v), v.size, int(hist_of_input), _ptr(out))
    return out


# ------------------------------------------------------------------ config 1
def config1(x: np.ndarray, bias: np.ndarray, want_t4: bool = False):
    x = np.ascontiguousarray(x, dtype=np.float32)
    bias = np.ascontiguousarray(bias, dtype=np.float32)
    assert x.size == bias.size
    t4 = np.empty_like(x) if want_t4 else None
    r = _lib.oracle_config1(_ptr(x), _ptr(bias), x.size, _ptr(t4) if want_t4 else None)
    r = np.float32(r)
    return (r, t4) if want_t4 else r


def config1_chain(x: np.ndarray, bias: np.ndarray):
    """(t1, t2, t3, t4): the four elementwise stages of config 1, every intermediate (reading C1-1)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    bias = np.ascontiguousarray(bias, dtype=np.float32)
    assert x.size == bias.size
    t = [np.empty_like(x) for _ in range(4)]
    _lib.oracle_config1_chain(_ptr(x), _ptr(bias), x.size, *[_ptr(a) for a in t])
    return tuple(t)


# ------------------------------------------------------------------ config 2
def jacobi5_sweep(u: np.ndarray) -> np.ndarray:
    u = np.ascontiguousarray(u, dtype=np.float32)
    out = np.empty_like(u)
    _lib.oracle_jacobi5_sweep(_ptr(u), u.shape[0], u.shape[1], _ptr(out))
    return out


def config2(u: np.ndarray, sweeps: int = 10) -> np.ndarray:
    u = np.ascontiguousarray(u, dtype=np.float32)
    out = np.empty_like(u)
    tmp = np.empty_like(u)
    _lib.oracle_config2(_ptr(u), u.shape[0], u.shape[1], sweeps, _ptr(out), _ptr(tmp))
    return out


# ------------------------------------------------------------------ config 3
def bf16_to_f64(b: int) -> float:
    return float(_lib.oracle_bf16_to_f64(int(b)))


def f64_to_bf16_rne(x: float) -> int:
    return int(_lib.oracle_f64_to_bf16_rne(float(x)))


def gelu_erf(z: float) -> float:
    return float(_lib.oracle_gelu_erf(float(z)))


def gemm_z_at(a: np.ndarray, b: np.ndarray, bias: np.ndarray, m: int, n: int) -> float:
    a = np.ascontiguousarray(a, dtype=np.uint16)
    b = np.ascontiguousarray(b, dtype=np.uint16)
    bias = np.ascontiguousarray(bias, dtype=np.float32)
    return float(_lib.oracle_gemm_z_at(_ptr(a), _ptr(b), _ptr(bias), b.shape[1], b.shape[0], m, n))


def config3(a: np.ndarray, b: np.ndarray, bias: np.ndarray) -> np.ndarray:
    """a: bf16 bits [M][K], b: bf16 bits [K][N], bias fp32 [N] -> bf16 bits [M][N]."""
    a = np.ascontiguousarray(a, dtype=np.uint16)
    b = np.ascontiguousarray(b, dtype=np.uint16)
    bias = np.ascontiguousarray(bias, dtype=np.float32)
    m, k = a.shape
    k2, n = b.shape
    assert k == k2 and bias.size == n
    c = np.empty((m, n), dtype=np.uint16)
    _lib.oracle_config3(_ptr(a), _ptr(b), _ptr(bias), m, n, k, _ptr(c))
    return c


def config3_sampled(a, b, bias, ms, ns) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.uint16)
    b = np.ascontiguousarray(b, dtype=np.uint16)
    bias = np.ascontiguousarray(bias, dtype=np.float32)
    ms = np.ascontiguousarray(ms, dtype=np.int64)
    ns = np.ascontiguousarray(ns, dtype=np.int64)
    out = np.empty(ms.size, dtype=np.uint16)
    _lib.oracle_config3_sampled(_ptr(a), _ptr(b), _ptr(bias), b.shape[1], b.shape[0],
                                _ptr(ms), _ptr(ns), ms.size, _ptr(out))
    return out


# ------------------------------------------------------------------ config 4
def gray_u8(rgb: np.ndarray) -> np.ndarray:
    rgb = np.ascontiguousarray(rgb, dtype=np.uint8)
    h, w, _ = rgb.shape
    out = np.empty((h, w), dtype=np.uint8)
    _lib.oracle_gray_u8(_ptr(rgb), h, w, _ptr(out))
    return out


def blur3x3_u8(g: np.ndarray) -> np.ndarray:
    g = np.ascontiguousarray(g, dtype=np.uint8)
    out = np.empty_like(g)
    _lib.oracle_blur3x3_u8(_ptr(g), g.shape[0], g.shape[1], _ptr(out))
    return out


def hist256_u8(p: np.ndarray) -> np.ndarray:
    p = np.ascontiguousarray(p, dtype=np.uint8)
    out = np.empty(256, dtype=np.uint32)
    _lib.oracle_hist256_u8(_ptr(p), p.size, _ptr(out))
    return out


def config4(rgb: np.ndarray) -> np.ndarray:
    """Byte image [blur uint8[h*w]][hist uint32[256]] of one config-4 frame."""
    rgb = np.ascontiguousarray(rgb, dtype=np.uint8)
    h, w, _ = rgb.shape
    tmp = np.empty(h * w, dtype=np.uint8)
    out = np.empty(h * w + 1024, dtype=np.uint8)
    _lib.oracle_config4(_ptr(rgb), h, w, _ptr(tmp), _ptr(out))
    return out


# ------------------------------------------------------------------ config 5: SSSP
SSSP_INF = 0x7FFFFFFF


def sssp_frontier_bf(row_ptr, col, w, src: int = 0):
    """(dist int32[V], rounds): frontier Bellman-Ford with synchronous rounds (readings S5-1..S5-4)."""
    row_ptr = np.ascontiguousarray(row_ptr, dtype=np.int32)
    col = np.ascontiguousarray(col, dtype=np.int32)
    w = np.ascontiguousarray(w, dtype=np.int32)
    v = row_ptr.size - 1
    dist = np.empty(max(v, 0), dtype=np.int32)
    scratch = np.empty(3 * max(v, 1), dtype=np.int32)
    rounds = _lib.oracle_sssp_frontier_bf(_ptr(row_ptr), _ptr(col), _ptr(w), v, src, _ptr(dist), _ptr(scratch))
    return dist, int(rounds)


def sssp_job(image: np.ndarray, *_params) -> np.ndarray:
    """Byte image [dist int32[V]][rounds, 0, 0, 0] of one config-5 job; image = [V, E, src, 0][row_ptr][col][w]."""
    img = np.ascontiguousarray(image).view(np.int32)
    v = int(img[0])
    out = np.empty(v + 4, dtype=np.int32)
    scratch = np.empty(3 * max(v, 1), dtype=np.int32)
    _lib.oracle_sssp_job(_ptr(img), _ptr(out), _ptr(scratch))
    return out.view(np.uint8)


# ------------------------------------------------------------------ config 6: Sobel chain
def sobel_u8(n: np.ndarray) -> np.ndarray:
    n = np.ascontiguousarray(n, dtype=np.uint8)
    out = np.empty_like(n)
    _lib.oracle_sobel_u8(_ptr(n), n.shape[0], n.shape[1], _ptr(out))
    return out


def mean3x3_u8(e: np.ndarray) -> np.ndarray:
    e = np.ascontiguousarray(e, dtype=np.uint8)
    out = np.empty_like(e)
    _lib.oracle_mean3x3_u8(_ptr(e), e.shape[0], e.shape[1], _ptr(out))
    return out


def threshold_u8(m: np.ndarray, thresh: int = 64) -> np.ndarray:
    m = np.ascontiguousarray(m, dtype=np.uint8)
    out = np.empty_like(m)
    _lib.oracle_threshold_u8(_ptr(m), m.size, thresh, _ptr(out))
    return out


def blend_u8(t: np.ndarray, n: np.ndarray) -> np.ndarray:
    t = np.ascontiguousarray(t, dtype=np.uint8)
    n = np.ascontiguousarray(n, dtype=np.uint8)
    assert t.size == n.size
    out = np.empty_like(t)
    _lib.oracle_blend_u8(_ptr(t), _ptr(n), t.size, _ptr(out))
    return out


def sobel_chain(rgb: np.ndarray) -> np.ndarray:
    """uint8[h*w]: the blended output of one config-6 frame (flat byte image)."""
    rgb = np.ascontiguousarray(rgb, dtype=np.uint8)
    h, w, _ = rgb.shape
    tmp = np.empty(3 * h * w, dtype=np.uint8)
    out = np.empty(h * w, dtype=np.uint8)
    _lib.oracle_sobel_chain(_ptr(rgb), h, w, _ptr(tmp), _ptr(out))
    return out
