"""Seeded synthetic input generators for the five workloads (BASELINE.json:configs[0..4]).

This module is shared test/bench infrastructure.  It holds NONE of the method's
arithmetic: it only draws inputs.  Both the CPU oracle's tests and the CUDA
path's tests/bench feed on it; neither `oracle/` nor `paper_2606_05495_b200/`
is imported here.

Generator (SURVEY.md §8(d) "Synthetic inputs"): one counter-based 64-bit mixer
(splitmix64 finaliser) keyed by (config, job_id, stream_tag); element i of a
stream is mix(key + (i+1)*GOLDEN).  Uniform values come from the top 24 bits,
Gaussians from Box-Muller evaluated in double and then cast.
"""
from __future__ import annotations

import numpy as np

GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)

# Frame sizes of config 4 (W, H), BASELINE.json:configs[4].
FRAME_SIZES = ((640, 480), (1280, 720), (1920, 1080))


def _mix(z: np.ndarray) -> np.ndarray:
    z = (z ^ (z >> np.uint64(30))) * _M1
    z = (z ^ (z >> np.uint64(27))) * _M2
    return z ^ (z >> np.uint64(31))


def _key(config: int, job_id: int, tag: int) -> np.uint64:
    with np.errstate(over="ignore"):
        k = np.array([(config + 1) * 0x100000001B3 + tag], dtype=np.uint64)
        k = _mix(k + GOLDEN)
        k = _mix(k ^ np.uint64(job_id & 0xFFFFFFFFFFFFFFFF))
    return k[0]


def raw_u64(config: int, job_id: int, tag: int, n: int) -> np.ndarray:
    """n 64-bit words of stream (config, job_id, tag)."""
    with np.errstate(over="ignore"):
        ctr = np.arange(1, n + 1, dtype=np.uint64) * GOLDEN + _key(config, job_id, tag)
        return _mix(ctr)


def uniform24(config: int, job_id: int, tag: int, n: int) -> np.ndarray:
    """n integers uniform in [0, 2^24) (top 24 bits of each word)."""
    return (raw_u64(config, job_id, tag, n) >> np.uint64(40)).astype(np.int64)


def uniform_unit(config: int, job_id: int, tag: int, n: int) -> np.ndarray:
    """n doubles uniform in [0, 1)."""
    return uniform24(config, job_id, tag, n).astype(np.float64) / float(1 << 24)


def gaussian(config: int, job_id: int, tag: int, n: int) -> np.ndarray:
    """n standard normal doubles (Box-Muller on two uniform streams)."""
    m = (n + 1) // 2
    u1 = (uniform24(config, job_id, tag, m).astype(np.float64) + 1.0) / float(1 << 24)  # (0,1]
    u2 = uniform_unit(config, job_id, tag + 0x5151, m)
    r = np.sqrt(-2.0 * np.log(u1))
    out = np.empty(2 * m, dtype=np.float64)
    out[0::2] = r * np.cos(2.0 * np.pi * u2)
    out[1::2] = r * np.sin(2.0 * np.pi * u2)
    return out[:n]


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """fp32 -> bf16 bit patterns (uint16), round-to-nearest-even.  Input preparation only."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    u = (u + np.uint64(0x7FFF) + ((u >> np.uint64(16)) & np.uint64(1))) >> np.uint64(16)
    return u.astype(np.uint16)


def bf16_bits_to_f64(b: np.ndarray) -> np.ndarray:
    """bf16 bit patterns -> exact double values (comparison helper)."""
    return (b.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


# ---------------------------------------------------------------- per-config jobs
def config0_job(job_id: int, n: int = 4096) -> np.ndarray:
    """int32[n] uniform in [0,1000) (BASELINE.json:configs[0])."""
    return (uniform24(0, job_id, 0, n) * 1000 >> 24).astype(np.int32)


def config1_job(job_id: int, n: int = 16384) -> np.ndarray:
    """fp32[2n] = [x uniform[-1,1] | bias uniform[-1,1]] (configs[1])."""
    x = uniform_unit(1, job_id, 0, n) * 2.0 - 1.0
    b = uniform_unit(1, job_id, 1, n) * 2.0 - 1.0
    return np.concatenate([x, b]).astype(np.float32)


def config2_job(job_id: int, h: int = 4096, w: int = 4096) -> np.ndarray:
    """fp32[h][w] N(0,1) (configs[2])."""
    return gaussian(2, job_id, 0, h * w).astype(np.float32).reshape(h, w)


def config3_job(job_id: int, m: int = 2048, n: int = 2048, k: int = 2048):
    """(A bf16 bits [m][k], B bf16 bits [k][n], bias fp32 [n]) (configs[3])."""
    a = f32_to_bf16_bits((gaussian(3, job_id, 0, m * k) * 0.02).astype(np.float32)).reshape(m, k)
    b = f32_to_bf16_bits((gaussian(3, job_id, 1, k * n) * 0.02).astype(np.float32)).reshape(k, n)
    bias = gaussian(3, job_id, 2, n).astype(np.float32)
    return a, b, bias


def config3_pack(a: np.ndarray, b: np.ndarray, bias: np.ndarray) -> np.ndarray:
    """host_in byte image of a config-3 job: [A][B][bias]."""
    return np.concatenate([a.reshape(-1).view(np.uint8), b.reshape(-1).view(np.uint8),
                           bias.reshape(-1).view(np.uint8)])


def config4_size(job_id: int):
    """(W, H) of frame job_id, uniform over FRAME_SIZES (configs[4])."""
    return FRAME_SIZES[int(uniform24(4, job_id, 7, 1)[0] * 3 >> 24)]


def config4_job(job_id: int, size=None) -> np.ndarray:
    """uint8[H][W][3] interleaved RGB, pixels uniform in [0,256)."""
    w, h = size if size is not None else config4_size(job_id)
    n = h * w * 3
    words = raw_u64(4, job_id, 0, (n + 7) // 8)
    return words.view(np.uint8)[:n].reshape(h, w, 3).copy()


# ---------------------------------------------------------------- paper workloads 5 (SSSP) and 6 (Sobel chain)
def sssp_job(job_id: int, v: int = 4096, mean_deg: int = 8) -> np.ndarray:
    """int32 image [V, E, src, 0][row_ptr[V+1]][col[E]][w[E]] of one synthetic SSSP graph (stands in for the paper's SSSP
    inputs, which are not available): directed, out-degree uniform in 1 .. 2*mean_deg - 1, targets uniform
    over the vertices, weights uniform in 1 .. 100, source = vertex 0.  Vertices nobody points at stay unreachable."""
    deg = 1 + uniform24(5, job_id, 0, v) % (2 * mean_deg - 1)
    row_ptr = np.zeros(v + 1, dtype=np.int64)
    np.cumsum(deg, out=row_ptr[1:])
    e = int(row_ptr[-1])
    col = (uniform24(5, job_id, 1, e) % v).astype(np.int32)
    w = (1 + uniform24(5, job_id, 2, e) % 100).astype(np.int32)
    return np.concatenate([np.array([v, e, 0, 0], np.int32), row_ptr.astype(np.int32), col, w])


def sssp_edges(job_id: int, v: int = 4096, mean_deg: int = 8) -> int:
    """E of sssp_job(job_id, v, mean_deg) without building the graph."""
    return int((1 + uniform24(5, job_id, 0, v) % (2 * mean_deg - 1)).sum())


def sssp_max_edges(v: int, mean_deg: int = 8) -> int:
    return v * (2 * mean_deg - 1)


def sobel_frame(job_id: int, size=None) -> np.ndarray:
    """uint8[H][W][3] frame for the Sobel chain (stands in for the paper's Sobel images): 16 x 16 blocks of a
    random colour (high nibble) plus 4 bits of per-pixel noise, so that there are flat areas and sharp edges -- on pure
    noise (config 4's frames) every pixel is an edge and the threshold stage would be constant.  Sizes as config 4."""
    w, h = size if size is not None else config4_size(job_id)
    bw, bh = (w + 15) // 16, (h + 15) // 16
    blocks = raw_u64(6, job_id, 0, (bw * bh * 3 + 7) // 8).view(np.uint8)[:bw * bh * 3].reshape(bh, bw, 3) & np.uint8(0xF0)
    full = np.repeat(np.repeat(blocks, 16, axis=0), 16, axis=1)[:h, :w, :]
    n = h * w * 3
    noise = raw_u64(6, job_id, 1, (n + 7) // 8).view(np.uint8)[:n].reshape(h, w, 3) & np.uint8(0x0F)
    return (full | noise).copy()
