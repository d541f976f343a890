"""checker -- glue between a workload and the CPU oracle: the oracle's output image of one job (out_j = F(in_j),
SURVEY.md 8(c)) and the comparison rule of each workload (BASELINE.json:north_star tolerances).

TEST INFRASTRUCTURE, NOT PRODUCT: imported by tests/, __graft_entry__.smoke() and bench.py's spot check / cpu_baseline /
--impl reference legs only.  Nothing under paper_2606_05495_b200/ imports it (tests/test_abi.py enforces that), and it
holds no arithmetic of the method: every expected value comes from oracle/.
"""
from __future__ import annotations

import numpy as np

import inputgen
import oracle


def oracle_out(wl, in_image: np.ndarray, dims) -> np.ndarray:
    """uint8 byte image of the job's host_out as the oracle computes it."""
    c, p = wl.config, wl.params
    if c == 0:
        return oracle.config0(in_image.view(np.int32), hist_of_input=(wl.variant & 0xff) == 1)
    if c == 1:
        f = in_image.view(np.float32)
        return np.array([oracle.config1(f[:p[0]], f[p[0]:])], np.float32).view(np.uint8)
    if c == 2:
        return oracle.config2(in_image.view(np.float32).reshape(p[0], p[1]), p[2]).reshape(-1).view(np.uint8)
    if c == 3:
        m, n, k = p
        a = in_image[:2 * m * k].view(np.uint16).reshape(m, k)
        b = in_image[2 * m * k:2 * m * k + 2 * k * n].view(np.uint16).reshape(k, n)
        bias = in_image[2 * m * k + 2 * k * n:].view(np.float32)
        return oracle.config3(a, b, bias).reshape(-1).view(np.uint8)
    if c == 4:
        w, h = dims[0], dims[1]
        return oracle.config4(in_image.reshape(h, w, 3))
    if c == 5:
        return oracle.sssp_job(in_image, *p)
    if c == 6:
        w, h = dims[0], dims[1]
        return oracle.sobel_chain(in_image.reshape(h, w, 3))
    raise ValueError(c)


def compare(wl, out: np.ndarray, ref: np.ndarray) -> None:
    """Assert that the CUDA path's output image `out` matches the oracle's `ref` under the workload's rule: bit-exact for
    the integer workloads (configs 0, 4, 5, 6) and -- reading C2-3 -- for the Jacobi stencil; 1e-6 relative for the fp32
    scalar of config 1; 2e-2 relative Frobenius error for the bf16 GEMM (config 3)."""
    c = wl.config
    if c in (0, 4, 6):
        assert out.shape == ref.shape and np.array_equal(out, ref), _first_diff(out, ref)
    elif c == 5:
        # what is unique is compared bit for bit (the distances); the round count depends on the relaxation order (reading
        # S5-4): the GPU relaxes in place, so it needs at least one round and at most the oracle's synchronous count
        g, r = out.view(np.int32), ref.view(np.int32)
        assert g.shape == r.shape and np.array_equal(g[:-4], r[:-4]), _first_diff(out[:-16], ref[:-16])
        assert 1 <= g[-4] <= r[-4] and not g[-3:].any(), (g[-4:].tolist(), r[-4:].tolist())
    elif c == 1:
        g, r = float(out.view(np.float32)[0]), float(ref.view(np.float32)[0])
        assert abs(g - r) <= 1e-6 * abs(r), (g, r)
    elif c == 2:
        g, r = out.view(np.float32).astype(np.float64), ref.view(np.float32).astype(np.float64)
        scale = np.abs(r).max()
        assert np.abs(g - r).max() <= 1e-6 * scale                      # reading C2-4
        big = np.abs(r) >= 1e-3 * scale
        assert np.all(np.abs(g - r)[big] <= 1e-6 * np.abs(r)[big])
        assert np.array_equal(out, ref)                                  # reading C2-3: same add order -> bit-exact
    elif c == 3:
        g, r = inputgen.bf16_bits_to_f64(out.view(np.uint16)), inputgen.bf16_bits_to_f64(ref.view(np.uint16))
        assert np.linalg.norm(g - r) / np.linalg.norm(r) <= 2e-2
        assert np.abs(g - r).max() <= 0.05 * max(1.0, np.abs(r).max())  # no wild single entries either
    else:
        raise ValueError(c)


def _first_diff(out, ref):
    if out.shape != ref.shape:
        return f"shape {out.shape} vs {ref.shape}"
    bad = np.nonzero(out != ref)[0]
    return f"{bad.size} bytes differ, first at {bad[0]}: {out[bad[0]]} vs {ref[bad[0]]}" if bad.size else ""
