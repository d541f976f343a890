"""tests-only glue: the CPU oracle's output image for one job of a workload (out_j = F(in_j))."""
import numpy as np

import oracle


def oracle_out(wl, in_image: np.ndarray, dims) -> np.ndarray:
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
    raise ValueError(c)
