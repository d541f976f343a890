"""Pins for the CPU oracle: every oracle function is checked against something other than itself --
closed forms, invariants, textbook constants (tests/golden/), library routines on special cases, and
pure-Python brute force on tiny inputs.  SURVEY.md §8(c) lists the pins per config.  CPU only."""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

import inputgen
import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _golden(name):
    rows = {}
    for line in open(os.path.join(GOLD, name)):
        line = line.split("#")[0].split()
        if line:
            rows.setdefault(line[0], []).append([float(x) for x in line[1:]])
    return rows


# =============================================================== config 0: scan + hist64
def test_c0_scan_last_is_sum_and_differences():
    v = inputgen.config0_job(11)
    s = oracle.scan_i32(v)
    assert int(s[-1]) == int(v.astype(np.int64).sum())
    assert s[0] == v[0]
    assert np.array_equal(np.diff(s.astype(np.int64)), v[1:].astype(np.int64))


def test_c0_all_ones_closed_form():
    v = np.ones(4096, np.int32)
    s = oracle.scan_i32(v)
    assert np.array_equal(s, np.arange(1, 4097, dtype=np.int32))
    h = oracle.hist_mod(s, 64)
    assert np.array_equal(h, np.full(64, 64, np.uint32))


def test_c0_bruteforce_tiny():
    for n in (1, 2, 7, 33, 64):
        v = inputgen.config0_job(100 + n, n)
        s = oracle.scan_i32(v)
        brute = [sum(int(v[k]) for k in range(i + 1)) for i in range(n)]  # O(n^2)
        assert s.tolist() == brute
        h = oracle.hist_mod(s, 64)
        hb = [sum(1 for x in brute if x % 64 == b) for b in range(64)]
        assert h.tolist() == hb


def test_c0_hist_mass_and_input_variant_closed_form():
    n = 4096
    v = (np.arange(n) % 1000).astype(np.int32)
    out = oracle.config0(v, hist_of_input=True)
    h = out[n * 4:].view(np.uint32)
    assert int(h.sum()) == n
    # per full thousand: values 0..999 -> 16 per bin for b<40 (1000 = 15*64+40), 15 for b>=40;
    # 4096 = 4 thousands + the values 0..95 (one more for every bin, one more again for b<32)
    expect = np.array([4 * (16 if b < 40 else 15) + 1 + (1 if b < 32 else 0) for b in range(64)], np.uint32)
    assert np.array_equal(h, expect)


def test_c0_chain_layout_and_stage_order():
    v = inputgen.config0_job(5)
    out = oracle.config0(v)
    assert out.size == 4096 * 4 + 256
    scan = out[:4096 * 4].view(np.int32)
    hist = out[4096 * 4:].view(np.uint32)
    assert np.array_equal(scan, np.cumsum(v.astype(np.int64)).astype(np.int32))  # library routine
    assert np.array_equal(hist, np.bincount(scan % 64, minlength=64).astype(np.uint32))
    assert int(hist.sum()) == 4096
    # reading C0-1: the histogram of the scan differs from the histogram of the input
    assert not np.array_equal(hist, np.bincount(v % 64, minlength=64).astype(np.uint32))


def test_c0_empty_and_single():
    assert oracle.scan_i32(np.zeros(0, np.int32)).size == 0
    assert oracle.hist_mod(np.zeros(0, np.int32)).sum() == 0
    assert oracle.scan_i32(np.array([7], np.int32)).tolist() == [7]


# =============================================================== config 1: fp32 chain + sum
def test_c1_zero_input_golden():
    g = _golden("config1_zero_input.txt")
    z = np.zeros(16384, np.float32)
    r, t4 = oracle.config1(z, z, want_t4=True)
    assert np.all(t4 == np.float32(g["t4"][0][0]))
    assert float(t4[0]) == g["t4"][0][0]
    assert float(r) == g["sum"][0][0]
    # the golden numbers themselves follow from exact rational arithmetic
    tenth = Fraction(float(np.float32(0.1)))
    sq = float(np.float32(float(tenth * tenth)))  # exact product -> one rounding to fp32 (double holds 48 bits)
    assert sq == g["t4"][0][0]
    assert float(np.float32(sq * 16384)) == g["sum"][0][0]


def test_c1_relu_kills_negative_branch():
    x = np.full(16384, -1.0, np.float32)
    assert float(oracle.config1(x, np.zeros_like(x))) == 0.0
    # bias is added BEFORE the ReLU: bias = +3 revives it: (2.5*-1+0.1+3)^2 = 0.6^2
    r = oracle.config1(x, np.full_like(x, 3.0))
    assert abs(float(r) / 16384 - 0.36) < 1e-6


def test_c1_each_step_is_one_fp32_rounding():
    j = inputgen.config1_job(3)
    x, b = j[:16384], j[16384:]
    _, t4 = oracle.config1(x, b, want_t4=True)
    # independent route: evaluate every step exactly in double (operands are fp32, so product and sums are
    # exact in double for these magnitudes) and round ONCE to fp32
    xd, bd = x.astype(np.float64), b.astype(np.float64)
    m = (2.5 * xd).astype(np.float32)
    t1 = (m.astype(np.float64) + float(np.float32(0.1))).astype(np.float32)
    t2 = (t1.astype(np.float64) + bd).astype(np.float32)
    t3 = np.maximum(t2, np.float32(0))
    t4r = (t3.astype(np.float64) ** 2).astype(np.float32)
    assert np.array_equal(t4, t4r)
    # and it is NOT the fused evaluation fl(2.5*x + 0.1) (reading C1-1): some elements must differ
    fused = (2.5 * xd + float(np.float32(0.1))).astype(np.float32)
    assert np.count_nonzero(fused != t1) > 100


def test_c1_chain_intermediates_each_one_rounding():
    """oracle_config1_chain (what K3..K6 are compared with element by element): every intermediate against the
    single-rounding route through double, and t4 against oracle_config1's own t4."""
    for job in (3, 11):
        j = inputgen.config1_job(job)
        x, b = j[:16384], j[16384:]
        t1, t2, t3, t4 = oracle.config1_chain(x, b)
        xd, bd = x.astype(np.float64), b.astype(np.float64)
        m = (2.5 * xd).astype(np.float32)
        r1 = (m.astype(np.float64) + float(np.float32(0.1))).astype(np.float32)
        r2 = (r1.astype(np.float64) + bd).astype(np.float32)
        r3 = np.where(r2 > 0, r2, np.float32(0)).astype(np.float32)
        r4 = (r3.astype(np.float64) * r3.astype(np.float64)).astype(np.float32)
        assert np.array_equal(t1, r1) and np.array_equal(t2, r2) and np.array_equal(t3, r3) and np.array_equal(t4, r4)
        assert np.array_equal(t4, oracle.config1(x, b, want_t4=True)[1])
        assert (t3 >= 0).all() and np.count_nonzero(t3 == 0) > 1000 and np.count_nonzero(t2 < 0) == np.count_nonzero(t3 == 0) - np.count_nonzero(t2 == 0)
        # a contracted fma(2.5, x, 0.1) would differ from t1 in many elements (reading C1-1)
        fused = (2.5 * xd + float(np.float32(0.1))).astype(np.float32)
        assert np.count_nonzero(fused != t1) > 100
    # tiny hand case: x = 0.5, bias = -2 -> t1 = fl(1.25 + 0.1f), t2 < 0, t3 = 0, t4 = 0
    t1, t2, t3, t4 = oracle.config1_chain(np.array([0.5], np.float32), np.array([-2.0], np.float32))
    assert float(t1[0]) == float(np.float32(1.25) + np.float32(0.1)) and t2[0] < 0 and t3[0] == 0 and t4[0] == 0


def test_c1_sum_in_double_vs_independent_double_chain():
    for job in (0, 1, 2):
        j = inputgen.config1_job(job)
        x, b = j[:16384], j[16384:]
        r, t4 = oracle.config1(x, b, want_t4=True)
        assert float(r) >= 0.0
        assert float(r) == float(np.float32(math.fsum(t4.astype(np.float64).tolist())))  # exact sum, one rounding
        dbl = np.maximum(2.5 * x.astype(np.float64) + 0.1 + b.astype(np.float64), 0.0) ** 2
        assert abs(float(r) - dbl.sum()) <= 1e-6 * dbl.sum()


def test_c1_tiny_python_bruteforce():
    x = np.array([0.5, -0.25, 0.75, -1.0, 0.0], np.float32)
    b = np.array([0.0, 1.0, -3.0, 2.45, -0.1], np.float32)
    f = np.float32
    acc = 0.0
    for xi, bi in zip(x, b):
        t = f(f(f(2.5) * xi) + f(0.1))
        t = f(t + bi)
        t = t if t > 0 else f(0)
        acc += float(f(t * t))
    assert float(oracle.config1(x, b)) == float(f(acc))


# =============================================================== config 2: Jacobi
def test_c2_constant_field_interior_and_zero_halo_edges():
    u = np.ones((16, 16), np.float32)
    o = oracle.jacobi5_sweep(u)
    assert np.all(o[1:-1, 1:-1] == np.float32(1.0))           # fl(0.2f*5) == 1
    f = np.float32
    assert o[0, 0] == f(0.2) * f(3) and o[0, 15] == f(0.2) * f(3) and o[15, 0] == f(0.2) * f(3)
    assert np.all(o[0, 1:-1] == f(0.2) * f(4)) and np.all(o[1:-1, 0] == f(0.2) * f(4))
    assert np.all(o[-1, 1:-1] == f(0.2) * f(4)) and np.all(o[1:-1, -1] == f(0.2) * f(4))
    for t in (2, 3, 5):
        o = oracle.config2(np.ones((32, 32), np.float32), t)
        assert np.all(o[t:-t, t:-t] == np.float32(1.0))
        assert o[t - 1, 16] != np.float32(1.0)


def _walks(t, dx, dy):
    """number of t-step walks over {stay, +-x, +-y} ending at (dx, dy) -- multinomial count"""
    cnt = 0
    for r in range(t + 1):              # right
        l = r - dx
        if l < 0: continue
        for up in range(t + 1 - r - l):
            d = up - dy
            if d < 0: continue
            s = t - r - l - up - d
            if s < 0: continue
            cnt += math.factorial(t) // (math.factorial(r) * math.factorial(l) * math.factorial(up)
                                         * math.factorial(d) * math.factorial(s))
    return cnt


def test_c2_unit_impulse_walk_counts_and_mass():
    n = 33
    u = np.zeros((n, n), np.float32)
    u[16, 16] = 1.0
    o2 = oracle.config2(u, 2).astype(np.float64)
    expect = {(0, 0): 5, (1, 0): 2, (0, 1): 2, (2, 0): 1, (0, 2): 1, (1, 1): 2, (2, 1): 0}
    for (dy, dx), c in expect.items():
        for sy in (1, -1):
            for sx in (1, -1):
                assert abs(o2[16 + sy * dy, 16 + sx * dx] - c / 25.0) <= 1e-6 * max(c / 25.0, 1e-30)
    for t in (1, 3, 4, 7):
        o = oracle.config2(u, t).astype(np.float64)
        for dy in range(-t - 1, t + 2):
            for dx in range(-t - 1, t + 2):
                want = _walks(t, dx, dy) * 0.2 ** t
                assert abs(o[16 + dy, 16 + dx] - want) <= 2e-6 * want + 1e-30
        assert abs(o.sum() - 1.0) < 1e-5            # mass conserved while it has not reached the edge
    # near the edge the zero halo loses mass
    e = np.zeros((8, 8), np.float32); e[0, 0] = 1.0
    assert abs(oracle.config2(e, 1).astype(np.float64).sum() - 0.6) < 1e-6


def test_c2_scaling_by_two_is_exact():
    u = inputgen.config2_job(7, 64, 48)
    a = oracle.config2(u, 10)
    b = oracle.config2(u * np.float32(2), 10)
    assert np.array_equal(b, a * np.float32(2))


def test_c2_association_order_pin():
    # ((c + w) + e): c=1e8, w=-1e8, e=1 -> 1 ; the other order c+(w+e) would give 0 in fp32
    u = np.zeros((3, 3), np.float32)
    u[1, 1], u[1, 0], u[1, 2] = 1e8, -1e8, 1.0
    o = oracle.jacobi5_sweep(u)
    assert o[1, 1] == np.float32(0.2) * np.float32(1.0)
    # n and s enter after w and e: c=1, w=1e8, e=-1e8 (cancel first), n=3, s=5 -> 0.2*9
    u = np.zeros((3, 3), np.float32)
    u[1, 1], u[1, 0], u[1, 2], u[0, 1], u[2, 1] = 1.0, 1e8, -1e8, 3.0, 5.0
    # (1+1e8) = 1e8 in fp32, + -1e8 = 0, +3 +5 = 8
    assert oracle.jacobi5_sweep(u)[1, 1] == np.float32(0.2) * np.float32(8.0)


def test_c2_fp64_bruteforce_8x8_and_nonsquare():
    for (h, w) in ((8, 8), (5, 9)):
        u = inputgen.config2_job(3, h, w)
        ref = [[float(u[i, j]) for j in range(w)] for i in range(h)]
        for _ in range(10):
            g = lambda i, j: ref[i][j] if 0 <= i < h and 0 <= j < w else 0.0
            ref = [[0.2 * (g(i, j) + g(i, j - 1) + g(i, j + 1) + g(i - 1, j) + g(i + 1, j)) for j in range(w)]
                   for i in range(h)]
        o = oracle.config2(u, 10).astype(np.float64)
        ref = np.array(ref)
        assert np.abs(o - ref).max() <= 1e-6 * np.abs(ref).max()


def test_c2_sweep_parity_and_input_untouched():
    u = inputgen.config2_job(1, 12, 12)
    keep = u.copy()
    s = u
    for t in range(0, 5):
        assert np.array_equal(oracle.config2(u, t), s)
        s = oracle.jacobi5_sweep(s)
    assert np.array_equal(u, keep)


# =============================================================== config 3: GEMM + bias + GELU
def test_c3_gelu_textbook_values():
    for line in open(os.path.join(GOLD, "gelu_values.txt")):
        line = line.split("#")[0].split()
        if line:
            z, want = float(line[0]), float(line[1])
            assert abs(oracle.gelu_erf(z) - want) < 5e-8
    # identity GELU(z) - GELU(-z) = z
    for z in (0.3, 1.7, 4.0):
        assert abs(oracle.gelu_erf(z) - oracle.gelu_erf(-z) - z) < 1e-14


def test_c3_bf16_rounding_rne():
    assert oracle.f64_to_bf16_rne(1.0) == 0x3F80
    assert oracle.f64_to_bf16_rne(1.0 + 2 ** -8) == 0x3F80          # tie -> even (down)
    assert oracle.f64_to_bf16_rne(1.0 + 3 * 2 ** -8) == 0x3F82      # tie -> even (up)
    assert oracle.f64_to_bf16_rne(1.0 + 2 ** -8 + 2 ** -30) == 0x3F81
    assert oracle.f64_to_bf16_rne(-0.0) == 0x8000
    assert oracle.f64_to_bf16_rne(float("inf")) == 0x7F80
    assert oracle.f64_to_bf16_rne(1.9999999) == 0x4000               # carry into the exponent
    import torch
    x = (inputgen.gaussian(9, 0, 0, 20000) * np.exp(inputgen.gaussian(9, 0, 1, 20000) * 8)).astype(np.float32)
    want = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    got = np.array([oracle.f64_to_bf16_rne(float(v)) for v in x], np.uint16)
    assert np.array_equal(got, want)
    for b in (0x0001, 0x007F, 0x0080, 0x3F80, 0xC020, 0x7F7F):
        assert oracle.f64_to_bf16_rne(oracle.bf16_to_f64(b)) == b


def _c3_check(c_bits, z):
    want = np.array([oracle.f64_to_bf16_rne(0.5 * v * (1.0 + math.erf(v / math.sqrt(2.0)))) for v in z.ravel()],
                    np.uint16).reshape(z.shape)
    assert np.array_equal(c_bits, want)


def test_c3_identity_B_and_zero_A():
    m = n = k = 32
    a, _, bias = inputgen.config3_job(4, m, n, k)
    eye = inputgen.f32_to_bf16_bits(np.eye(k, dtype=np.float32)).reshape(k, n)
    c = oracle.config3(a, eye, bias)
    _c3_check(c, inputgen.bf16_bits_to_f64(a) + bias.astype(np.float64)[None, :])      # bias indexed by column n
    zero = np.zeros((m, k), np.uint16)
    _, b, _ = inputgen.config3_job(5, m, n, k)
    c = oracle.config3(zero, b, bias)
    _c3_check(c, np.broadcast_to(bias.astype(np.float64)[None, :], (m, n)))


def test_c3_nonsquare_vs_exact_fractions_and_library_matmul():
    m, n, k = 5, 7, 16
    a, b, bias = inputgen.config3_job(6, m, n, k)
    a = a.reshape(-1)[:m * k].reshape(m, k); b = b.reshape(-1)[:k * n].reshape(k, n); bias = bias[:n]
    ad, bd = inputgen.bf16_bits_to_f64(a), inputgen.bf16_bits_to_f64(b)
    for i in range(m):
        for j in range(n):
            exact = sum(Fraction(float(ad[i, kk])) * Fraction(float(bd[kk, j])) for kk in range(k)) \
                + Fraction(float(bias[j]))
            assert abs(oracle.gemm_z_at(a, b, bias, i, j) - float(exact)) <= 1e-15 * max(1.0, abs(float(exact)))
    m, n, k = 48, 80, 64     # all different: a transposed operand or swapped index cannot pass
    a, b, bias = inputgen.config3_job(7, m, n, k)
    # larger-magnitude operands so that A*B, not the bias, dominates z
    a = inputgen.f32_to_bf16_bits((inputgen.gaussian(3, 70, 0, m * k)).astype(np.float32)).reshape(m, k)
    b = inputgen.f32_to_bf16_bits((inputgen.gaussian(3, 70, 1, k * n) * 0.2).astype(np.float32)).reshape(k, n)
    z = inputgen.bf16_bits_to_f64(a) @ inputgen.bf16_bits_to_f64(b) + bias.astype(np.float64)[None, :]
    c = oracle.config3(a, b, bias)
    got = inputgen.bf16_bits_to_f64(c)
    want = 0.5 * z * (1.0 + np.vectorize(math.erf)(z / math.sqrt(2.0)))
    # equal up to the final bf16 rounding (2^-9 relative) -- and bit-equal wherever the library z is not
    # within 1e-12 of a rounding boundary
    assert np.abs(got - want).max() <= 2 ** -8 * np.abs(want).max()
    assert np.linalg.norm(got - want) / np.linalg.norm(want) < 3e-3
    ms = np.array([0, 47, 13, 5], np.int64); ns = np.array([79, 0, 40, 5], np.int64)
    assert np.array_equal(oracle.config3_sampled(a, b, bias, ms, ns), c[ms, ns])


# =============================================================== config 4: gray -> blur -> hist256
def test_c4_gray_weights_and_identity():
    v = np.arange(256, dtype=np.uint8)
    img = np.stack([v, v, v], axis=-1).reshape(16, 16, 3)
    assert np.array_equal(oracle.gray_u8(img).ravel(), v)                  # 77+150+29 = 256
    px = lambda r, g, b: int(oracle.gray_u8(np.array([[[r, g, b]]], np.uint8))[0, 0])
    assert px(255, 0, 0) == (77 * 255) >> 8 == 76
    assert px(0, 255, 0) == (150 * 255) >> 8 == 149
    assert px(0, 0, 255) == (29 * 255) >> 8 == 28
    assert px(1, 1, 0) == 0 and px(200, 100, 50) == (77 * 200 + 150 * 100 + 29 * 50) >> 8


def test_c4_blur_golden_impulse_and_clamp():
    g = _golden("blur_impulse.txt")
    img = np.zeros((9, 11), np.uint8); img[4, 5] = 255
    o = oracle.blur3x3_u8(img)
    assert o[3:6, 4:7].ravel().tolist() == [int(x) for x in g["interior"][0]]
    assert int(o.sum()) == sum(int(x) for x in g["interior"][0])
    img = np.zeros((6, 7), np.uint8); img[0, 0] = 255
    o = oracle.blur3x3_u8(img)
    assert [int(o[0, 0]), int(o[0, 1]), int(o[1, 0]), int(o[1, 1])] == [int(x) for x in g["corner"][0]]
    # constant image stays constant, borders included
    for val in (0, 1, 17, 255):
        c = np.full((7, 5), val, np.uint8)
        assert np.all(oracle.blur3x3_u8(c) == val)


def test_c4_blur_bruteforce_and_separable():
    for (h, w) in ((4, 5), (1, 1), (1, 6), (7, 1), (2, 2)):
        gimg = oracle.gray_u8(inputgen.config4_job(40 + h * w, (w, h)))
        o = oracle.blur3x3_u8(gimg)
        k = [[1, 2, 1], [2, 4, 2], [1, 2, 1]]
        for y in range(h):
            for x in range(w):
                acc = 0
                for dy in (-1, 0, 1):
                    for dx in (-1, 0, 1):
                        yy = min(max(y + dy, 0), h - 1); xx = min(max(x + dx, 0), w - 1)
                        acc += k[dy + 1][dx + 1] * int(gimg[yy, xx])
                assert int(o[y, x]) == acc >> 4
    gimg = oracle.gray_u8(inputgen.config4_job(3, (64, 48)))
    p = np.pad(gimg.astype(np.int32), 1, mode="edge")                      # library pad + separable passes
    rows = p[:, :-2] + 2 * p[:, 1:-1] + p[:, 2:]
    sep = (rows[:-2] + 2 * rows[1:-1] + rows[2:]) >> 4
    assert np.array_equal(oracle.blur3x3_u8(gimg), sep.astype(np.uint8))


def test_c4_chain_layout_and_hist_mass():
    f = inputgen.config4_job(9, (64, 48))
    out = oracle.config4(f)
    assert out.size == 64 * 48 + 1024
    blur = out[:64 * 48].reshape(48, 64)
    hist = out[64 * 48:].copy().view(np.uint32)
    assert int(hist.sum()) == 64 * 48
    assert np.array_equal(blur, oracle.blur3x3_u8(oracle.gray_u8(f)))
    assert np.array_equal(hist, np.bincount(blur.ravel(), minlength=256).astype(np.uint32))  # C4-4: of the blur
    assert np.array_equal(oracle.hist256_u8(np.array([0, 255, 255, 7], np.uint8))[[0, 7, 255]], [1, 1, 2])


# =============================================================== the generator is what DESIGN.md says it is
def test_inputgen_distributions():
    v = inputgen.config0_job(0)
    assert v.dtype == np.int32 and v.min() >= 0 and v.max() < 1000 and v.size == 4096
    assert not np.array_equal(v, inputgen.config0_job(1)) and np.array_equal(v, inputgen.config0_job(0))
    j = inputgen.config1_job(0)
    assert j.dtype == np.float32 and j.size == 32768 and j.min() >= -1 and j.max() <= 1 and abs(j.mean()) < 0.02
    u = inputgen.config2_job(0, 256, 256)
    assert abs(u.mean()) < 0.02 and abs(u.std() - 1) < 0.02
    a, b, bias = inputgen.config3_job(0, 64, 64, 64)
    assert abs(inputgen.bf16_bits_to_f64(a).std() - 0.02) < 2e-3 and abs(bias.std() - 1) < 0.3
    sizes = [inputgen.config4_size(j) for j in range(300)]
    assert set(sizes) == set(inputgen.FRAME_SIZES)
    f = inputgen.config4_job(0, (32, 16))
    assert f.shape == (16, 32, 3) and f.dtype == np.uint8 and abs(f.mean() - 127.5) < 8


# =============================================================== config 5: SSSP, frontier Bellman-Ford
def _csr(v, edges):
    """edges: list of (u, t, w) -> row_ptr, col, w in CSR order."""
    edges = sorted(edges, key=lambda e: e[0])
    row_ptr = np.zeros(v + 1, np.int32)
    for u, _, _ in edges:
        row_ptr[u + 1] += 1
    row_ptr = np.cumsum(row_ptr).astype(np.int32)
    return row_ptr, np.array([e[1] for e in edges], np.int32), np.array([e[2] for e in edges], np.int32)


def _dijkstra(v, row_ptr, col, w, src):
    import heapq
    dist = [oracle.SSSP_INF] * v
    dist[src] = 0
    pq = [(0, src)]
    while pq:
        d, u = heapq.heappop(pq)
        if d > dist[u]:
            continue
        for e in range(row_ptr[u], row_ptr[u + 1]):
            nd = d + int(w[e])
            if nd < dist[col[e]]:
                dist[col[e]] = nd
                heapq.heappush(pq, (nd, int(col[e])))
    return np.array(dist, np.int32)


def test_c5_path_graph_closed_form():
    # 0 -> 1 -> 2 -> ... -> 9 with weight 3: dist[k] = 3k, and the frontier needs one round per hop plus the round that
    # finds nothing left to improve (reading S5-3)
    v = 10
    rp, col, w = _csr(v, [(k, k + 1, 3) for k in range(v - 1)])
    dist, rounds = oracle.sssp_frontier_bf(rp, col, w, 0)
    assert dist.tolist() == [3 * k for k in range(v)]
    assert rounds == v                        # rounds 1..9 settle vertices 1..9, round 10 relaxes the last vertex's (no) edges
    # started in the middle: everything upstream is unreachable (reading S5-2)
    dist, _ = oracle.sssp_frontier_bf(rp, col, w, 4)
    assert dist.tolist() == [oracle.SSSP_INF] * 4 + [0, 3, 6, 9, 12, 15]


def test_c5_hand_graph_with_a_shortcut_found_late():
    # 0 -1-> 1 -1-> 2 -1-> 3 and the direct but dearer edge 0 -10-> 3; 3 -1-> 4.  The direct edge is seen first (round 1:
    # dist[3] = 10), the three-hop path wins in round 3 (dist[3] = 3) and vertex 4 is corrected in round 4.
    rp, col, w = _csr(5, [(0, 1, 1), (0, 3, 10), (1, 2, 1), (2, 3, 1), (3, 4, 1)])
    dist, rounds = oracle.sssp_frontier_bf(rp, col, w, 0)
    assert dist.tolist() == [0, 1, 2, 3, 4] and rounds == 5
    # zero-weight edges and a cycle do not loop for ever (weights >= 0, reading S5-1)
    rp, col, w = _csr(3, [(0, 1, 0), (1, 2, 0), (2, 0, 0)])
    dist, rounds = oracle.sssp_frontier_bf(rp, col, w, 0)
    assert dist.tolist() == [0, 0, 0] and rounds == 3
    # a source without edges: one round that relaxes nothing
    rp, col, w = _csr(3, [(1, 2, 5)])
    dist, rounds = oracle.sssp_frontier_bf(rp, col, w, 0)
    assert dist.tolist() == [0, oracle.SSSP_INF, oracle.SSSP_INF] and rounds == 1


def test_c5_against_dijkstra_and_the_triangle_inequality():
    for job, (v, deg) in enumerate([(50, 2), (300, 3), (2000, 4), (4096, 8)]):
        img = inputgen.sssp_job(job, v, deg)
        assert img[0] == v and img[2] == 0
        e = int(img[1])
        rp, col, w = img[4:4 + v + 1], img[5 + v:5 + v + e], img[5 + v + e:5 + v + 2 * e]
        assert rp[0] == 0 and rp[-1] == e and img.size == 4 + v + 1 + 2 * e and w.min() >= 1 and w.max() <= 100
        dist, rounds = oracle.sssp_frontier_bf(rp, col, w, 0)
        assert np.array_equal(dist, _dijkstra(v, rp, col, w, 0))            # an independent algorithm (binary heap)
        # invariant of any correct answer: no edge can still be relaxed, and every finite distance is attained by some edge
        src_of = np.repeat(np.arange(v), np.diff(rp))
        fin = dist[src_of] != oracle.SSSP_INF
        assert np.all(dist[col][fin].astype(np.int64) <= dist[src_of][fin].astype(np.int64) + w[fin])
        tight = np.zeros(v, bool)
        tight[col[fin][dist[col][fin].astype(np.int64) == dist[src_of][fin].astype(np.int64) + w[fin]]] = True
        reach = dist != oracle.SSSP_INF
        assert np.all(tight[reach][1:] | (np.nonzero(reach)[0][1:] == 0))   # every reached vertex but the source has a tight in-edge
        assert 1 <= rounds <= v
        # the whole-job image: [dist][rounds, 0, 0, 0]
        out = oracle.sssp_job(img).view(np.int32)
        assert np.array_equal(out[:v], dist) and out[v:].tolist() == [rounds, 0, 0, 0]
    # unreachable vertices exist in the sparse cases and stay at INF
    img = inputgen.sssp_job(0, 50, 2)
    assert (oracle.sssp_job(img).view(np.int32)[:50] == oracle.SSSP_INF).any()


# =============================================================== config 6: Sobel chain
def _brute_3x3(img, fn):
    h, w = img.shape
    out = np.zeros((h, w), np.int64)
    for y in range(h):
        for x in range(w):
            nb = [[int(img[min(max(y + dy, 0), h - 1), min(max(x + dx, 0), w - 1)]) for dx in (-1, 0, 1)] for dy in (-1, 0, 1)]
            out[y, x] = fn(nb)
    return out


def test_c6_sobel_closed_forms():
    # constant image: no edges anywhere, borders included (clamp-to-edge keeps it constant)
    assert not oracle.sobel_u8(np.full((7, 9), 200, np.uint8)).any()
    # vertical step 0 | 40 between columns 3 and 4: gx = (1 + 2 + 1) * 40 = 160 on both sides of the step, gy = 0
    img = np.zeros((6, 8), np.uint8)
    img[:, 4:] = 40
    e = oracle.sobel_u8(img)
    assert np.all(e[:, 3] == 160) and np.all(e[:, 4] == 160) and not e[:, :3].any() and not e[:, 5:].any()
    # a taller step saturates: 4 * 100 = 400 -> 255 (reading S6-2)
    img[:, 4:] = 100
    assert np.all(oracle.sobel_u8(img)[:, 3:5] == 255)
    # horizontal step: the transposed kernel gives the transposed picture
    assert np.array_equal(oracle.sobel_u8(img.T.copy()), oracle.sobel_u8(img).T)
    # single bright pixel 10 in the middle: |gx| + |gy| ring 20 / 20 / 20 on the four-neighbours' ... per tap by hand
    img = np.zeros((5, 5), np.uint8)
    img[2, 2] = 10
    want = np.array([[20, 20, 20], [20, 0, 20], [20, 20, 20]])          # corners |±10| + |±10|, edges |±20| + 0
    assert np.array_equal(oracle.sobel_u8(img)[1:4, 1:4], want)


def test_c6_stages_against_per_pixel_brute_force():
    rng_img = inputgen.sobel_frame(77, (45, 37))                            # (w, h) = (45, 37) RGB frame: blocks + noise
    n = oracle.gray_u8(rng_img)
    kx = [[-1, 0, 1], [-2, 0, 2], [-1, 0, 1]]
    sob = _brute_3x3(n, lambda nb: min(255, abs(sum(kx[i][j] * nb[i][j] for i in range(3) for j in range(3)))
                                       + abs(sum(kx[j][i] * nb[i][j] for i in range(3) for j in range(3)))))
    e = oracle.sobel_u8(n)
    assert np.array_equal(e, sob)
    m = oracle.mean3x3_u8(e)
    assert np.array_equal(m, _brute_3x3(e, lambda nb: sum(map(sum, nb)) // 9))
    t = oracle.threshold_u8(m, 64)
    assert np.array_equal(t, np.where(m >= 64, 255, 0)) and set(np.unique(t)) <= {0, 255} and 0 < (t == 255).mean() < 1
    out = oracle.blend_u8(t, n)
    assert np.array_equal(out, ((128 * t.astype(np.int64) + 128 * n.astype(np.int64)) >> 8))
    # the chain is the composition of its stages
    assert np.array_equal(oracle.sobel_chain(rng_img).reshape(n.shape), out)


def test_c6_mean_threshold_blend_special_cases():
    img = np.zeros((5, 5), np.uint8)
    img[2, 2] = 255
    m = oracle.mean3x3_u8(img)
    assert np.all(m[1:4, 1:4] == 255 // 9) and m.sum() == 9 * 28                  # impulse -> 3 x 3 patch of 28
    assert np.array_equal(oracle.mean3x3_u8(np.full((4, 6), 77, np.uint8)), np.full((4, 6), 77, np.uint8))
    v = np.arange(256, dtype=np.uint8)
    assert oracle.threshold_u8(v, 64).tolist() == [0] * 64 + [255] * 192          # >= is inclusive
    assert np.array_equal(oracle.blend_u8(v, v), v)                                # blending a picture with itself
    assert oracle.blend_u8(np.array([255], np.uint8), np.array([0], np.uint8))[0] == 127    # (128 * 255) >> 8 truncates
    # a flat frame has no edges: the mask is empty and the output is the normalised frame at half intensity
    flat = np.full((6, 7, 3), 90, np.uint8)
    assert np.all(oracle.sobel_chain(flat) == 45)
