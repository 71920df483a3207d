"""Pins for the oracle's fp64 dequant-matmul (G1-G6).  CPU only."""
from fractions import Fraction

import numpy as np

from oracle import er_oracle as O
from paper_2606_18967_b200 import inputs as I


def _bf16_fraction(u):
    u = int(u)
    sign = -1 if (u >> 15) & 1 else 1
    e = (u >> 7) & 0xFF
    m = u & 0x7F
    if e == 0:
        return sign * Fraction(m, 1 << 7) * Fraction(1, 1 << 126)
    return sign * (1 + Fraction(m, 1 << 7)) * (Fraction(2) ** (e - 127))


def test_one_hot_reads_out_dequantized_matrix():
    # x[m] = e_k  ->  y[m][n] = q[n][k] * s[k//128][n] exactly
    N, K = 128, 256
    codes = I.random_codes(N, K, seed=2)
    qw = O.pack_codes(codes)
    rng = np.random.default_rng(0)
    scales = O.f32_to_bf16_rne(rng.uniform(0.001, 0.01, size=(K // 128, N)).astype(np.float32))
    x = np.zeros((K, K), dtype=np.uint16)
    x[np.arange(K), np.arange(K)] = 0x3F80
    y = O.w4a16_gemm(x, qw, scales)                      # [K][N]
    s = O.bf16_to_f32(scales).astype(np.float64)
    for k in range(K):
        assert np.array_equal(y[k], codes[:, k].astype(np.float64) * s[k // 128])


def test_integer_probe_is_exact():
    # s = 1, X in {-1,0,1,2}, raw codes in [-8,7]: the result is an exact integer
    N, K, M = 128, 1024, 5
    codes = I.random_codes(N, K, seed=4)
    rng = np.random.default_rng(7)
    xi = rng.integers(-1, 3, size=(M, K))
    x = O.f32_to_bf16_rne(xi.astype(np.float32))
    scales = np.full((K // 128, N), 0x3F80, dtype=np.uint16)
    y = O.w4a16_gemm(x, O.pack_codes(codes), scales)
    assert np.array_equal(y, (xi.astype(np.int64) @ codes.astype(np.int64).T).astype(np.float64))


def test_against_exact_rational_brute_force():
    # tiny shape, pure-Python Fractions: transposed operands, wrong group index or dropped scale all fail here
    N, K, M = 128, 256, 2
    w = I.as_u16(I.weight_bf16(N, K, seed=11))
    x = I.as_u16(I.activation_bf16(M, K, seed=12))
    qw, scales = O.quantize_pack(w)
    codes = O.unpack_codes(qw)
    y = O.w4a16_gemm(x, qw, scales)
    for m in range(M):
        for n in range(N):
            acc = Fraction(0)
            for k in range(K):
                acc += _bf16_fraction(x[m, k]) * int(codes[n, k]) * _bf16_fraction(scales[k // 128, n])
            assert abs(float(acc) - y[m, n]) <= 1e-12 * max(1.0, abs(float(acc)))


def test_k_split_invariance_and_linearity():
    N, K, M = 128, 1024, 4
    w = I.as_u16(I.weight_bf16(N, K, seed=21))
    x = I.as_u16(I.activation_bf16(M, K, seed=22))
    qw, scales = O.quantize_pack(w)
    y = O.w4a16_gemm(x, qw, scales)
    acc = np.zeros_like(y)
    for g in range(K // 128):
        qw_g = O.pack_codes(O.unpack_codes(qw)[:, g * 128:(g + 1) * 128])      # the packed form of one k-group
        acc += O.w4a16_gemm(x[:, g * 128:(g + 1) * 128], qw_g, scales[g:g + 1])
    assert np.allclose(acc, y, rtol=1e-12, atol=1e-14)
    # linearity with bf16-exact operands: X and 2X
    x2 = O.f32_to_bf16_rne(O.bf16_to_f32(x) * np.float32(2))
    assert np.array_equal(O.w4a16_gemm(x2, qw, scales), 2 * y)


def test_quantized_matmul_close_to_unquantized():
    # the dequantized weight approximates W: relative Frobenius error of RTN-4bit g128 on N(0, .02) is ~ 9 %
    N, K = 128, 1024
    w = I.as_u16(I.weight_bf16(N, K, seed=31))
    qw, scales = O.quantize_pack(w)
    wd = O.dequantize(qw, scales)
    wf = O.bf16_to_f32(w).astype(np.float64)
    rel = np.linalg.norm(wd - wf) / np.linalg.norm(wf)
    assert 0.05 < rel < 0.15


def test_bf16_output_rounding_vs_tolerance_finding():
    # DESIGN.md G3: the north_star tolerance is judged on the fp32 output; bf16 rounding of y alone uses most of it.
    N, K, M = 256, 2048, 4
    w = I.as_u16(I.weight_bf16(N, K, seed=0))
    x = I.as_u16(I.activation_bf16(M, K, seed=1))
    qw, scales = O.quantize_pack(w)
    y = O.w4a16_gemm(x, qw, scales)
    tol = 1e-2 * np.sqrt(np.mean(y ** 2)) + 1e-3
    y32 = y.astype(np.float32)
    assert np.max(np.abs(y32.astype(np.float64) - y)) < 1e-3 * tol


# ---- bf16_gemm (lm_head / target-side linears) ----

def test_bf16_gemm_matches_exact_rational_arithmetic():
    # pure-Python Fractions on a tiny shape: a transposed operand, a dropped k or a wrong widening fails this
    from fractions import Fraction
    rng = np.random.default_rng(5)
    M, N, K = 3, 4, 7
    x = O.f32_to_bf16_rne(rng.standard_normal((M, K)).astype(np.float32))
    w = O.f32_to_bf16_rne((rng.standard_normal((N, K)) * 0.02).astype(np.float32))
    xf, wf = O.bf16_to_f32(x), O.bf16_to_f32(w)
    y = O.bf16_gemm(x, w)
    assert y.shape == (M, N)
    for m in range(M):
        for n in range(N):
            exact = sum(Fraction(float(xf[m, k])) * Fraction(float(wf[n, k])) for k in range(K))
            assert abs(Fraction(float(y[m, n])) - exact) <= abs(exact) * Fraction(1, 10 ** 12) + Fraction(1, 10 ** 300)


def test_bf16_gemm_integers_and_one_hot():
    rng = np.random.default_rng(6)
    M, N, K = 5, 6, 256
    xi = rng.integers(-3, 4, size=(M, K)).astype(np.float32)
    wi = rng.integers(-8, 8, size=(N, K)).astype(np.float32)
    y = O.bf16_gemm(O.f32_to_bf16_rne(xi), O.f32_to_bf16_rne(wi))
    assert np.array_equal(y, (xi.astype(np.int64) @ wi.astype(np.int64).T).astype(np.float64))
    # one-hot rows read the weight matrix out, transposed
    eye = np.zeros((K, K), np.float32)
    eye[np.arange(K), np.arange(K)] = 1
    w = O.f32_to_bf16_rne(rng.standard_normal((N, K)).astype(np.float32))
    assert np.array_equal(O.bf16_gemm(O.f32_to_bf16_rne(eye), w), O.bf16_to_f32(w).astype(np.float64).T)
