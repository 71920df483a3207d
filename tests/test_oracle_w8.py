"""Pins of the W8A16 oracle functions (oracle/er_oracle.py; Table 4 "RTN W8") against
exact arithmetic and against the already-pinned W4 functions -- nothing here calls the product."""
from fractions import Fraction

import numpy as np

from oracle import er_oracle as O


def _bf16(x):
    return O.f32_to_bf16_rne(np.asarray(x, dtype=np.float32))


def _frac(u16):
    return Fraction(float(O.bf16_to_f32(np.array([u16], dtype=np.uint16))[0]))


def test_error_bound_and_range_in_exact_arithmetic():
    rng = np.random.default_rng(1)
    w = _bf16(rng.standard_normal((128, 256)) * 0.02)
    w[3, :128] = 0                                       # an all-zero group
    w[5, 7] = _bf16([0.9])[0]                            # an outlier
    q, s = O.quantize_codes8(w)
    assert q.min() >= -127 and q.max() <= 127
    assert np.all(q[3, :128] == 0) and s[0, 3] == 0
    for n in (0, 3, 5, 77):
        for g in (0, 1):
            sf = _frac(s[g, n])
            for k in range(g * 128, (g + 1) * 128, 5):
                wf = _frac(w[n, k])
                if sf == 0:
                    assert wf == 0
                    continue
                err = abs(wf - int(q[n, k]) * sf)
                assert err <= sf / 2 or abs(int(q[n, k])) == 127     # |w - q s| <= s / 2 unless clamped
    # every group reaches +-127 or +-126 at its maximum (s = RNE(amax / 127) is within 2^-9 of amax / 127)
    assert np.all(np.abs(q).reshape(128, 2, 128).max(axis=2)[s.T != 0] >= 126)


def test_rounding_against_fractions_brute_force():
    # one group whose scale is fixed by a maximum of 127 * 2^-6, every other element a different bf16 value: the code
    # must be the ties-to-even rounding of the exact quotient
    vals = np.arange(0x3B00, 0x3B00 + 127, dtype=np.uint16)          # bf16 bit patterns near 2^-9 ... 2^-8
    row = np.concatenate([vals, _bf16([127 * 2.0 ** -6])]).astype(np.uint16)[None, :]
    row = np.repeat(row, 128, axis=0)
    q, s = O.quantize_codes8(row)
    sf = _frac(s[0, 0])
    assert sf == Fraction(1, 64)
    for k in range(128):
        t = _frac(row[0, k]) / sf
        fl = t.numerator // t.denominator
        r = t - fl
        want = fl + (1 if r > Fraction(1, 2) or (r == Fraction(1, 2) and fl % 2 == 1) else 0)
        assert int(q[0, k]) == min(max(want, -127), 127)


def test_scale_doubling_and_sign_symmetry():
    rng = np.random.default_rng(2)
    w = (rng.standard_normal((128, 128)) * 0.05).astype(np.float32)
    q1, s1 = O.quantize_codes8(_bf16(w))
    q2, s2 = O.quantize_codes8(_bf16(2 * w))
    q3, _ = O.quantize_codes8(_bf16(-w))
    assert np.array_equal(q1, q2) and np.array_equal(q3, -q1)
    assert np.array_equal(O.bf16_to_f32(s2), 2 * O.bf16_to_f32(s1))


def test_two_plane_storage_identity_and_round_trip():
    rng = np.random.default_rng(3)
    q = rng.integers(-127, 128, size=(256, 384)).astype(np.int16)
    q[0, :4] = [-127, 127, 0, -1]
    s = _bf16(rng.random((3, 256)) * 0.01 + 0.001)
    qw2, s2 = O.pack_codes8(q, s)
    assert qw2.shape == (256, 96) and s2.shape == (6, 256)
    planes = O.unpack_codes(qw2).astype(np.int32) + 8                 # the pinned W4 unpacker: stored nibbles
    p = planes.reshape(256, 3, 2, 128)
    assert np.array_equal(16 * p[:, :, 0] + p[:, :, 1], q.reshape(256, 3, 128).astype(np.int32) + 128)
    assert p.min() >= 0 and p.max() <= 15
    assert np.array_equal(O.unpack_codes8(qw2), q)
    assert np.array_equal(s2[1::2], s) and np.array_equal(O.bf16_to_f32(s2[0::2]), 16 * O.bf16_to_f32(s))


def test_gemm_equals_two_w4_contractions_plus_offset_term():
    # y = sum_g s_g sum_k x q, q = 16 (a - 8) + (b - 8) + 8: the pinned W4 oracle on [x, x] with scales (16 s, s), plus
    # 8 s_g sum_{k in g} x_k
    rng = np.random.default_rng(4)
    N, K, M = 128, 384, 5
    w = _bf16(rng.standard_normal((N, K)) * 0.03)
    x = _bf16(rng.standard_normal((M, K)))
    qw2, s2 = O.quantize_pack8(w)
    y = O.w8a16_gemm(x, qw2, s2)
    xf = O.bf16_to_f32(x).astype(np.float64).reshape(M, K // 128, 128)
    x2 = _bf16(np.concatenate([xf, xf], axis=2).reshape(M, 2 * K))
    y4 = O.w4a16_gemm(x2, qw2, s2)
    corr = 8.0 * np.einsum("mg,gn->mn", xf.sum(axis=2), O.bf16_to_f32(s2[1::2]).astype(np.float64))
    assert np.allclose(y, y4 + corr, rtol=0, atol=1e-12 * np.abs(y).max())


def test_gemm_fraction_brute_force_and_one_hot():
    rng = np.random.default_rng(5)
    N, K, M = 128, 128, 2
    q = rng.integers(-127, 128, size=(N, K)).astype(np.int16)
    s = _bf16(rng.random((1, N)) * 0.02 + 0.001)
    x = _bf16(rng.standard_normal((M, K)))
    qw2, s2 = O.pack_codes8(q, s)
    y = O.w8a16_gemm(x, qw2, s2)
    for m in range(M):
        for n in (0, 17, 127):
            ref = sum(_frac(x[m, k]) * int(q[n, k]) * _frac(s[0, n]) for k in range(K))
            assert abs(float(ref) - y[m, n]) <= 1e-12 * max(1.0, abs(float(ref)))
    e = np.zeros((1, K), dtype=np.float32)
    e[0, 9] = 1.0
    assert np.array_equal(O.w8a16_gemm(_bf16(e), qw2, s2)[0],
                          q[:, 9].astype(np.float64) * O.bf16_to_f32(s[0]).astype(np.float64))


def test_w8_is_closer_than_w4():
    # Table 4's premise: the W8 drafter is the more accurate one
    rng = np.random.default_rng(6)
    w = _bf16(rng.standard_normal((128, 512)) * 0.02)
    wf = O.bf16_to_f32(w).astype(np.float64)
    q8, s8 = O.quantize_codes8(w)
    d8 = q8 * np.repeat(O.bf16_to_f32(s8).astype(np.float64).T, 128, axis=1)
    d4 = O.dequantize(*O.quantize_pack(w))
    assert np.abs(wf - d8).mean() < 0.1 * np.abs(wf - d4).mean()
