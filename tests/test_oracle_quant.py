"""Pins for the oracle's RTN quantizer / packer (Q1-Q12).  CPU only."""
from fractions import Fraction

import numpy as np
import pytest

from oracle import er_oracle as O
from paper_2606_18967_b200 import inputs as I


def _bf16_fraction(u):
    """Exact rational value of a finite bf16 bit pattern."""
    u = int(u)
    sign = -1 if (u >> 15) & 1 else 1
    e = (u >> 7) & 0xFF
    m = u & 0x7F
    if e == 0:
        return sign * Fraction(m, 1 << 7) * Fraction(1, 1 << 126)
    return sign * (1 + Fraction(m, 1 << 7)) * (Fraction(2) ** (e - 127))


def _rne_fraction(fr):
    """Round a Fraction to the nearest integer, ties to even."""
    fl = fr.numerator // fr.denominator
    rem = fr - fl
    if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and fl % 2 == 1):
        return fl + 1
    return fl


def test_bf16_helpers_roundtrip_all_patterns():
    u = np.arange(65536, dtype=np.uint16)
    f = O.bf16_to_f32(u)
    finite = np.isfinite(f)
    assert np.array_equal(O.f32_to_bf16_rne(f[finite]), u[finite])
    # ties-to-even on the dropped half: 1 + 2^-8 is halfway between 1 and 1 + 2^-7 -> 1 (even)
    assert O.f32_to_bf16_rne(np.float32(1.0 + 2.0 ** -8)) == 0x3F80
    # 1 + 3*2^-8 is halfway between 1+2^-7 (odd) and 1+2^-6 (even) -> up
    assert O.f32_to_bf16_rne(np.float32(1.0 + 3 * 2.0 ** -8)) == 0x3F82
    assert O.f32_to_bf16_rne(np.float32(1.0 + 2.0 ** -8 + 2.0 ** -20)) == 0x3F81


def test_pack_roundtrip_every_nibble_every_position():
    # all 16 nibble values at all 8 word positions (Q10), in every 16-byte chunk of a block row
    codes = np.zeros((128, 128), dtype=np.int8)
    for v in range(16):
        for pos in range(8):
            for chunk in range(4):
                codes[8 * v + pos, 32 * chunk + pos * 4 % 32 + pos % 4] = v - 8
    packed = O.pack_codes(codes)
    assert packed.dtype == np.uint32 and packed.shape == (128, 16)
    assert np.array_equal(O.unpack_codes(packed), codes)
    rng = np.random.default_rng(1)
    rc = rng.integers(-8, 8, size=(256, 384), dtype=np.int8)
    assert np.array_equal(O.unpack_codes(O.pack_codes(rc)), rc)
    cc = I.counting_codes(128, 256)
    assert np.array_equal(O.unpack_codes(O.pack_codes(cc)), cc)


def test_pack_layout_is_the_documented_index_function():
    # ER_PACK_V2 (Q11), written independently of the oracle's vectorised packer, element by element:
    # block (T, g) of 128 rows x 128 k starts at word (T * G + g) * 2048; inside it row r keeps its place (16 words),
    # its 16-byte chunks are XOR-permuted by (r >> 1) & 3; the word of logical k-octet j holds k = 8 j + pi[i] in
    # bits [4i, 4i+4), pi = (0,2,4,6,1,3,5,7), nibble = q + 8: (word >> 4t) & 0x000F000F is the pair (k=2t, 2t+1).
    rng = np.random.default_rng(3)
    N, K = 256, 384
    G = K // 128
    codes = rng.integers(-8, 8, size=(N, K), dtype=np.int8)
    flat = O.pack_codes(codes).reshape(-1)
    for n in (0, 1, 2, 3, 5, 6, 127, 128, 131, 255):
        for jj in range(K // 8):
            T, r, g, j = n // 128, n % 128, jj // 16, jj % 16
            idx = (T * G + g) * 2048 + r * 16 + ((j // 4) ^ ((r >> 1) & 3)) * 4 + j % 4
            wv = int(flat[idx])
            for t in range(4):
                pair = (wv >> (4 * t)) & 0x000F000F
                assert (pair & 0xFFFF) - 8 == codes[n, 8 * jj + 2 * t]
                assert (pair >> 16) - 8 == codes[n, 8 * jj + 2 * t + 1]


def test_error_bound_and_code_range_on_config_like_weights():
    w = I.as_u16(I.weight_bf16(256, 1024, seed=0, outlier_frac=0.001))
    codes, scales = O.quantize_codes(w)
    wf = O.bf16_to_f32(w).astype(np.float64)
    s = O.bf16_to_f32(scales).astype(np.float64)          # [G][N]
    s_full = np.repeat(s.T, 128, axis=1)
    err = np.abs(wf - codes.astype(np.float64) * s_full)
    assert np.all(err <= s_full / 2)                       # |w - q s| <= s/2  (north_star)
    assert codes.min() >= -7 and codes.max() <= 7          # -8 is never produced (Q7)
    # every group holds a code of magnitude 7 at its amax element
    assert np.all(np.abs(codes).reshape(256, 8, 128).max(axis=2) == 7)


def test_idempotent_special_case():
    # W = s0 * q0 with s0 a power of two and +-7 in every group -> exactly (q0, s0)
    rng = np.random.default_rng(1)
    q0 = rng.integers(-7, 8, size=(8, 512)).astype(np.float32)
    q0[:, ::128] = 7
    q0[:, 1::256] = -7
    s0 = np.float32(2.0 ** -6)
    w = O.f32_to_bf16_rne(q0 * s0)
    codes, scales = O.quantize_codes(w)
    assert np.array_equal(codes, q0.astype(np.int8))
    assert np.all(O.bf16_to_f32(scales) == s0)


def test_scale_doubling_and_sign_symmetry():
    w = I.as_u16(I.weight_bf16(32, 512, seed=5))
    c1, s1 = O.quantize_codes(w)
    w2 = O.f32_to_bf16_rne(O.bf16_to_f32(w) * np.float32(2))
    c2, s2 = O.quantize_codes(w2)
    assert np.array_equal(c1, c2)
    assert np.array_equal(O.bf16_to_f32(s2), O.bf16_to_f32(s1) * np.float32(2))
    wn = w ^ np.uint16(0x8000)
    c3, s3 = O.quantize_codes(wn)
    assert np.array_equal(c3, -c1) and np.array_equal(s3, s1)


def test_zero_group():
    w = np.zeros((2, 256), dtype=np.uint16)
    w[1, 130] = 0x3F80
    codes, scales = O.quantize_codes(w)
    assert scales[0, 0] == 0 and scales[1, 0] == 0 and scales[0, 1] == 0
    assert np.all(codes[0] == 0) and codes[1, 130] == 7 and np.count_nonzero(codes[1]) == 1


def test_brute_force_all_bf16_values_against_exact_rationals():
    # every finite bf16 w against a handful of group maxima: scale and code must equal what exact rational
    # arithmetic gives (s = RNE_bf16(amax/7) exactly; q = RNE_ties_even(w/s) exactly) -- Q4, Q6.
    amaxes = [0x3D23, 0x3CA4, 0x3F80, 0x3E99, 0x4049]       # arbitrary positive bf16 patterns
    allw = np.arange(65536, dtype=np.uint16)
    for am in amaxes:
        am_f = float(O.bf16_to_f32(np.uint16(am)))
        cand = allw[np.isfinite(O.bf16_to_f32(allw)) & (np.abs(O.bf16_to_f32(allw)) <= am_f)]
        rng = np.random.default_rng(am)
        pick = rng.choice(cand, size=127 * 24, replace=False).reshape(24, 127)
        w = np.concatenate([np.full((24, 1), am, dtype=np.uint16), pick], axis=1)
        codes, scales = O.quantize_codes(w)
        # exact scale: nearest bf16 to amax/7
        target = _bf16_fraction(am) / 7
        s_u = int(scales[0, 0])
        s_fr = _bf16_fraction(s_u)
        for nb in (s_u - 1, s_u + 1):
            assert abs(s_fr - target) <= abs(_bf16_fraction(nb) - target)
        assert np.all(scales == s_u)
        for n in range(24):
            for k in range(0, 128, 5):
                assert int(codes[n, k]) == _rne_fraction(_bf16_fraction(w[n, k]) / s_fr)


def test_workload_statistics_config3():
    # sanity of the generator, not of the quantizer: ~12 % of groups hold a 20x outlier, ~22 % of codes are 0
    w = I.as_u16(I.weight_bf16(512, 3584, seed=I.seed_of("cfg3", 0, "qkv"), outlier_frac=0.001))
    codes, _ = O.quantize_codes(w)
    assert 0.15 < np.mean(codes == 0) < 0.30


def test_table4_byte_ratio_from_layout():
    # PAPER.md Table 4 (tests/golden/table4_ratio.txt): the W4 g128 + bf16-scale layout reproduces the
    # paper's idealized drafter/target ratio from byte counts alone (within 2 %).
    sh = I.SHAPE_7B
    lin = sum(N * K for _, N, K in sh.linears()) * sh.layers
    emb = sh.vocab * sh.hidden
    rows = [l.split() for l in open(__file__.rsplit("/", 1)[0] + "/golden/table4_ratio.txt") if not l.startswith("#")]
    for bits, printed, _ in rows:
        per_w = int(bits) / 8 + 2 / 128
        ratio = (lin * per_w + 2 * emb * 2) / (lin * 2 + 2 * emb * 2)
        assert abs(ratio - float(printed)) / float(printed) < 0.02
