"""GPU parity: er_quantize_pack / er_unpack_codes vs the oracle, bit-exact (Q1-Q12)."""
import numpy as np
import pytest
import torch

from oracle import er_oracle as O
from paper_2606_18967_b200 import er, inputs as I

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _check_exact(w):
    qw, sc = er.quantize_pack(w)
    torch.cuda.synchronize()
    qw_ref, sc_ref = O.quantize_pack(I.as_u16(w))
    qw_np = qw.cpu().numpy().view(np.uint32)
    sc_np = I.as_u16(sc)
    assert np.array_equal(sc_np, sc_ref), f"scale mismatches: {(sc_np != sc_ref).sum()}"
    assert np.array_equal(qw_np, qw_ref), f"packed word mismatches: {(qw_np != qw_ref).sum()}"
    return qw, sc


def test_config0_whole_matrix_bit_exact():
    w = I.weight_bf16(2048, 2048, I.seed_of("cfg0", "w"), device=DEV)
    qw, _ = _check_exact(w)
    codes = er.unpack_codes(qw).cpu().numpy()
    assert np.array_equal(codes, O.unpack_codes(qw.cpu().numpy().view(np.uint32)))
    assert codes.min() >= -7 and codes.max() == 7


@pytest.mark.parametrize("N,K", [(128, 128), (128, 384), (256, 1152), (384, 640), (128, 4096)])
def test_ragged_shapes_bit_exact(N, K):
    w = I.weight_bf16(N, K, I.seed_of("ragged", N, K), device=DEV, outlier_frac=0.001)
    _check_exact(w)


def test_outliers_and_ties_bit_exact():
    # config-3 value structure: 0.1 % outliers at 20x; ~0.24 % of quotients are exact ties
    w = I.weight_bf16(1024, 3584, I.seed_of("cfg3", "layer0", "o"), device=DEV, outlier_frac=0.001)
    _check_exact(w)


def test_strided_input_and_special_groups():
    base = I.weight_bf16(128, 1024, 7, device=DEV)
    w = base[:, :512]                       # ldw = 1024 > K = 512
    assert w.stride(0) == 1024
    qw, sc = er.quantize_pack(w)
    qr, sr = O.quantize_pack(I.as_u16(w.contiguous()))
    assert np.array_equal(qw.cpu().numpy().view(np.uint32), qr) and np.array_equal(I.as_u16(sc), sr)
    z = torch.zeros((128, 256), dtype=torch.bfloat16, device=DEV)
    z[0, :128] = 1.0                        # a group of equal values; other groups all zero (Q8)
    z[1, 130] = -3.0
    z[2, 0] = 1e-38                         # denormal-range scale
    z[2, 1] = 4e-39
    _check_exact(z)


def test_exhaustive_bf16_values_against_fixed_scales():
    # every finite bf16 value as w, against a handful of group maxima (brute force over 2^16 values)
    u = np.arange(65536, dtype=np.uint16)
    f = O.bf16_to_f32(u)
    for amax_bits in (0x3F80, 0x3C23, 0x4110, 0x3DCC, 0x3FFF):
        amax = float(O.bf16_to_f32(np.uint16(amax_bits)))
        keep = np.isfinite(f) & (np.abs(f) <= amax)
        vals = u[keep]
        pad = (-len(vals)) % (127 * 128)                     # whole 128-row blocks
        vals = np.concatenate([vals, np.zeros(pad, dtype=np.uint16)])
        rows = vals.reshape(-1, 127)
        full = np.concatenate([np.full((rows.shape[0], 1), amax_bits, dtype=np.uint16), rows], axis=1)
        w = I.from_u16(full, DEV)
        _check_exact(w)


def test_sampled_groups_of_a_7b_layer():
    # config 3: 1 % of groups of a large tensor checked against the oracle on the sampled rows only
    N, K = 4608, 3584
    w = I.weight_bf16(N, K, I.seed_of("cfg3", 5, "qkv"), device=DEV, outlier_frac=0.001)
    qw, sc = er.quantize_pack(w)
    rng = np.random.default_rng(5)
    rows = np.sort(rng.choice(N, size=N // 100, replace=False))
    codes_ref, sr = O.quantize_codes(I.as_u16(w[torch.from_numpy(rows).to(DEV)]))
    codes = er.unpack_codes(qw).cpu().numpy()
    assert np.array_equal(codes[rows], codes_ref)
    assert np.array_equal(I.as_u16(sc)[:, rows], sr)
    # and two whole 128-row blocks, packed bytes compared directly
    for T in (0, N // 128 - 1):
        qr, sr = O.quantize_pack(I.as_u16(w[T * 128:(T + 1) * 128]))
        G = K // 128
        got = qw.cpu().numpy().view(np.uint32).reshape(-1)[T * G * 2048:(T + 1) * G * 2048]
        assert np.array_equal(got, qr.reshape(-1))


def test_batched_equals_separate_calls():
    # er_quantize_pack_batched: several matrices (different shapes, one strided) in one launch, bit-identical to
    # separate calls; more matrices than fit one launch (> 8) are chained
    shapes = [(128, 128), (256, 1152), (384, 640), (128, 4096), (512, 512), (128, 256), (256, 128), (128, 1024),
              (640, 384), (128, 128)]
    items, refs = [], []
    for i, (N, K) in enumerate(shapes):
        w = I.weight_bf16(N, K + (16 if i == 2 else 0), I.seed_of("batched", i), device=DEV)[:, :K]
        q1, s1 = er.quantize_pack(w)
        q2 = torch.zeros_like(q1)
        s2 = torch.zeros_like(s1)
        items.append((w, q2, s2))
        refs.append((q1, s1))
    er.quantize_pack_batched(items)
    torch.cuda.synchronize()
    for (w, q2, s2), (q1, s1) in zip(items, refs):
        assert torch.equal(q1, q2) and torch.equal(s1.view(torch.int16), s2.view(torch.int16))


def test_every_positive_finite_bf16_value_as_group_maximum():
    # DESIGN.md Q4: the kernel computes s = bf16_rne(amax * (1/7)); the reading is IEEE division.  There are only 32 640
    # positive finite bf16 values: each one is the maximum of one group here, and the stored scale bits (and codes) must
    # equal the oracle's, which divides.  (255 row tiles of 128 rows x one group.)
    amax = np.arange(0x0001, 0x7F80, dtype=np.uint16)          # every positive finite bf16, denormals included
    assert len(amax) == 0x7F80 - 1
    n = ((len(amax) + 127) // 128) * 128
    a = np.concatenate([amax, np.full(n - len(amax), 0x3F80, dtype=np.uint16)])
    rng = np.random.default_rng(11)
    w = np.zeros((n, 128), dtype=np.uint16)
    w[:, 0] = a ^ (rng.integers(0, 2, size=n).astype(np.uint16) << 15)          # random sign
    # the rest of the group: random fractions of the maximum (same exponent range), so codes are exercised as well
    frac = rng.random((n, 127), dtype=np.float32) * 2 - 1
    rest = O.f32_to_bf16_rne((O.bf16_to_f32(a)[:, None] * frac).astype(np.float32))
    w[:, 1:] = rest
    wt = I.from_u16(w, DEV)
    qw, sc = er.quantize_pack(wt)
    torch.cuda.synchronize()
    codes_ref, sr = O.quantize_codes(w)
    assert np.array_equal(I.as_u16(sc), sr), "scale bits differ from the IEEE division for some amax"
    assert np.array_equal(er.unpack_codes(qw).cpu().numpy(), codes_ref)


def test_config3_layer0_all_four_linears_bit_exact():
    # BASELINE.json configs[3]: "fully on layer 0" -- packed words and scales of QKV, O, gate/up and down of layer 0
    # (233 M parameters, N(0, 0.02) with 0.1 % outliers at 20x) byte-compared with the oracle, in row chunks so that the
    # numpy oracle stays within a few GB
    for name, N, K in I.SHAPE_7B.linears():
        w = I.weight_bf16(N, K, I.seed_of("cfg3", 0, name), device=DEV, outlier_frac=0.001)
        qw, sc = er.quantize_pack(w)
        torch.cuda.synchronize()
        G = K // 128
        qw_np = qw.cpu().numpy().view(np.uint32).reshape(-1)
        sc_np = I.as_u16(sc)
        chunk = 2048 if K <= 4096 else 512
        for r0 in range(0, N, chunk):
            r1 = min(N, r0 + chunk)
            qr, sr = O.quantize_pack(I.as_u16(w[r0:r1]))
            assert np.array_equal(qw_np[(r0 // 128) * G * 2048:(r1 // 128) * G * 2048], qr.reshape(-1)), (name, r0)
            assert np.array_equal(sc_np[:, r0:r1], sr), (name, r0)
        del w, qw, sc


@pytest.mark.parametrize("layer", [1, 9, 18, 27])
def test_config3_other_layers_sampled_one_percent_of_groups(layer):
    # the remaining layers: a seeded 1 % of the (row, group) pairs of every linear against the oracle
    for name, N, K in I.SHAPE_7B.linears():
        w = I.weight_bf16(N, K, I.seed_of("cfg3", layer, name), device=DEV, outlier_frac=0.001)
        qw, sc = er.quantize_pack(w)
        codes = er.unpack_codes(qw)
        torch.cuda.synchronize()
        G = K // 128
        rng = np.random.default_rng(I.seed_of("cfg3", "sample", layer, name))
        pick = np.sort(rng.choice(N * G, size=max(1, N * G // 100), replace=False))
        rows, groups = pick // G, pick % G
        rt, gt = torch.from_numpy(rows).to(DEV), torch.from_numpy(groups).to(DEV)
        kk = gt[:, None] * 128 + torch.arange(128, device=DEV)[None, :]
        wg = w[rt[:, None], kk].contiguous()                       # [n_pick][128]: one group per row
        cref, sref = O.quantize_codes(I.as_u16(wg))                # scales [1][n_pick]
        assert np.array_equal(codes[rt[:, None], kk].cpu().numpy(), cref), (layer, name)
        assert np.array_equal(I.as_u16(sc[gt, rt].contiguous().view(1, -1)), sref), (layer, name)
        del w, qw, sc, codes
