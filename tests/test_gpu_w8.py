"""GPU parity of the W8A16 drafter (Table 4 "RTN W8") through the C ABI:
er_quantize_pack8 bit for bit against the oracle (packed planes and scales), er_w8a16_gemm within the W4 linear's
tolerance max|y_f32 - y_ref| <= 1e-2 * rms(y_ref) + 1e-3 on the fp32 output (exact on integer probes), bf16 output ==
bf16_rne(fp32 output), deterministic."""
import numpy as np
import pytest
import torch

from oracle import er_oracle as O
from paper_2606_18967_b200 import er, inputs as I

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _u32(t):
    return t.cpu().numpy().view(np.uint32)


@pytest.mark.parametrize("N,K", [(128, 128), (256, 2048), (3584, 3584), (512, 18944)])
def test_quantize_pack8_bit_exact(N, K):
    w = I.weight_bf16(N, K, I.seed_of("w8", N, K), device=DEV, outlier_frac=0.001)
    if N == 256:
        w[3, :128] = 0                               # an all-zero group: scale +0, codes 0
        w[5, 128:256] = 1e-39                        # denormal maximum
    qw, sc = er.quantize_pack8(w)
    torch.cuda.synchronize()
    qr, sr = O.quantize_pack8(I.as_u16(w))
    assert np.array_equal(I.as_u16(sc), sr)
    assert np.array_equal(_u32(qw), qr)
    # the planes through the library's own unpacker: (a - 8, b - 8)
    codes = torch.empty((N, 2 * K), dtype=torch.int8, device=DEV)
    er._check(er.load().er_unpack_codes(qw.data_ptr(), N, 2 * K, codes.data_ptr(), None), "unpack")
    torch.cuda.synchronize()
    p = codes.cpu().numpy().astype(np.int32).reshape(N, K // 128, 2, 128) + 8
    assert np.array_equal((16 * p[:, :, 0] + p[:, :, 1] - 128).reshape(N, K), O.unpack_codes8(qr))


def _check_gemm(x, qw, sc, exact=False, cols=None):
    y32 = er.w8a16_gemm(x, qw, sc, out_dtype=torch.float32)
    y16 = er.w8a16_gemm(x, qw, sc, out_dtype=torch.bfloat16)
    y32b = er.w8a16_gemm(x, qw, sc, out_dtype=torch.float32)
    torch.cuda.synchronize()
    assert torch.equal(y32, y32b)
    assert np.array_equal(I.as_u16(y16), O.f32_to_bf16_rne(y32.cpu().numpy()))
    qh, sh = _u32(qw), I.as_u16(sc)
    if cols is not None:                              # whole 128-row tiles only: the oracle on a slice of N
        rows = np.asarray(cols)
        K2 = qh.shape[1] * 8
        codes = O.unpack_codes8(qh)[rows]
        s = O.bf16_to_f32(sh[1::2][:, rows]).astype(np.float64)
        ref = O.bf16_to_f32(I.as_u16(x)).astype(np.float64) @ (codes * np.repeat(s.T, 128, axis=1)).T
        got = y32.cpu().numpy()[:, rows]
    else:
        ref = O.w8a16_gemm(I.as_u16(x), qh, sh)
        got = y32.cpu().numpy()
    if exact:
        assert np.array_equal(got.astype(np.float64), ref)
    else:
        tol = 1e-2 * float(np.sqrt(np.mean(ref ** 2))) + 1e-3
        assert float(np.abs(got - ref).max()) <= tol
    return y32


@pytest.mark.parametrize("M", [1, 3, 8, 16, 17, 32, 33, 64, 65, 130, 256])
def test_gemm_every_batch_size(M):
    N, K = 512, 1024
    w = I.weight_bf16(N, K, I.seed_of("w8g", "w"), device=DEV)
    x = I.activation_bf16(M, K, I.seed_of("w8g", "x", M), device=DEV)
    qw, sc = er.quantize_pack8(w)
    _check_gemm(x, qw, sc)


@pytest.mark.parametrize("K", [3584, 18944])
@pytest.mark.parametrize("M", [1, 16, 64, 130, 256])
def test_integer_probe_bit_exact(M, K):
    # power-of-two scales, X in {-1, 0, 1, 2}, codes over the whole int8 range: every partial sum is an exact integer
    N = 256
    rng = np.random.default_rng(K + M)
    q = rng.integers(-127, 128, size=(N, K)).astype(np.int16)
    q[0, :4] = [-127, 127, 0, -1]
    su = np.full((K // 128, N), 0x3B80, dtype=np.uint16)          # 2^-8
    su[1::2] = 0x3C00                                             # alternate groups 2^-7
    qw2, s2 = O.pack_codes8(q, su)
    qw = torch.from_numpy(qw2.view(np.int32)).to(DEV)
    sc = torch.from_numpy(s2.view(np.int16)).to(DEV).view(torch.bfloat16)
    x = torch.from_numpy(rng.integers(-1, 3, size=(M, K)).astype(np.float32)).to(DEV).to(torch.bfloat16)
    _check_gemm(x, qw, sc, exact=True)


def test_one_hot_reads_out_dequantised_matrix():
    N, K = 256, 256
    rng = np.random.default_rng(7)
    q = rng.integers(-127, 128, size=(N, K)).astype(np.int16)
    su = O.f32_to_bf16_rne((rng.random((K // 128, N)) * 0.02 + 0.001).astype(np.float32))
    qw2, s2 = O.pack_codes8(q, su)
    qw = torch.from_numpy(qw2.view(np.int32)).to(DEV)
    sc = torch.from_numpy(s2.view(np.int16)).to(DEV).view(torch.bfloat16)
    wd = q.astype(np.float64) * np.repeat(O.bf16_to_f32(su).astype(np.float64).T, 128, axis=1)     # exact products
    for k0 in range(0, K, 64):
        x = torch.zeros((64, K), dtype=torch.bfloat16, device=DEV)
        x[torch.arange(64), k0 + torch.arange(64)] = 1.0
        y = er.w8a16_gemm(x, qw, sc, out_dtype=torch.float32).cpu().numpy().astype(np.float64)
        # q * s = (16 s)(a - 8) + s b with fp32 roundings of the two products' sum: 15-bit significands, exact in fp32
        assert np.array_equal(y, wd[:, k0:k0 + 64].T)


@pytest.mark.parametrize("name,N,K", [("qkv", 4608, 3584), ("down", 3584, 18944)])
@pytest.mark.parametrize("M", [1, 16, 64])
def test_7b_shapes_sampled_tiles(name, N, K, M):
    w = I.weight_bf16(N, K, I.seed_of("w8", name), device=DEV, outlier_frac=0.001)
    x = I.activation_bf16(M, K, I.seed_of("w8", name, M), device=DEV)
    qw, sc = er.quantize_pack8(w)
    tiles = np.sort(np.random.default_rng(M).choice(N // 128, size=2, replace=False))
    cols = np.concatenate([np.arange(t * 128, (t + 1) * 128) for t in tiles])
    y8 = _check_gemm(x, qw, sc, cols=cols)
    # Table 4's premise on this data: the W8 drafter's outputs are closer to the bf16 linear than the W4 drafter's
    y4 = er.w4a16_gemm(x, *er.quantize_pack(w), out_dtype=torch.float32)
    ref = x.float() @ w.float().t()
    assert float((y8 - ref).abs().mean()) < 0.2 * float((y4 - ref).abs().mean())


def test_refresh_then_gemm_back_to_back():
    # no host synchronisation between the W8 refresh and the GEMM that reads its output (stream order only)
    N, K, M = 1024, 2048, 4
    w = I.weight_bf16(N, K, 5, device=DEV)
    x = I.activation_bf16(M, K, 6, device=DEV)
    qw = torch.zeros((N, 2 * K // 8), dtype=torch.int32, device=DEV)
    sc = torch.zeros((2 * K // 128, N), dtype=torch.bfloat16, device=DEV)
    ws = torch.zeros(er.load().er_w8_gemm_workspace_bytes(M, N, K), dtype=torch.uint8, device=DEV)
    er.quantize_pack8(w, qw, sc)
    y = er.w8a16_gemm(x, qw, sc, out_dtype=torch.float32, workspace=ws)
    torch.cuda.synchronize()
    ref = O.w8a16_gemm(I.as_u16(x), *O.quantize_pack8(I.as_u16(w)))
    assert float(np.abs(y.cpu().numpy() - ref).max()) <= 1e-2 * float(np.sqrt(np.mean(ref ** 2))) + 1e-3


def test_argument_validation():
    lib = er.load()
    z = torch.zeros(4096, dtype=torch.uint8, device=DEV)
    p = z.data_ptr()
    assert lib.er_quantize_pack8(None, 128, 128, 128, 128, p, p, None) == 1
    assert lib.er_quantize_pack8(p, 100, 128, 128, 128, p, p, None) == 2
    assert lib.er_quantize_pack8(p, 128, 128, 128, 64, p, p, None) == 2
    assert lib.er_w8a16_gemm(p, 1, 128, 128, p, p, 128, 128, p, 128, 0, p, 16, None) == 5
    assert lib.er_w8_gemm_workspace_bytes(1, 128, 128) >= er.COUNTER_BYTES
