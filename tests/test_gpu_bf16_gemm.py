"""GPU parity: er_bf16_gemm (bf16 weights: the drafter's lm_head; the target-side linears behind T_p /
T_V of Eq. 1) vs the fp64 oracle.  Tolerance as for the W4A16 linear (north_star):
max|y_f32 - y_ref| <= 1e-2 * rms(y_ref) + 1e-3 on the fp32 output; bf16 output == bf16_rne(fp32 output) bit for bit."""
import numpy as np
import pytest
import torch

from oracle import er_oracle as O
from paper_2606_18967_b200 import er, inputs as I

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _tol(y_ref):
    return 1e-2 * float(np.sqrt(np.mean(np.square(y_ref)))) + 1e-3


def _check(x, w, exact=False, cols=None):
    y32 = er.bf16_gemm(x, w, out_dtype=torch.float32)
    y16 = er.bf16_gemm(x, w, out_dtype=torch.bfloat16)
    y32b = er.bf16_gemm(x, w, out_dtype=torch.float32)
    torch.cuda.synchronize()
    assert torch.equal(y32, y32b)                                   # deterministic
    assert np.array_equal(I.as_u16(y16), O.f32_to_bf16_rne(y32.cpu().numpy()))
    assert torch.isfinite(y32).all()
    if cols is None:
        y_ref = O.bf16_gemm(I.as_u16(x), I.as_u16(w))
        got = y32.cpu().numpy().astype(np.float64)
    else:
        ct = torch.from_numpy(cols).to(DEV)
        y_ref = O.bf16_gemm(I.as_u16(x), I.as_u16(w[ct].contiguous()))
        got = y32[:, ct].cpu().numpy().astype(np.float64)
    if exact:
        assert np.array_equal(got, y_ref)
    else:
        err = np.abs(got - y_ref).max()
        assert err <= _tol(y_ref), f"max|d|={err} tol={_tol(y_ref)}"
    return y32


@pytest.mark.parametrize("M", [1, 2, 7, 16, 17, 32, 64, 65, 128, 129, 256, 300])
def test_m_sweep(M):
    N, K = 512, 1152
    w = I.weight_bf16(N, K, I.seed_of("bf16", "w"), device=DEV)
    x = I.activation_bf16(M, K, I.seed_of("bf16", "x", M), device=DEV)
    _check(x, w)


@pytest.mark.parametrize("M", [1, 16, 256])
def test_integer_probe_bit_exact(M):
    N, K = 384, 3584
    rng = np.random.default_rng(M)
    x = torch.from_numpy(rng.integers(-2, 3, size=(M, K)).astype(np.float32)).to(DEV).to(torch.bfloat16)
    w = torch.from_numpy(rng.integers(-8, 8, size=(N, K)).astype(np.float32)).to(DEV).to(torch.bfloat16)
    _check(x, w, exact=True)


def test_one_hot_reads_out_the_weight_matrix():
    N, K = 256, 512
    w = I.weight_bf16(N, K, 3, device=DEV)
    for k0 in range(0, K, 256):
        x = torch.zeros((256, K), dtype=torch.bfloat16, device=DEV)
        x[torch.arange(256), k0 + torch.arange(256)] = 1.0
        y = er.bf16_gemm(x, w, out_dtype=torch.float32)
        assert torch.equal(y, w[:, k0:k0 + 256].float().t())


def test_rows_beyond_m_untouched_and_strided_operands():
    N, K, M = 256, 640, 5
    wbig = I.weight_bf16(N, K + 64, 1, device=DEV)
    xbig = I.activation_bf16(M, K + 8, 2, device=DEV)
    w, x = wbig[:, :K], xbig[:, :K]                       # row strides K + 64 / K + 8
    y = torch.full((8, N + 16), 7.0, dtype=torch.float32, device=DEV)
    er.bf16_gemm(x, w, y=y[:M, :N])
    torch.cuda.synchronize()
    assert torch.all(y[M:] == 7.0) and torch.all(y[:, N:] == 7.0)
    ref = O.bf16_gemm(I.as_u16(x.contiguous()), I.as_u16(w.contiguous()))
    assert np.abs(y[:M, :N].cpu().numpy() - ref).max() <= _tol(ref)


@pytest.mark.parametrize("M", [1, 16, 64, 256])
def test_lm_head_full_size_sampled_columns(M):
    # config 2's lm_head [152064 x 3584] in the launch configuration bench.py times; the oracle on 512 sampled columns
    N, K = 152064, 3584
    w = I.weight_bf16(N, K, I.seed_of("cfg2", "lm_head"), device=DEV)
    x = I.activation_bf16(M, K, I.seed_of("cfg2", "lm_head", "x", M), device=DEV)
    rng = np.random.default_rng(M)
    tiles = np.sort(rng.choice(N // 128, size=4, replace=False))
    cols = np.concatenate([np.arange(t * 128, (t + 1) * 128) for t in tiles])
    y = _check(x, w, cols=cols)
    # every column against torch's own bf16 matmul (a library routine; fp32 accumulation in a different order)
    ref = (x.float() @ w.float().t())
    rms = float(ref.pow(2).mean().sqrt())
    assert float((y - ref).abs().max()) <= 1e-3 * rms + 1e-4


def test_target_side_linears_at_verify_batch():
    # f1: the target model's linears at M = B * (gamma + 1) rows (T_V) and at M = B (T_p), 7B shapes, B = 16, gamma = 4
    for name, N, K in (("qkv", 4608, 3584), ("down", 3584, 18944)):
        w = I.weight_bf16(N, K, I.seed_of("f1", name), device=DEV)
        for M in (16, 80):
            x = I.activation_bf16(M, K, I.seed_of("f1", name, M), device=DEV)
            cols = np.arange(256) + 128 * (M % 7)
            _check(x, w, cols=cols)


def test_argument_validation():
    lib = er.load()
    w = torch.zeros((128, 128), dtype=torch.bfloat16, device=DEV)
    x = torch.zeros((1, 128), dtype=torch.bfloat16, device=DEV)
    y = torch.zeros((1, 128), dtype=torch.float32, device=DEV)
    ws = torch.zeros(lib.er_bf16_gemm_workspace_bytes(1, 128, 128), dtype=torch.uint8, device=DEV)
    s = torch.cuda.current_stream().cuda_stream
    call = lambda **k: lib.er_bf16_gemm(k.get("x", x.data_ptr()), k.get("M", 1), k.get("K", 128), 128, w.data_ptr(),
                                        k.get("N", 128), 128, y.data_ptr(), 128, k.get("dt", 1), ws.data_ptr(),
                                        k.get("wsb", ws.numel()), s)
    assert call() == 0
    assert call(x=None) == 1 and call(N=100) == 2 and call(K=100) == 2 and call(M=0) == 2
    assert call(dt=3) == 4 and call(wsb=16) == 5
    assert lib.er_bf16_gemm_workspace_bytes(1, 100, 128) == 0
