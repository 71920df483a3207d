"""GPU parity: er_w4a16_gemm (tcgen05 path) and er_w4a16_gemm_simt vs the fp64 oracle (G1-G6).
Tolerance (BASELINE.json north_star): max|y_f32 - y_ref| <= 1e-2 * rms(y_ref) + 1e-3 per call, judged on the
fp32 output; the bf16 output is pinned exactly as bf16_rne(fp32 output)."""
import numpy as np
import pytest
import torch

from oracle import er_oracle as O
from paper_2606_18967_b200 import er, inputs as I

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _tol(y_ref):
    return 1e-2 * float(np.sqrt(np.mean(np.square(y_ref)))) + 1e-3


def _dev_weights(codes, scales_u16):
    qw = torch.from_numpy(O.pack_codes(codes).view(np.int32)).to(DEV)
    sc = I.from_u16(scales_u16, DEV)
    return qw, sc


def _random_scales(G, N, seed):
    rng = np.random.default_rng(seed)
    s = (rng.random((G, N), dtype=np.float32) * 0.01 + 0.001).astype(np.float32)
    return O.f32_to_bf16_rne(s)


def _check(x, qw, sc, simt=False, exact=False):
    y32 = er.w4a16_gemm(x, qw, sc, out_dtype=torch.float32, simt=simt)
    y16 = er.w4a16_gemm(x, qw, sc, out_dtype=torch.bfloat16, simt=simt)
    torch.cuda.synchronize()
    y_ref = O.w4a16_gemm(I.as_u16(x), qw.cpu().numpy().view(np.uint32), I.as_u16(sc))
    got = y32.cpu().numpy().astype(np.float64)
    if exact:
        assert np.array_equal(got, y_ref), f"max diff {np.abs(got - y_ref).max()}"
    else:
        err = np.abs(got - y_ref).max()
        assert err <= _tol(y_ref), f"max|d|={err} tol={_tol(y_ref)}"
    # bf16 output == RNE(fp32 output), bit for bit
    assert np.array_equal(I.as_u16(y16), O.f32_to_bf16_rne(y32.cpu().numpy()))
    return y32


@pytest.mark.parametrize("simt", [True, False])
def test_config0(simt):
    w = I.weight_bf16(2048, 2048, I.seed_of("cfg0", "w"), device=DEV)
    x = I.activation_bf16(4, 2048, I.seed_of("cfg0", "x"), device=DEV)
    qw, sc = er.quantize_pack(w)
    _check(x, qw, sc, simt=simt)


@pytest.mark.parametrize("simt,rows", [(True, 256), (False, 64), (False, 256)])
def test_one_hot_reads_out_dequantised_matrix(simt, rows):
    # x[m] = e_k: y[m][n] must equal q[n][k] * s[k//128][n] exactly, at every batch size and in both kernels (pins
    # layout, dequant, transpose, and that q * s is never rounded: the product has up to 12 significant bits)
    N, K = 256, 512
    codes = I.random_codes(N, K, 3)          # includes -8
    su = _random_scales(K // 128, N, 4)
    qw, sc = _dev_weights(codes, su)
    wd = O.dequantize(O.pack_codes(codes), su)      # [N][K] fp64, exact
    for k0 in range(0, K, rows):
        x = torch.zeros((rows, K), dtype=torch.bfloat16, device=DEV)
        x[torch.arange(rows), k0 + torch.arange(rows)] = 1.0
        y = er.w4a16_gemm(x, qw, sc, out_dtype=torch.float32, simt=simt).cpu().numpy().astype(np.float64)
        assert np.array_equal(y, wd[:, k0:k0 + rows].T)


def test_counting_pattern_layout():
    N, K = 128, 256
    codes = I.counting_codes(N, K)
    su = np.full((K // 128, N), 0x3F80, dtype=np.uint16)   # scale 1.0
    qw, sc = _dev_weights(codes, su)
    x = torch.zeros((16, K), dtype=torch.bfloat16, device=DEV)
    ks = [0, 1, 2, 7, 8, 9, 63, 64, 127, 128, 129, 191, 200, 254, 255, 77]
    for m, k in enumerate(ks):
        x[m, k] = 1.0
    y = er.w4a16_gemm(x, qw, sc, out_dtype=torch.float32).cpu().numpy()
    for m, k in enumerate(ks):
        assert np.array_equal(y[m], codes[:, k].astype(np.float32)), (m, k)


@pytest.mark.parametrize("K", [3584, 18944])
@pytest.mark.parametrize("M", [1, 16, 64])
def test_integer_probe_bit_exact(M, K):
    # s = power of two, X in {-1,0,1,2}, raw codes in [-8,7]: every partial sum is an exact integer < 2^24
    N = 256
    codes = I.random_codes(N, K, K + M)
    su = np.full((K // 128, N), 0x3F80, dtype=np.uint16)
    su[1::2] = 0x4000                        # alternate groups scaled by 2.0
    qw, sc = _dev_weights(codes, su)
    rng = np.random.default_rng(M)
    x = torch.from_numpy(rng.integers(-1, 3, size=(M, K)).astype(np.float32)).to(DEV).to(torch.bfloat16)
    _check(x, qw, sc, exact=True)


@pytest.mark.parametrize("M", [1, 2, 3, 8, 16, 17, 32, 33, 64, 65, 100, 128, 256])
def test_m_sweep_and_ragged_k(M):
    N, K = 512, 1152                         # 4.5 k-blocks of 256: ragged last block
    w = I.weight_bf16(N, K, I.seed_of("msweep", "w"), device=DEV)
    x = I.activation_bf16(M, K, I.seed_of("msweep", "x", M), device=DEV)
    qw, sc = er.quantize_pack(w)
    _check(x, qw, sc)


def test_rows_independent_and_unwritten_rows_untouched():
    N, K, M = 256, 512, 5
    w = I.weight_bf16(N, K, 1, device=DEV)
    qw, sc = er.quantize_pack(w)
    x = I.activation_bf16(M, K, 2, device=DEV)
    y = torch.full((8, N), 123.0, dtype=torch.float32, device=DEV)
    er.w4a16_gemm(x, qw, sc, y=y[:M])
    assert torch.all(y[M:] == 123.0)
    perm = torch.tensor([3, 0, 4, 1, 2], device=DEV)
    y2 = er.w4a16_gemm(x[perm].contiguous(), qw, sc, out_dtype=torch.float32)
    assert torch.equal(y2, y[:M][perm])


@pytest.mark.parametrize("splits", [1, 2, 3, 7])
def test_split_k_counts_agree_and_are_deterministic(splits):
    N, K, M = 256, 3584, 16
    codes = I.random_codes(N, K, 9)
    su = np.full((K // 128, N), 0x3F80, dtype=np.uint16)
    qw, sc = _dev_weights(codes, su)
    rng = np.random.default_rng(1)
    x = torch.from_numpy(rng.integers(-1, 3, size=(M, K)).astype(np.float32)).to(DEV).to(torch.bfloat16)
    for small in (1, 0):                                 # M <= 8 would take the warp-level-MMA kernel: both kernels
        with er.dev_library() as lib:
            assert lib.er_dev_gemm_tuning(1, splits) == 0
            assert lib.er_dev_gemm_tuning(6, small) == 0
            ws = er.gemm_workspace(M, N, K, DEV)
            for Mx in (M, 8):
                y1 = er.w4a16_gemm(x[:Mx], qw, sc, out_dtype=torch.float32, workspace=ws)
                y2 = er.w4a16_gemm(x[:Mx], qw, sc, out_dtype=torch.float32, workspace=ws)   # workspace reuse: counters self-reset
                torch.cuda.synchronize()
                ref = O.w4a16_gemm(I.as_u16(x[:Mx]), qw.cpu().numpy().view(np.uint32), su)
                assert np.array_equal(y1.cpu().numpy().astype(np.float64), ref), (small, Mx)
                assert torch.equal(y1, y2)


def _sampled_columns_check(x, qw, sc, N, K, seed, label, y=None):
    """Launches the GEMM (fp32 out) and checks the 256 output columns of two sampled 128-row tiles against the
    fp64 oracle evaluated on the same device inputs."""
    M = x.shape[0]
    if y is None:
        y = er.w4a16_gemm(x, qw, sc, out_dtype=torch.float32)
    torch.cuda.synchronize()
    rng = np.random.default_rng(seed)
    G = K // 128
    blocks = qw.view(N // 128, G * 2048)                    # ER_PACK_V2: one row of this view per 128-row tile
    tiles = np.sort(rng.choice(N // 128, size=2, replace=False))
    cols = np.concatenate([np.arange(t * 128, (t + 1) * 128) for t in tiles])
    ct = torch.from_numpy(cols).to(DEV)
    qsel = blocks[torch.from_numpy(tiles).to(DEV)].cpu().numpy().view(np.uint32).reshape(256, K // 8)
    y_ref = O.w4a16_gemm(I.as_u16(x), qsel, I.as_u16(sc[:, ct].contiguous()))
    got = y[:, ct].cpu().numpy().astype(np.float64)
    err = np.abs(got - y_ref).max()
    assert err <= _tol(y_ref), f"{label} M={M}: max|d|={err} tol={_tol(y_ref)}"
    # ALL N columns: the tensor-core kernel against the plain CUDA-core kernel (same contract, different summation
    # order), which is itself pinned to the oracle on the sampled tiles -- stream-K range boundaries fall in different
    # places in every tile, so the sample alone would not see a mistake there
    y_simt = er.w4a16_gemm(x, qw, sc, out_dtype=torch.float32, simt=True)
    torch.cuda.synchronize()
    err_s = np.abs(y_simt[:, ct].cpu().numpy().astype(np.float64) - y_ref).max()
    assert err_s <= _tol(y_ref), f"{label} M={M}: SIMT max|d|={err_s}"
    rms = float(y_simt.float().pow(2).mean().sqrt())
    gap = float((y - y_simt).abs().max())
    gap_tol = 1e-4 * rms + 1e-5
    assert gap <= gap_tol, f"{label} M={M}: tensor-core kernel vs SIMT over all columns: {gap} (rms {rms})"
    assert torch.isfinite(y).all()
    return y


@pytest.mark.parametrize("name,N,K", [("qkv", 4608, 3584), ("o", 3584, 3584), ("gate_up", 37888, 3584),
                                      ("down", 3584, 18944)])
@pytest.mark.parametrize("M", [1, 8, 16, 256])
def test_config1_full_size_sampled_columns(name, N, K, M):
    # full 7B-layer shapes in the launch configuration bench.py times
    w = I.weight_bf16(N, K, I.seed_of("cfg1", name), device=DEV)
    x = I.activation_bf16(M, K, I.seed_of("cfg1", name, "x", M), device=DEV)
    qw, sc = er.quantize_pack(w)
    _sampled_columns_check(x, qw, sc, N, K, N + M, name)


@pytest.mark.parametrize("name,N,K", [("qkv", 7168, 5120), ("o", 5120, 5120), ("gate_up", 55296, 5120),
                                      ("down", 5120, 27648)])
@pytest.mark.parametrize("M", [1, 8, 32])
def test_config4_32b_shapes_sampled_columns(name, N, K, M):
    # BASELINE.json configs[4]: the 32B-class linears at batch 1-32
    w = I.weight_bf16(N, K, I.seed_of("cfg4", name), device=DEV)
    x = I.activation_bf16(M, K, I.seed_of("cfg4", name, "x", M), device=DEV)
    qw, sc = er.quantize_pack(w)
    del w
    _sampled_columns_check(x, qw, sc, N, K, N + M, name)


def test_config2_layer_chain_teacher_forced_shrinking_batch():
    # BASELINE.json configs[2]: the linears of one 7B drafter layer chained through real data dependencies while the
    # active batch shrinks 256 -> 1; every GEMM is checked on the input the GPU actually fed it (errors do not
    # compound).  Glue: attention := first 3584 columns of QKV, SiLU(gate) * up, RMS renormalisation.
    H, FF = 3584, 18944
    shapes = {"qkv": (4608, H), "o": (H, H), "gate_up": (2 * FF, H), "down": (H, FF)}
    W = {}
    for n, (N, K) in shapes.items():
        w = I.weight_bf16(N, K, I.seed_of("cfg2", n), device=DEV)
        W[n] = er.quantize_pack(w)
        del w
    ws = er.gemm_workspace(256, 2 * FF, H, DEV)

    def renorm(t):
        t = t.float()
        return (t / t.pow(2).mean(dim=1, keepdim=True).sqrt().clamp_min(1e-6)).to(torch.bfloat16)

    for M in (256, 128, 64, 16, 4, 1):
        h = I.activation_bf16(M, H, I.seed_of("cfg2", "x", M), device=DEV)

        def lin(n, x):
            N, K = shapes[n]
            y = er.w4a16_gemm(x, W[n][0], W[n][1], out_dtype=torch.float32, workspace=ws)
            return _sampled_columns_check(x, W[n][0], W[n][1], N, K, N + M, f"chain {n}", y=y)

        qkv = lin("qkv", h)
        att = renorm(qkv[:, :H])
        o = lin("o", att)
        h2 = renorm(h.float() + o)
        gu = lin("gate_up", h2)
        act = renorm(torch.nn.functional.silu(gu[:, :FF]) * gu[:, FF:])
        d = lin("down", act)
        assert torch.isfinite(d).all()


def test_programmatic_dependent_launch_does_not_change_results():
    # er_w4a16_gemm is launched with programmatic stream serialization; back-to-back calls that depend on each other
    # (same Y / workspace, chained X) must give the same bits with it switched off
    N, K, M = 3584, 3584, 8
    w = I.weight_bf16(N, K, I.seed_of("pdl", "w"), device=DEV)
    qw, sc = er.quantize_pack(w)
    x0 = I.activation_bf16(M, K, I.seed_of("pdl", "x"), device=DEV)
    ws = er.gemm_workspace(M, N, K, DEV)
    outs = []
    with er.dev_library() as lib:
        for pdl in (1, 0):
            assert lib.er_dev_gemm_tuning(3, pdl) == 0
            x = x0
            for _ in range(4):          # y feeds the next call: a chain of dependent launches
                y = er.w4a16_gemm(x, qw, sc, out_dtype=torch.bfloat16, workspace=ws)
                x = (y.float() / y.float().pow(2).mean().sqrt()).to(torch.bfloat16)
            torch.cuda.synchronize()
            outs.append(y.clone())
    assert torch.equal(outs[0], outs[1])
    # ... and the shipped library gives those bits too
    x = x0
    for _ in range(4):
        y = er.w4a16_gemm(x, qw, sc, out_dtype=torch.bfloat16, workspace=ws)
        x = (y.float() / y.float().pow(2).mean().sqrt()).to(torch.bfloat16)
    torch.cuda.synchronize()
    assert torch.equal(y, outs[0])


def test_refresh_then_gemm_back_to_back_sees_the_new_weights():
    # er_quantize_pack immediately followed by er_w4a16_gemm on the same stream, repeatedly with DIFFERENT weights in
    # the same buffers (the per-RL-step refresh): the GEMM (programmatic dependent launch: its prologue
    # overlaps the refresh kernel's tail) must never read stale packed words
    N, K = 37888, 3584
    qw = torch.empty((N, K // 8), dtype=torch.int32, device=DEV)
    sc = torch.empty((K // 128, N), dtype=torch.bfloat16, device=DEV)
    ws = er.gemm_workspace(16, N, K, DEV)
    for M in (4, 16):
        x = I.activation_bf16(M, K, I.seed_of("b2b", "x", M), device=DEV)
        ws_ = [I.weight_bf16(N, K, I.seed_of("b2b", r), device=DEV) for r in range(3)]
        ys = []
        for r in range(3):
            er.quantize_pack(ws_[r], qw, sc)
            ys.append(er.w4a16_gemm(x, qw, sc, out_dtype=torch.float32, workspace=ws))
        torch.cuda.synchronize()
        for r in range(3):               # the same, with a device synchronisation between refresh and GEMM
            er.quantize_pack(ws_[r], qw, sc)
            torch.cuda.synchronize()
            y = er.w4a16_gemm(x, qw, sc, out_dtype=torch.float32, workspace=ws)
            torch.cuda.synchronize()
            assert torch.equal(y, ys[r]), (M, r)


@pytest.mark.parametrize("mode", ["cluster", "tile_split", "stream_k"])
def test_partition_modes_agree_with_the_oracle_and_are_deterministic(mode):
    # the same problem under the three work partitions (cluster reduction through DSMEM; k parts per tile with
    # an L2 ticket; stream-K ranges): each within tolerance of the oracle and bit-identical run to run
    N, K, M = 4608, 3584, 16
    w = I.weight_bf16(N, K, I.seed_of("modes", "w"), device=DEV)
    x = I.activation_bf16(M, K, I.seed_of("modes", "x"), device=DEV)
    qw, sc = er.quantize_pack(w)
    with er.dev_library() as lib:
        lib.er_dev_gemm_tuning(5, 1 if mode == "cluster" else 0)
        lib.er_dev_gemm_tuning(4, 0 if mode == "stream_k" else 1)
        for Mx in (M, 8, 3):          # M <= 8 without a cluster goes through the warp-level-MMA kernel
            y1 = _sampled_columns_check(x[:Mx], qw, sc, N, K, 7, mode)
            y2 = er.w4a16_gemm(x[:Mx], qw, sc, out_dtype=torch.float32)
            torch.cuda.synchronize()
            assert torch.equal(y1, y2)


@pytest.mark.parametrize("M", [1, 5, 8])
def test_both_small_batch_kernels_agree_with_the_oracle(M):
    # M <= 8 on a plan without a cluster runs the warp-level-MMA kernel (w4a16_gemm_small.cu); the development
    # library can send the same problem through the tcgen05 kernel: both against the oracle, on a shape with whole
    # tiles and partial tiles per CTA (stream-K) and on a raw-nibble matrix that contains the code -8
    for N, K in ((37888, 3584), (1024, 1152)):
        codes = I.random_codes(N, K, N + M) if N == 1024 else None
        if codes is None:
            w = I.weight_bf16(N, K, I.seed_of("small", N), device=DEV)
            qw, sc = er.quantize_pack(w)
            del w
        else:
            qw, sc = _dev_weights(codes, _random_scales(K // 128, N, 5))
        x = I.activation_bf16(M, K, I.seed_of("small", "x", M), device=DEV)
        with er.dev_library() as lib:
            for small in (1, 0):
                lib.er_dev_gemm_tuning(6, small)
                _sampled_columns_check(x, qw, sc, N, K, N + M + small, f"small_mma={small}")


@pytest.mark.parametrize("M", [1, 16, 64])
def test_heavy_tailed_activations_stay_within_tolerance(M):
    # the -136 offset of the stored nibble is folded into the contraction (fp32 accumulation of x * (136 + q) and of
    # -136 * x): activations with 100x outliers (as LLM hidden states have) must not cost accuracy
    N, K = 512, 3584
    w = I.weight_bf16(N, K, I.seed_of("tail", "w"), device=DEV)
    qw, sc = er.quantize_pack(w)
    g = torch.Generator(device="cpu").manual_seed(I.seed_of("tail", "x", M) % (2 ** 31))
    x = torch.randn(M, K, generator=g)
    mask = torch.rand(M, K, generator=g) < 0.002
    x = torch.where(mask, x * 100.0, x).to(torch.bfloat16).to(DEV)
    _check(x, qw, sc)


@pytest.mark.parametrize("M", [17, 32, 33, 64, 100, 128, 129, 256, 300])
def test_large_batch_kernel_every_m(M):
    # w4a16_gemm_large.cu (A operand = bf16_rne(q * s), one accumulator over K) forced for every M > 16 through the
    # development library: whole tiles, stream-K ranges with partial tiles (forced CTA counts), several batch chunks
    # (M = 300 > 256), ragged M; within the stated tolerance of the oracle and bit-identical run to run
    N, K = 1024, 1152
    w = I.weight_bf16(N, K, I.seed_of("large", "w"), device=DEV)
    x = I.activation_bf16(M, K, I.seed_of("large", "x", M), device=DEV)
    qw, sc = er.quantize_pack(w)
    y_ref = O.w4a16_gemm(I.as_u16(x), qw.cpu().numpy().view(np.uint32), I.as_u16(sc))
    with er.dev_library() as lib:
        assert lib.er_dev_gemm_tuning(7, 2) == 0
        for ctas in (0, 5, 37):
            assert lib.er_dev_gemm_tuning(1, ctas) == 0
            y1 = er.w4a16_gemm(x, qw, sc, out_dtype=torch.float32)
            y2 = er.w4a16_gemm(x, qw, sc, out_dtype=torch.float32)
            yb = er.w4a16_gemm(x, qw, sc, out_dtype=torch.bfloat16)
            torch.cuda.synchronize()
            err = np.abs(y1.cpu().numpy().astype(np.float64) - y_ref).max()
            assert err <= _tol(y_ref), (M, ctas, err, _tol(y_ref))
            assert torch.equal(y1, y2)
            assert np.array_equal(I.as_u16(yb), O.f32_to_bf16_rne(y1.cpu().numpy()))


def test_large_batch_kernel_exact_cases():
    # power-of-two scales: q * s is exact in bf16, so the large-batch kernel must reproduce the integer probe bit for bit
    # (pins its layout, k order, accumulate flags and split-K reduction); general scales: a one-hot X reads out
    # bf16_rne(q * s) exactly
    N, K, M = 256, 3584, 200
    codes = I.random_codes(N, K, 21)
    su = np.full((K // 128, N), 0x3F80, dtype=np.uint16)
    su[1::2] = 0x4000
    qw, sc = _dev_weights(codes, su)
    rng = np.random.default_rng(3)
    x = torch.from_numpy(rng.integers(-1, 3, size=(M, K)).astype(np.float32)).to(DEV).to(torch.bfloat16)
    ref = O.w4a16_gemm(I.as_u16(x), qw.cpu().numpy().view(np.uint32), su)
    su2 = _random_scales(K // 128, N, 22)
    qw2, sc2 = _dev_weights(codes, su2)
    wd = O.dequantize(O.pack_codes(codes), su2)                   # fp64 q * s
    wd_bf16 = O.bf16_to_f32(O.f32_to_bf16_rne(wd.astype(np.float32))).astype(np.float64)
    with er.dev_library() as lib:
        lib.er_dev_gemm_tuning(7, 2)
        for ctas in (0, 11):
            lib.er_dev_gemm_tuning(1, ctas)
            y = er.w4a16_gemm(x, qw, sc, out_dtype=torch.float32)
            assert np.array_equal(y.cpu().numpy().astype(np.float64), ref), ctas
        lib.er_dev_gemm_tuning(1, 0)
        xo = torch.zeros((256, K), dtype=torch.bfloat16, device=DEV)
        xo[torch.arange(256), 1000 + torch.arange(256)] = 1.0
        y = er.w4a16_gemm(xo, qw2, sc2, out_dtype=torch.float32).cpu().numpy().astype(np.float64)
        assert np.array_equal(y, wd_bf16[:, 1000:1256].T)


@pytest.mark.parametrize("mode", ["cluster", "stream_k"])
@pytest.mark.parametrize("M", [17, 32])
def test_partition_modes_at_m_17_to_32(mode, M):
    # 16 < M <= 32 also runs the parts of a tile as a thread-block cluster (DSMEM reduction) on the small linears
    N, K = 3584, 3584
    w = I.weight_bf16(N, K, I.seed_of("modes32", "w"), device=DEV)
    x = I.activation_bf16(M, K, I.seed_of("modes32", "x", M), device=DEV)
    qw, sc = er.quantize_pack(w)
    with er.dev_library() as lib:
        lib.er_dev_gemm_tuning(5, 1 if mode == "cluster" else 0)
        lib.er_dev_gemm_tuning(4, 0 if mode == "stream_k" else 1)
        y1 = _sampled_columns_check(x, qw, sc, N, K, 9, mode)
        y2 = er.w4a16_gemm(x, qw, sc, out_dtype=torch.float32)
        torch.cuda.synchronize()
        assert torch.equal(y1, y2)

@pytest.mark.parametrize("wide", [0, 2])
@pytest.mark.parametrize("M", [65, 130, 200, 256, 300])
def test_exact_kernels_above_64_rows_every_plan(M, wide):
    # M > 64 runs either in chunks of 64 batch rows (w4a16_gemm.cu, dev key 8 = 0) or in tiles of 128 batch rows
    # (w4a16_gemm_wide.cu, key 8 = 2: always); (chunk, weight tile) = a tile of its own: whole tiles (key 9 = 1), stream-K
    # ranges whose partial tiles go through the workspace (key 9 = 2, and forced CTA counts), the last chunk ragged;
    # integer probe: bit-exact against the oracle, i.e. no rounding of q * s at any M
    N, K = 1024, 1152
    codes = I.random_codes(N, K, 31)
    su = np.full((K // 128, N), 0x3F80, dtype=np.uint16)
    su[1::2] = 0x4000
    qw, sc = _dev_weights(codes, su)
    rng = np.random.default_rng(M)
    x = torch.from_numpy(rng.integers(-1, 3, size=(M, K)).astype(np.float32)).to(DEV).to(torch.bfloat16)
    ref = O.w4a16_gemm(I.as_u16(x), qw.cpu().numpy().view(np.uint32), su)
    su2 = _random_scales(K // 128, N, 32)
    qw2, sc2 = _dev_weights(codes, su2)
    xg = I.activation_bf16(M, K, I.seed_of("exact64", M), device=DEV)
    ref2 = O.w4a16_gemm(I.as_u16(xg), qw2.cpu().numpy().view(np.uint32), su2)
    with er.dev_library() as lib:
        assert lib.er_dev_gemm_tuning(8, wide) == 0
        for ctas, units in ((0, 1), (0, 2), (5, 0), (37, 0), (148, 0)):
            assert lib.er_dev_gemm_tuning(1, ctas) == 0 and lib.er_dev_gemm_tuning(9, units) == 0
            y = er.w4a16_gemm(x, qw, sc, out_dtype=torch.float32)
            y2 = er.w4a16_gemm(x, qw, sc, out_dtype=torch.float32)
            yb = er.w4a16_gemm(x, qw, sc, out_dtype=torch.bfloat16)
            assert np.array_equal(y.cpu().numpy().astype(np.float64), ref), (M, ctas, units)
            assert torch.equal(y, y2)
            assert np.array_equal(I.as_u16(yb), O.f32_to_bf16_rne(y.cpu().numpy()))
            yg = er.w4a16_gemm(xg, qw2, sc2, out_dtype=torch.float32).cpu().numpy().astype(np.float64)
            assert np.abs(yg - ref2).max() <= 1e-5 * np.sqrt(np.mean(ref2 ** 2)) + 1e-6, (M, ctas, units)   # fp32 summation only


@pytest.mark.parametrize("M", [65, 128, 200])
def test_above_64_rows_long_k_few_tiles_automatic_plan(M):
    # the shape class of `down` (few weight tiles, long K): the cost model picks the 128-row kernel with a TILE SPLIT (k
    # CTAs per tile, one partial tile each, ticket reduction); integer probe: bit-exact, deterministic
    N, K = 256, 18944
    codes = I.random_codes(N, K, 41)
    su = np.full((K // 128, N), 0x3F80, dtype=np.uint16)
    su[1::2] = 0x4000
    qw, sc = _dev_weights(codes, su)
    rng = np.random.default_rng(M)
    x = torch.from_numpy(rng.integers(-1, 3, size=(M, K)).astype(np.float32)).to(DEV).to(torch.bfloat16)
    ref = O.w4a16_gemm(I.as_u16(x), qw.cpu().numpy().view(np.uint32), su)
    y = er.w4a16_gemm(x, qw, sc, out_dtype=torch.float32)
    y2 = er.w4a16_gemm(x, qw, sc, out_dtype=torch.float32)
    torch.cuda.synchronize()
    assert np.array_equal(y.cpu().numpy().astype(np.float64), ref)
    assert torch.equal(y, y2)
