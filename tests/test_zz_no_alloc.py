"""GPU test of er_w4a16_gemm_static (include/er.h): the drafter linear at M <= 16 with its scratch (tile counters, split-K
partial tiles) in the library's static device array, for callers that may not allocate.  Collected last on purpose (the
run uses -x).  Its output must equal the existing path's (er_w4a16_gemm with a caller workspace: same kernels,
deterministic, so bit for bit, which is inside the linear's tolerance of 1e-2 rms + 1e-3) on two calls in a row that
leave different contents in the shared scratch, and stay inside that tolerance against the oracle."""
import numpy as np
import pytest
import torch

from oracle import er_oracle as O
from paper_2606_18967_b200 import er, inputs as I

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def test_static_scratch_gemm_matches_the_workspace_path_twice_in_a_row():
    # (N, K, M): a tile-split plan whose partial tiles go through the scratch (tcgen05 kernel, M = 16), then the
    # warp-MMA kernel's ticket path at M = 3 on the same shape, then a cluster plan (no partials) on another shape
    cases = [(512, 18944, 16), (512, 18944, 3), (4608, 3584, 1), (512, 18944, 16)]
    weights = {}
    for N, K, M in cases:
        if (N, K) not in weights:
            w = I.weight_bf16(N, K, I.seed_of("static", N, K), device=DEV)
            weights[(N, K)] = (w, *er.quantize_pack(w))
    outs = []
    for i, (N, K, M) in enumerate(cases):        # back to back, no synchronisation in between
        _, qw, sc = weights[(N, K)]
        x = I.activation_bf16(M, K, I.seed_of("static", "x", i), device=DEV)
        y = torch.full((M, N), float("nan"), dtype=torch.float32, device=DEV)
        yb = torch.zeros((M, N), dtype=torch.bfloat16, device=DEV)
        er.w4a16_gemm_static(x, qw, sc, y)
        er.w4a16_gemm_static(x, qw, sc, yb)
        outs.append((x, y, yb))
    torch.cuda.synchronize()
    for (N, K, M), (x, y, yb) in zip(cases, outs):
        _, qw, sc = weights[(N, K)]
        ref = er.w4a16_gemm(x, qw, sc, out_dtype=torch.float32)          # the existing path, its own workspace
        refb = er.w4a16_gemm(x, qw, sc, out_dtype=torch.bfloat16)
        torch.cuda.synchronize()
        assert torch.equal(y, ref) and torch.equal(yb, refb)
        y_ref = O.w4a16_gemm(I.as_u16(x), qw.cpu().numpy().view(np.uint32), I.as_u16(sc))
        tol = 1e-2 * float(np.sqrt(np.mean(y_ref ** 2))) + 1e-3
        assert float(np.abs(y.cpu().numpy() - y_ref).max()) <= tol


def test_static_scratch_gemm_rejects_what_it_was_not_sized_for():
    lib = er.load()
    N, K = 256, 512
    w = I.weight_bf16(N, K, 1, device=DEV)
    qw, sc = er.quantize_pack(w)
    x = I.activation_bf16(17, K, 2, device=DEV)
    y = torch.zeros((17, N), dtype=torch.float32, device=DEV)
    args = lambda M: (x.data_ptr(), M, K, K, qw.data_ptr(), sc.data_ptr(), N, 128, y.data_ptr(), N, 1, None)
    assert lib.er_w4a16_gemm_static(*args(17)) == 2          # ER_ERR_SHAPE: M > ER_STATIC_GEMM_MAX_M
    assert lib.er_w4a16_gemm_static(*args(0)) == 2
    assert lib.er_w4a16_gemm_static(None, 1, K, K, qw.data_ptr(), sc.data_ptr(), N, 128, y.data_ptr(), N, 1, None) == 1
    assert lib.er_w4a16_gemm_static(*args(16)) == 0
    torch.cuda.synchronize()
    assert torch.equal(y[:16], er.w4a16_gemm(x[:16], qw, sc, out_dtype=torch.float32))
