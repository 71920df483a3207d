"""GPU parity of the HOST-buffer entry points (include/er.h "HOST-buffer forms"): same results as the
device forms, bit for bit, and the oracle's for the integer outputs."""
import numpy as np
import pytest
import torch

from oracle import er_oracle as O
from paper_2606_18967_b200 import er, inputs as I

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def test_quantize_and_gemm_host_match_device_forms_and_oracle():
    N, K, M = 384, 1152, 5
    w = I.weight_bf16(N, K, 21, device="cpu", outlier_frac=0.001).pin_memory()
    x = I.activation_bf16(M, K, 22, device="cpu").pin_memory()
    lib = er.load()
    arena = er.host_arena(max(lib.er_quantize_host_arena_bytes(N, K), lib.er_gemm_host_arena_bytes(M, N, K)), DEV)
    qw = torch.empty((N, K // 8), dtype=torch.int32, device=DEV)
    sc = torch.empty((K // 128, N), dtype=torch.bfloat16, device=DEV)
    er.quantize_pack_host(w, qw, sc, arena)
    y_host = torch.empty((M, N), dtype=torch.float32).pin_memory()
    for _ in range(2):                                   # arena reuse: counters self-reset
        er.w4a16_gemm_host(x, qw, sc, y_host, arena)
    torch.cuda.synchronize()
    qr, sr = O.quantize_pack(I.as_u16(w))
    assert np.array_equal(qw.cpu().numpy().view(np.uint32), qr) and np.array_equal(I.as_u16(sc), sr)
    y_dev = er.w4a16_gemm(x.to(DEV), qw, sc, out_dtype=torch.float32)
    assert torch.equal(y_dev.cpu(), y_host)
    y_ref = O.w4a16_gemm(I.as_u16(x), qr, sr)
    assert np.abs(y_host.numpy() - y_ref).max() <= 1e-2 * np.sqrt(np.mean(y_ref ** 2)) + 1e-3


def test_spec_verify_host_matches_device_form():
    B, gamma, V = 6, 3, 20011
    lt, ld = I.verify_logits_f32(B, gamma, V, 31, draft_noise=0.5)
    tgt, drf = torch.from_numpy(lt).pin_memory(), torch.from_numpy(ld).pin_memory()
    toks = torch.from_numpy(I.sample_draft_tokens(O.softmax64(ld), 32)).pin_memory()
    ua, us = torch.from_numpy(I.uniforms((B, gamma), 33)).pin_memory(), torch.from_numpy(I.uniforms((B,), 34)).pin_memory()
    acc_h = torch.empty((B,), dtype=torch.int32).pin_memory()
    out_h = torch.empty((B, gamma + 1), dtype=torch.int32).pin_memory()
    arena = er.host_arena(er.load().er_verify_host_arena_bytes(B, gamma, V, er.ER_F32), DEV)
    er.spec_verify_host(tgt, drf, toks, ua, us, True, 1.0, acc_h, out_h, arena)
    acc_d, out_d = er.spec_verify(tgt.to(DEV), drf.to(DEV), toks.to(DEV), ua.to(DEV), us.to(DEV), True, 1.0)
    torch.cuda.synchronize()
    assert torch.equal(acc_h, acc_d.cpu()) and torch.equal(out_h, out_d.cpu())
    acc_ref, _ = O.spec_verify(lt, ld, toks.numpy(), ua.numpy(), us.numpy(), inputs_are_logits=True)
    assert np.array_equal(acc_h.numpy(), acc_ref)


def test_host_arena_too_small_is_refused():
    lib = er.load()
    x = torch.zeros((4, 256), dtype=torch.bfloat16).pin_memory()
    y = torch.zeros((4, 128), dtype=torch.bfloat16).pin_memory()
    qw = torch.zeros((128, 32), dtype=torch.int32, device=DEV)
    sc = torch.zeros((2, 128), dtype=torch.bfloat16, device=DEV)
    small = torch.empty(1024, dtype=torch.uint8, device=DEV)
    assert lib.er_w4a16_gemm_host(x.data_ptr(), 4, 256, qw.data_ptr(), sc.data_ptr(), 128, 128, y.data_ptr(), 0,
                                  small.data_ptr(), small.numel(), None) == 5
