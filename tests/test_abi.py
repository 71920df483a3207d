"""CPU-only checks of the C-ABI boundary: the library builds/loads, exports every symbol include/er.h
declares, size queries, and every argument-validation path (validation happens before any launch, so these
need no GPU)."""
import ctypes
import os
import re

import pytest

from paper_2606_18967_b200 import er

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "er.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(er_[a-z0-9_]+)\s*\(", text)))


def test_library_loads_and_exports_every_declared_symbol():
    lib = er.load()
    names = _declared_symbols()
    assert {"er_quantize_pack", "er_w4a16_gemm", "er_spec_verify"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in er.h but not exported"
    assert lib.er_abi_version() == 1


def _exported(path):
    import subprocess
    out = subprocess.run(["nm", "-D", "--defined-only", path], check=True, capture_output=True, text=True).stdout
    return sorted({ln.split()[-1] for ln in out.splitlines() if " T " in ln and ln.split()[-1].startswith("er_")})


def test_export_list_equals_the_header_both_directions():
    # the shipped library exports exactly what include/er.h declares -- no tuning hooks, no debug entry
    # points; the development knobs (csrc/er_dev.h) exist only in liber_b200_dev.so
    from paper_2606_18967_b200 import build
    assert _exported(build.build_library()) == _declared_symbols()
    dev = set(_exported(build.build_library(dev=True)))
    assert dev - set(_declared_symbols()) == {"er_dev_gemm_tuning", "er_dev_verify_cluster"}


def test_bf16_gemm_validation():
    lib = er.load()
    buf = (ctypes.c_uint8 * 4096)()
    p = (ctypes.addressof(buf) + 15) & ~15
    big = 1 << 30
    assert lib.er_bf16_gemm(None, 1, 128, 128, p, 128, 128, p, 128, 0, p, big, None) == 1
    assert lib.er_bf16_gemm(p, 1, 128, 128, p, 100, 128, p, 128, 0, p, big, None) == 2
    assert lib.er_bf16_gemm(p, 1, 128, 128, p, 128, 64, p, 128, 0, p, big, None) == 2      # ldw < K
    assert lib.er_bf16_gemm(p, 1, 128, 128, p, 128, 128, p, 128, 7, p, big, None) == 4
    assert lib.er_bf16_gemm(p + 2, 1, 128, 128, p, 128, 128, p, 128, 0, p, big, None) == 3
    assert lib.er_bf16_gemm(p, 1, 128, 128, p, 128, 128, p, 128, 0, p, 16, None) == 5
    assert lib.er_bf16_gemm_workspace_bytes(1, 128, 128) >= er.COUNTER_BYTES


def test_status_strings():
    lib = er.load()
    assert lib.er_status_str(0) == b"ER_OK"
    for s in range(1, 8):
        assert lib.er_status_str(s).startswith(b"ER_ERR_")


def test_size_queries():
    assert er.packed_bytes(4608, 3584) == 4608 * 3584 // 2
    assert er.scales_bytes(4608, 3584) == (3584 // 128) * 4608 * 2
    assert er.packed_bytes(128, 100) == 0           # K % 128 != 0
    assert er.packed_bytes(100, 128) == 0           # N % 128 != 0 (ER_PACK_V2 blocks are 128 rows)
    assert er.scales_bytes(128, 256, 64) == 0        # only group 128
    assert er.gemm_workspace_bytes(1, 4608, 3584) >= er.COUNTER_BYTES
    assert er.gemm_workspace_bytes(1, 100, 3584) == 0   # N % 128 != 0
    # bytes/weight of the packed format: 0.5 + 2/128
    N, K = 37888, 3584
    assert (er.packed_bytes(N, K) + er.scales_bytes(N, K)) / (N * K) == 0.515625


def test_quantize_pack_validation():
    lib = er.load()
    buf = (ctypes.c_uint8 * 4096)()
    p = ctypes.addressof(buf)
    p = (p + 15) & ~15
    assert lib.er_quantize_pack(None, 128, 128, 128, 128, p, p, None) == 1
    assert lib.er_quantize_pack(p, 128, 100, 128, 128, p, p, None) == 2
    assert lib.er_quantize_pack(p, 128, 128, 128, 64, p, p, None) == 2
    assert lib.er_quantize_pack(p, 128, 128, 64, 128, p, p, None) == 2     # ldw < K
    assert lib.er_quantize_pack(p + 2, 128, 128, 128, 128, p, p, None) == 3
    assert lib.er_quantize_pack(p, 128, 128, 132, 128, p, p, None) == 3    # ldw % 8


def test_gemm_validation():
    lib = er.load()
    buf = (ctypes.c_uint8 * 4096)()
    p = (ctypes.addressof(buf) + 15) & ~15
    big = 1 << 30
    assert lib.er_w4a16_gemm(None, 1, 128, 128, p, p, 128, 128, p, 128, 0, p, big, None) == 1
    assert lib.er_w4a16_gemm(p, 0, 128, 128, p, p, 128, 128, p, 128, 0, p, big, None) == 2
    assert lib.er_w4a16_gemm(p, 1, 128, 128, p, p, 100, 128, p, 128, 0, p, big, None) == 2
    assert lib.er_w4a16_gemm(p, 1, 128, 128, p, p, 128, 128, p, 128, 5, p, big, None) == 4
    assert lib.er_w4a16_gemm(p + 4, 1, 128, 128, p, p, 128, 128, p, 128, 0, p, big, None) == 3
    assert lib.er_w4a16_gemm(p, 1, 128, 128, p, p, 128, 128, p, 128, 0, None, 0, None) == 5
    assert lib.er_w4a16_gemm(p, 1, 128, 128, p, p, 128, 128, p, 128, 0, p, 16, None) == 5
    assert lib.er_w4a16_gemm_simt(p, 1, 100, 128, p, p, 128, 128, p, 128, 0, None) == 2


def test_verify_validation():
    lib = er.load()
    buf = (ctypes.c_uint8 * 4096)()
    p = (ctypes.addressof(buf) + 15) & ~15
    f = ctypes.c_float
    assert lib.er_spec_verify(p, p, 1, 0, f(1.0), p, p, p, 1, 0, 8, p, p, None) == 2      # gamma < 1
    assert lib.er_spec_verify(p, p, 1, 0, f(1.0), p, p, p, 1, 17, 8, p, p, None) == 2     # gamma > 16
    assert lib.er_spec_verify(p, p, 0, 0, f(1.0), p, p, p, 1, 2, 8, p, p, None) == 4      # bf16 probabilities
    assert lib.er_spec_verify(p, p, 1, 1, f(0.0), p, p, p, 1, 2, 8, p, p, None) == 2      # temperature
    assert lib.er_spec_verify(None, p, 1, 0, f(1.0), p, p, p, 1, 2, 8, p, p, None) == 1
    assert lib.er_spec_verify(None, None, 1, 0, f(1.0), None, None, None, 0, 2, 8, None, None, None) == 0  # B == 0


def test_no_cpu_fallback_without_gpu():
    """On a box without a B200 the compute calls must fail loudly, never compute on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    lib = er.load()
    buf = (ctypes.c_uint8 * 65536)()
    p = (ctypes.addressof(buf) + 15) & ~15
    st = lib.er_quantize_pack(p, 128, 128, 128, 128, p + 1024, p + 2048, None)
    assert st in (6, 7)
    with pytest.raises(ValueError):
        er.quantize_pack(torch.zeros((128, 128), dtype=torch.bfloat16))
