"""paper_2606_18967_b200 -- the B200-native hot path of EfficientRollout's
self-speculative decoding: er_quantize_pack, er_w4a16_gemm, er_spec_verify.

The compute lives in the C-ABI library built from csrc/ (see include/er.h);
`paper_2606_18967_b200.er` is the thin ctypes binding.  Importing the package
does not load the library; the first call does, and fails loudly if it is
missing (there is no CPU fallback).
"""
__all__ = ["er", "inputs"]
