"""Seeded synthetic input generators shared by the oracle tests, the GPU parity
tests and bench.py.

This module holds NONE of the method's arithmetic (no quantizer, no dequant, no
softmax, no sampler): it only draws random tensors with the shapes and value
structure of the paper's workloads (BASELINE.json
configs 0-4) and hands the SAME bytes to both sides.  bf16 tensors are returned
as torch.bfloat16 (device or host); `as_u16` gives the raw 16-bit patterns as a
numpy uint16 array, which is what the numpy oracle consumes.

The paper measured on Qwen2.5 / Llama3.1 weights and SimpleRL / DAPO-Math
rollouts; none of that is needed here: these tensors take
only the shapes and value distributions and stand in for them.
"""
from __future__ import annotations

import zlib
from dataclasses import dataclass

import numpy as np
import torch

# ---- model shapes (BASELINE.json configs 1-4) ------------------------------

@dataclass(frozen=True)
class ModelShape:
    name: str
    hidden: int
    qkv_out: int
    ffn: int
    layers: int
    vocab: int

    def linears(self):
        """(name, N, K) of the four quantized linears of one decoder layer:
        W[N][K] row-major like torch nn.Linear.weight (FFN + QKVO)."""
        h, f = self.hidden, self.ffn
        return [("qkv", self.qkv_out, h), ("o", h, h), ("gate_up", 2 * f, h), ("down", h, f)]


SHAPE_7B = ModelShape("7b", 3584, 4608, 18944, 28, 152064)
SHAPE_32B = ModelShape("32b", 5120, 7168, 27648, 64, 152064)
M_SWEEP = (1, 2, 4, 8, 16, 32, 64, 128, 256)


def seed_of(*parts) -> int:
    """Stable 31-bit seed from a tuple of names / ints (config, layer, tensor)."""
    return zlib.crc32("/".join(str(p) for p in parts).encode()) & 0x7FFFFFFF


def _gen(device, seed):
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return g


def as_u16(t: torch.Tensor) -> np.ndarray:
    """Raw bit patterns of a bf16 tensor as numpy uint16 (host copy)."""
    assert t.dtype == torch.bfloat16
    return t.detach().contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def from_u16(a: np.ndarray, device="cpu") -> torch.Tensor:
    return torch.from_numpy(a.view(np.int16).copy()).view(torch.bfloat16).to(device)


# ---- weights / activations ----------------------------------------------------

def weight_bf16(N, K, seed, device="cpu", std=0.02, outlier_frac=0.0, outlier_mul=20.0):
    """bf16 W[N][K] ~ N(0, std); optionally a fraction of elements multiplied by
    `outlier_mul` (config 3: 0.1 % outliers at 20x)."""
    g = _gen(device, seed)
    w = torch.empty((N, K), dtype=torch.float32, device=device).normal_(0.0, std, generator=g)
    if outlier_frac > 0.0:
        mask = torch.empty((N, K), dtype=torch.float32, device=device).uniform_(0, 1, generator=g) < outlier_frac
        w = torch.where(mask, w * outlier_mul, w)
    return w.to(torch.bfloat16)


def activation_bf16(M, K, seed, device="cpu"):
    """bf16 X[M][K] ~ N(0, 1)."""
    g = _gen(device, seed)
    return torch.empty((M, K), dtype=torch.float32, device=device).normal_(0.0, 1.0, generator=g).to(torch.bfloat16)


def random_codes(N, K, seed):
    """int8 codes uniform in [-8, 7] (raw-nibble GEMM tests, includes -8)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    return rng.integers(-8, 8, size=(N, K), dtype=np.int8)


def counting_codes(N, K):
    """q[n][k] = ((131 n + 7 k) mod 15) - 7 : catches any layout permutation."""
    n = np.arange(N, dtype=np.int64)[:, None]
    k = np.arange(K, dtype=np.int64)[None, :]
    return (((131 * n + 7 * k) % 15) - 7).astype(np.int8)


# ---- speculative-verify inputs -------------------------------------------------

def uniforms(shape, seed):
    """fp32 uniforms in [0, 1) (numpy PCG64; 24-bit mantissa draws)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    return rng.random(size=shape, dtype=np.float32)


def verify_logits_f32(B, gamma, V, seed, std=2.0, draft_noise=None):
    """Independent N(0, std^2) logits for target [B, gamma+1, V] and draft
    [B, gamma, V] (config 0), or draft = target + N(0, draft_noise^2) (config 4).
    Returned as float32 numpy arrays; callers cast / softmax as the config says."""
    rng = np.random.Generator(np.random.PCG64(seed))
    tgt = rng.standard_normal(size=(B, gamma + 1, V), dtype=np.float32) * np.float32(std)
    if draft_noise is None:
        drf = rng.standard_normal(size=(B, gamma, V), dtype=np.float32) * np.float32(std)
    else:
        drf = tgt[:, :gamma, :] + rng.standard_normal(size=(B, gamma, V), dtype=np.float32) * np.float32(draft_noise)
    return tgt, drf


def sample_draft_tokens(q_probs: np.ndarray, seed) -> np.ndarray:
    """x_i ~ q_i by inverse CDF on host so that E[accept] = sum min(p, q) holds
    (the drafter samples its own tokens).  q_probs: [B, gamma, V]
    non-negative rows (need not be normalised exactly)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    B, G, V = q_probs.shape
    out = np.empty((B, G), dtype=np.int32)
    for b in range(B):
        for i in range(G):
            c = np.cumsum(q_probs[b, i].astype(np.float64))
            r = rng.random() * c[-1]
            out[b, i] = min(int(np.searchsorted(c, r, side="right")), V - 1)
    return out


# ---- device-side generators for the full-size workloads (bench.py; too large for the numpy path) -----

def verify_logits_bf16_device(B, gamma, V, seed, device, std=2.0, draft_noise=0.5):
    """Config-4 verify inputs generated on `device`: target bf16 [B, gamma+1, V] = bf16(N(0, std^2)),
    draft bf16 [B, gamma, V] = bf16(target_fp32 + N(0, draft_noise^2)) on the first gamma positions."""
    g = _gen(device, seed)
    tgt32 = torch.empty((B, gamma + 1, V), dtype=torch.float32, device=device).normal_(0.0, std, generator=g)
    noise = torch.empty((B, gamma, V), dtype=torch.float32, device=device).normal_(0.0, draft_noise, generator=g)
    drf = (tgt32[:, :gamma, :] + noise).to(torch.bfloat16)
    return tgt32.to(torch.bfloat16), drf


def sample_draft_tokens_gumbel(draft_logits: torch.Tensor, seed, temperature=1.0) -> torch.Tensor:
    """x_i ~ softmax(draft_logits_i / T) by the Gumbel-max trick (argmax of logit/T + Gumbel noise): an exact
    sampler that needs no normalisation, so no part of the method's arithmetic lives here.  int32 [B, gamma]."""
    g = _gen(draft_logits.device, seed)
    u = torch.empty(draft_logits.shape, dtype=torch.float32, device=draft_logits.device).uniform_(1e-20, 1.0, generator=g)
    gumbel = -torch.log(-torch.log(u))
    return torch.argmax(draft_logits.float() / temperature + gumbel, dim=-1).to(torch.int32)


def uniforms_device(shape, seed, device):
    """fp32 uniforms in [0, 1) on `device`."""
    g = _gen(device, seed)
    return torch.empty(shape, dtype=torch.float32, device=device).uniform_(0.0, 1.0, generator=g).clamp_(max=1.0 - 2.0 ** -24)
