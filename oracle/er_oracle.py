"""CPU ORACLE -- TEST INFRASTRUCTURE ONLY.

A plain, slow, obviously-correct numpy implementation of what the hot path of
EfficientRollout's self-speculative decoding computes.  It is independent of the
CUDA path: it shares no code, header, table or helper with
`paper_2606_18967_b200/csrc`, and nothing under the product package imports it.
Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline /
`--impl reference` legs may import this module.

What the paper fixes and what it leaves open is listed in DESIGN.md
("Readings of the paper"); each function cites the passage it follows.

Parity pins (tests/test_oracle_*.py, `-m "not gpu"`):
  quantize_pack   pinned: error bound |w - q s| <= s/2, idempotent special case,
                  scale doubling, sign symmetry, brute force over all 2^16 bf16
                  values against exact rational arithmetic, nibble round trip.
  w4a16_gemm      pinned: one-hot read-out, exact-integer probe, pure-Python
                  Fraction brute force on tiny shapes, K-split invariance.
  bf16_gemm       pinned: pure-Python Fraction brute force, exact-integer case, one-hot read-out.
  quantize_codes8 / pack_codes8 / w8a16_gemm (W8A16)  pinned: |w - q s| <= s/2 in exact
                  arithmetic, brute force over bf16 values against Fractions, plane identity 16 a + b = q + 128,
                  round trip, the sum of two W4-oracle contractions plus the 8 s sum(x) term, Fraction brute force.
  spec_verify     pinned: q = p accepts everything, one-hot / zero-probability
                  cases, exact rational enumeration showing the output
                  distribution equals p (the theorem of ref. [29] the paper
                  relies on), scipy softmax.
  token_in_widened_interval  pinned on a hand-built dyadic CDF with R != 1 (rule V10: edges at
                  0.9e-5 / 1.1e-5, zero-mass token, first token, out-of-range ids).
  block_efficiency pinned to the values the paper prints (Table 2).
No function here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np

GROUP = 128          # quantization group along K (BASELINE.json north_star; Q2)
QMAX = 7             # symmetric int4: scale = amax / 7 (BASELINE.json configs[0])
PACK_PERM = (0, 2, 4, 6, 1, 3, 5, 7)   # nibble i of a word holds logical k = 8 j + PACK_PERM[i] (Q11)


# ----------------------------------------------------------------------------
# bf16 helpers (the oracle's own; bf16 is the upper 16 bits of an IEEE fp32)
# ----------------------------------------------------------------------------

def bf16_to_f32(u16: np.ndarray) -> np.ndarray:
    """Exact widening: bf16 bit pattern (uint16) -> float32."""
    u16 = np.asarray(u16, dtype=np.uint16)
    return (u16.astype(np.uint32) << np.uint32(16)).view(np.float32)


def f32_to_bf16_rne(x: np.ndarray) -> np.ndarray:
    """float32 -> bf16 bit pattern, round-to-nearest-even on the dropped 16 bits
    (finite inputs; NaN is outside the contract, Q9)."""
    b = np.asarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    lsb = (b >> np.uint64(16)) & np.uint64(1)
    b = b + np.uint64(0x7FFF) + lsb
    return (b >> np.uint64(16)).astype(np.uint16)


# ----------------------------------------------------------------------------
# (2) drafter refresh: RTN W4, group 128 along K  ("lightweight RTN
#     quantization to the FFN and QKVO projection layers", L150 Alg.1 line 3,
#     L429 "vanilla round-to-nearest (RTN) 4-bit"; layout per DESIGN.md Q1-Q12)
# ----------------------------------------------------------------------------

def quantize_codes(w_u16: np.ndarray, group: int = GROUP):
    """bf16 W[N][K] (uint16 bit patterns) -> (codes int8 [N][K] in [-8,7],
    scales uint16 bf16 bit patterns [K/group][N]).

    Per group of `group` consecutive k of one row (Q2):
      amax = max |float(w)|                                     (Q3)
      s    = bf16_RNE( fp32(amax) / fp32(7) )   IEEE fp32 divide (Q4)
      q    = clamp( rint( fp32(w) / fp32(s) ), -8, 7 )  ties-to-even, divide by
             the ROUNDED scale, IEEE fp32 divide                 (Q5-Q7)
      s == 0  ->  all q = 0, s stored +0                         (Q8)
    """
    w_u16 = np.asarray(w_u16, dtype=np.uint16)
    N, K = w_u16.shape
    assert K % group == 0
    G = K // group
    w = bf16_to_f32(w_u16).reshape(N, G, group)
    amax = np.max(np.abs(w), axis=2)                                   # [N][G] fp32, exact
    s_u16 = f32_to_bf16_rne(amax / np.float32(QMAX))                   # fp32 IEEE division
    s = bf16_to_f32(s_u16)                                             # rounded scale, as fp32
    safe = np.where(s == 0, np.float32(1), s)
    with np.errstate(invalid="ignore"):
        ratio = (w / safe[:, :, None]).astype(np.float32)              # fp32 IEEE division
    q = np.rint(ratio)                                                 # round-half-to-even
    q = np.clip(q, -8, 7)
    q = np.where((s == 0)[:, :, None], np.float32(0), q)
    codes = q.astype(np.int8).reshape(N, K)
    s_u16 = np.where(s == 0, np.uint16(0), s_u16)
    return codes, np.ascontiguousarray(s_u16.T)                        # scales [G][N]


TILE_ROWS = 128      # rows of W per packed block (Q11, ER_PACK_V2)


def _word_slot(r: np.ndarray, j: np.ndarray) -> np.ndarray:
    """ER_PACK_V2 (Q11): position, in 32-bit words, of logical word j (0..15, 8 codes each) of row r
    (0..127) inside its 128-row x 128-k block of 128 x 16 words: the row keeps its place, its four 16-byte chunks
    are permuted by XOR with bits 1..2 of the row index."""
    chunk, within = j // 4, j % 4
    return r * 16 + (chunk ^ ((r >> 1) & 3)) * 4 + within


def pack_codes(codes: np.ndarray) -> np.ndarray:
    """int8 codes [N][K] in [-8,7] -> uint32 qweight, N*K/8 words returned as [N][K/8] (ER_PACK_V2, DESIGN.md
    Q10-Q11).  Stored nibble u = q + 8 (offset binary); a word carries the 8 codes of logical k = 8 j + PACK_PERM[i]
    in bits [4 i, 4 i + 4).  Words are stored block by block: block (T, g) = rows 128 T .. 128 T + 127, k = 128 g ..
    128 g + 127, blocks ordered T-major then g, each block 128 x 16 words laid out by _word_slot."""
    codes = np.asarray(codes, dtype=np.int8)
    N, K = codes.shape
    assert K % GROUP == 0 and N % TILE_ROWS == 0
    u = (codes.astype(np.int32) + 8).astype(np.uint32).reshape(N, K // 8, 8)
    word = np.zeros((N, K // 8), dtype=np.uint32)          # word[n][jj], jj = k // 8 (row-major, logical)
    for i in range(8):
        word |= u[:, :, PACK_PERM[i]] << np.uint32(4 * i)
    T, G = N // TILE_ROWS, K // GROUP
    out = np.zeros((T, G, TILE_ROWS * 16), dtype=np.uint32)
    r = np.arange(TILE_ROWS)[:, None]
    j = np.arange(16)[None, :]
    slot = _word_slot(r, j)                                 # [128][16]
    blocks = word.reshape(T, TILE_ROWS, G, 16).transpose(0, 2, 1, 3)   # [T][G][r][j]
    out[:, :, slot.reshape(-1)] = blocks.reshape(T, G, TILE_ROWS * 16)
    return out.reshape(N, K // 8)


def unpack_codes(qweight: np.ndarray) -> np.ndarray:
    """Inverse of pack_codes: uint32 [N][K/8] (ER_PACK_V2 storage) -> int8 codes [N][K]."""
    qweight = np.asarray(qweight, dtype=np.uint32)
    N, J = qweight.shape
    K = J * 8
    assert K % GROUP == 0 and N % TILE_ROWS == 0
    T, G = N // TILE_ROWS, K // GROUP
    r = np.arange(TILE_ROWS)[:, None]
    j = np.arange(16)[None, :]
    slot = _word_slot(r, j)
    stored = qweight.reshape(T, G, TILE_ROWS * 16)
    blocks = stored[:, :, slot.reshape(-1)].reshape(T, G, TILE_ROWS, 16)
    word = blocks.transpose(0, 2, 1, 3).reshape(N, J)       # logical word[n][k // 8]
    codes = np.empty((N, J, 8), dtype=np.int8)
    for i in range(8):
        nib = (word >> np.uint32(4 * i)) & np.uint32(0xF)
        codes[:, :, PACK_PERM[i]] = nib.astype(np.int32) - 8
    return codes.reshape(N, K)


def quantize_pack(w_u16: np.ndarray, group: int = GROUP):
    """The refresh call: bf16 W[N][K] -> (qweight uint32 [N][K/8], scales bf16 bits [K/group][N])."""
    codes, scales = quantize_codes(w_u16, group)
    return pack_codes(codes), scales


# ----------------------------------------------------------------------------
# (1) drafter linear: y = X . dequant(Wq)^T  (BASELINE.json north_star; PAPER.md:L99-L101,
#     L175 "Marlin weight-only quantization kernel", L467 "on-the-fly dequantization")
# ----------------------------------------------------------------------------

def dequantize(qweight: np.ndarray, scales_u16: np.ndarray, group: int = GROUP) -> np.ndarray:
    """fp64 W_d[N][K] = q[n][k] * float(s[k // group][n]); exact (4-bit x 8-bit significand)."""
    codes = unpack_codes(qweight).astype(np.float64)
    s = bf16_to_f32(scales_u16).astype(np.float64)                     # [G][N]
    return codes * np.repeat(s.T, group, axis=1)


def w4a16_gemm(x_u16: np.ndarray, qweight: np.ndarray, scales_u16: np.ndarray, group: int = GROUP) -> np.ndarray:
    """y_ref[m][n] = sum_k double(x[m][k]) * (double(q[n][k]) * double(s[k//group][n])),
    fp64 [M][N].  The definition written out; the contraction itself is numpy's fp64 matmul
    (a library primitive used as one step, no blocking or reordering of ours)."""
    x = bf16_to_f32(x_u16).astype(np.float64)
    return x @ dequantize(qweight, scales_u16, group).T



# ----------------------------------------------------------------------------
# (f3) W8A16 drafter (Table 4 "RTN W8").  Same conventions as W4 with 127 in
#      place of 7; readings (W1-W3): symmetric, group 128, bf16 scale = bf16_RNE(amax / 127), codes
#      clamped to [-127, 127]; stored as TWO nibble planes per group in the W4 layout, so that the W4 kernels can
#      contract it: q + 128 = 16 a + b, a, b in [0, 15].
# ----------------------------------------------------------------------------
QMAX8 = 127


def quantize_codes8(w_u16: np.ndarray, group: int = GROUP):
    """bf16 W[N][K] -> (codes int16 [N][K] in [-127, 127], scales uint16 bf16 bits [K/group][N]); per group:
    s = bf16_RNE(fp32(amax) / fp32(127)), q = clamp(rint(fp32(w) / fp32(s)), -127, 127), s == 0 -> q = 0."""
    w_u16 = np.asarray(w_u16, dtype=np.uint16)
    N, K = w_u16.shape
    assert K % group == 0
    G = K // group
    w = bf16_to_f32(w_u16).reshape(N, G, group)
    amax = np.max(np.abs(w), axis=2)
    s_u16 = f32_to_bf16_rne(amax / np.float32(QMAX8))
    s = bf16_to_f32(s_u16)
    safe = np.where(s == 0, np.float32(1), s)
    with np.errstate(invalid="ignore"):
        ratio = (w / safe[:, :, None]).astype(np.float32)
    q = np.clip(np.rint(ratio), -QMAX8, QMAX8)
    q = np.where((s == 0)[:, :, None], np.float32(0), q)
    s_u16 = np.where(s == 0, np.uint16(0), s_u16)
    return q.astype(np.int16).reshape(N, K), np.ascontiguousarray(s_u16.T)


def pack_codes8(codes8: np.ndarray, scales_u16: np.ndarray, group: int = GROUP):
    """W8 codes + scales -> the two-plane W4 storage: (qweight uint32 [N][2K/8], scales' bf16 bits [2K/group][N]).
    Group g of the W8 matrix becomes groups 2g (plane of the high nibbles a, scale 16 s) and 2g + 1 (plane of the low
    nibbles b, scale s) of a W4 matrix with 2K columns, packed by pack_codes (stored nibble = plane value)."""
    codes8 = np.asarray(codes8, dtype=np.int32)
    N, K = codes8.shape
    G = K // group
    u = (codes8 + 128).reshape(N, G, group)
    assert u.min() >= 1 and u.max() <= 255
    planes = np.stack([u >> 4, u & 15], axis=2)                      # [N][G][2][group], values 0..15
    codes4 = (planes.reshape(N, 2 * K) - 8).astype(np.int8)          # pack_codes stores q4 + 8 = the plane value
    s = bf16_to_f32(np.asarray(scales_u16, dtype=np.uint16))         # [G][N]
    s16 = f32_to_bf16_rne(s * np.float32(16))                        # exact (a power of two) unless it overflows
    scales2 = np.stack([s16, np.asarray(scales_u16, dtype=np.uint16)], axis=1).reshape(2 * G, N)
    return pack_codes(codes4), np.ascontiguousarray(scales2)


def unpack_codes8(qweight2: np.ndarray, group: int = GROUP) -> np.ndarray:
    """Inverse of pack_codes8 on the codes: two-plane storage -> int16 codes [N][K] in [-127, 127]."""
    planes = unpack_codes(qweight2).astype(np.int32) + 8             # [N][2K], values 0..15
    N, K2 = planes.shape
    p = planes.reshape(N, K2 // (2 * group), 2, group)
    return (16 * p[:, :, 0, :] + p[:, :, 1, :] - 128).reshape(N, K2 // 2).astype(np.int16)


def quantize_pack8(w_u16: np.ndarray, group: int = GROUP):
    """The W8 refresh call: bf16 W[N][K] -> (qweight uint32 [N][2K/8] two-plane, scales' bf16 bits [2K/group][N])."""
    return pack_codes8(*quantize_codes8(w_u16, group), group)


def w8a16_gemm(x_u16: np.ndarray, qweight2: np.ndarray, scales2_u16: np.ndarray, group: int = GROUP) -> np.ndarray:
    """y_ref[m][n] = sum_k double(x[m][k]) * double(q[n][k]) * double(s[k // group][n]), fp64; q from the two planes,
    s = the low plane's scale (row 2g + 1 of scales')."""
    x = bf16_to_f32(x_u16).astype(np.float64)
    q = unpack_codes8(qweight2, group).astype(np.float64)
    s = bf16_to_f32(np.asarray(scales2_u16, dtype=np.uint16)[1::2]).astype(np.float64)   # [G][N]
    return x @ (q * np.repeat(s.T, group, axis=1)).T


def bf16_gemm(x_u16: np.ndarray, w_u16: np.ndarray) -> np.ndarray:
    """y_ref[m][n] = sum_k double(x[m][k]) * double(w[n][k]) with bf16 weights W[N][K] (the drafter's lm_head kept in
    higher precision; the target model's linears behind T_p / T_V of Eq. 1).
    The definition written out; numpy's fp64 matmul is the library primitive used as the one step."""
    x = bf16_to_f32(x_u16).astype(np.float64)
    w = bf16_to_f32(w_u16).astype(np.float64)
    return x @ w.T


# ----------------------------------------------------------------------------
# (3) speculative verification by rejection sampling  ("preserves the
#     target-model distribution through rejection sampling"; L445 accept / first
#     rejection resampled "from the adjusted target distribution" / bonus token;
#     L544 exact SD needs the full distribution at the rejected position, ref. [29])
# ----------------------------------------------------------------------------

def softmax64(logits, temperature: float = 1.0) -> np.ndarray:
    """fp64 softmax over the last axis of float32(logits)/T with max-subtraction (V7)."""
    z = np.asarray(logits, dtype=np.float32).astype(np.float64) / np.float64(temperature)
    z = z - np.max(z, axis=-1, keepdims=True)
    e = np.exp(z)
    return e / np.sum(e, axis=-1, keepdims=True)


def spec_verify(target, draft, draft_tokens, u_accept, u_sample, *, inputs_are_logits: bool,
                temperature: float = 1.0, return_diag: bool = False):
    """Textbook speculative rejection sampling, one sequence at a time.

    target [B][gamma+1][V], draft [B][gamma][V]: float32 probabilities, or logits (any
    float dtype already widened to float32 by the caller) when inputs_are_logits.
    draft_tokens int32 [B][gamma]; u_accept fp32 [B][gamma] in [0,1); u_sample fp32 [B].

    Steps (V1-V12):
      1. p_i, q_i in fp64 (softmax64 for logits; widening for probabilities).
      2. n = 0; for i = 1..gamma: accept iff fp32(u_i) * fp32(q_i(x_i)) < fp32(p_i(x_i))
         -- one fp32 multiply, then a strict compare; stop at the first failure.
      3. n < gamma: w = max(0, p_{n+1} - q_{n+1});  n == gamma: w = p_{gamma+1} (bonus).
         R = sum_v w(v); if R == 0 fall back to w = p_{n+1}.
      4. token = min{ v : C(v) > r R },  C = inclusive prefix sum of w in vocab order.
      5. accept_count = n; out_tokens = x_1..x_n, token, then -1 padding.
    """
    target = np.asarray(target)
    draft = np.asarray(draft)
    B, G1, V = target.shape
    gamma = G1 - 1
    assert draft.shape == (B, gamma, V)
    x = np.asarray(draft_tokens, dtype=np.int64).reshape(B, gamma)
    ua = np.asarray(u_accept, dtype=np.float32).reshape(B, gamma)
    us = np.asarray(u_sample, dtype=np.float32).reshape(B)

    accept_count = np.zeros(B, dtype=np.int32)
    out_tokens = np.full((B, gamma + 1), -1, dtype=np.int32)
    diag = []
    for b in range(B):
        if inputs_are_logits:
            p = softmax64(target[b], temperature)
            q = softmax64(draft[b], temperature)
        else:
            p = target[b].astype(np.float64)
            q = draft[b].astype(np.float64)
        n = 0
        margins = []
        for i in range(gamma):
            pf = np.float32(p[i, x[b, i]])
            qf = np.float32(q[i, x[b, i]])
            lhs = np.float32(ua[b, i] * qf)          # fp32 multiply, round to nearest
            margins.append(abs(float(lhs) - float(pf)) / max(float(pf), 1e-300))
            if lhs < pf:
                n += 1
            else:
                break
        if n < gamma:
            w = np.maximum(0.0, p[n] - q[n])
        else:
            w = p[gamma].copy()
        R = float(np.sum(w))
        if R == 0.0:
            w = p[n].copy()
            R = float(np.sum(w))
        C = np.cumsum(w)                             # fp64, ascending v
        thr = float(us[b]) * R
        tok = int(np.searchsorted(C, thr, side="right"))   # first v with C(v) > thr
        tok = min(tok, V - 1)
        accept_count[b] = n
        out_tokens[b, :n] = x[b, :n]
        out_tokens[b, n] = tok
        if return_diag:
            diag.append({"margins": margins, "C": C, "R": R, "w": w, "r": float(us[b])})
    if return_diag:
        return accept_count, out_tokens, diag
    return accept_count, out_tokens


def token_in_widened_interval(d: dict, token: int, slack: float = 1e-5) -> bool:
    """Rule V10: a device token t' that differs from the oracle's passes iff
    w(t') > 0 and r lies in t' 's own fp64 CDF interval widened by `slack` on both sides:
    C(t'-1)/R - slack <= r < C(t')/R + slack."""
    C, R, w, r = d["C"], d["R"], d["w"], d["r"]
    if token < 0 or token >= len(C) or not (w[token] > 0):
        return False
    lo = (C[token - 1] if token > 0 else 0.0) / R
    hi = C[token] / R
    return (lo - slack) <= r < (hi + slack)


# ----------------------------------------------------------------------------
# block efficiency: tau = (1 - alpha^(gamma+1)) / (1 - alpha)
# ----------------------------------------------------------------------------

def block_efficiency(alpha: float, gamma: float) -> float:
    if alpha == 1.0:
        return gamma + 1.0
    return (1.0 - alpha ** (gamma + 1.0)) / (1.0 - alpha)
