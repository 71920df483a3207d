"""TEST INFRASTRUCTURE ONLY -- the oracle of SURVEY.md 8(f) f2: the roofline cost model, the SD toggle policy pi_SD,
the block-efficiency bookkeeping, the adaptive draft-length controller and the two-step calibration of
arxiv/paper_2606_18967, written out from the paper in plain Python / numpy fp64.  Only tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / reference legs may import it; the product (csrc/sd_policy.cu behind include/er.h) shares
no code with it.

Notation follows the paper.  Every function cites the passage it restates.  Pins (tests/test_oracle_policy.py): closed
forms of tau(alpha, gamma) (gamma = 1: 1 + alpha; alpha -> 1: gamma + 1; geometric series by brute force), the roofline
times at hand-computed points on both sides of the memory / compute crossover, Eq. 3 at a threshold case worked by hand,
Alg. 1 line 11-12 on hand-written tau histories, exact recovery of planted parameters by the calibration on noise-free
sweeps (memory-bound, compute-bound and mixed), and the rollout driver against a closed form for constant costs.

Readings where the paper is silent (P1-P5):
  P1  the fit of PAPER.md:L478-L484 is ordinary least squares on seconds; a sample is treated as memory-bound or
      compute-bound by the current estimate and the classification / fit pair is iterated to a fixed point (the paper
      names the parameters of each of its two steps, not the estimator).
  P2  c_V is fitted from the verification sweep with max{M_T, (gamma + 1) C} evaluated with the step-1 parameters.
  P3  min / max of Alg. 1 line 11 run over the last P recorded tau values; with fewer than P values recorded the draft
      length is kept (a condition cannot have "persisted for P consecutive training steps", earlier).
  P4  alpha from tau by bisection on [0, 1]: tau is strictly increasing in alpha.
  P5  the rollout driver is OUR measurement harness (a fluid model of a shrinking batch), not a part of the paper.
"""
from __future__ import annotations

import dataclasses

import numpy as np


@dataclasses.dataclass
class RooflineModel:
    """PAPER.md:L111 (M_T, M_D, C), L455-L469 (parameter details).  SI units: bytes, flop, seconds."""
    W_T: float            # target weight bytes
    W_D: float            # W4 drafter weight bytes (lm_head etc. stay in higher precision)
    C_dense: float        # dense flop per token (FFN, QKVO, lm_head)
    C_attn: float         # attention flop per token and per token of context
    kappa: float          # theoretical KV bytes per token of context
    F_eff: float          # flop/s, calibration stage 1
    BW_eff: float         # bytes/s
    rho_kappa: float      # kappa_eff = rho_kappa * kappa
    eta_D: float
    c_T: float            # seconds per sequence of the batch
    c_D: float
    c_V: float
    c_comm: float = 0.0   # PAPER.md:L473 Eq. 4 (TP > 1); 0 for TP = 1


def tau_of_alpha(alpha: float, gamma: int) -> float:
    """tau = (1 - alpha^(gamma+1)) / (1 - alpha) = sum_{i=0..gamma} alpha^i."""
    if alpha == 1.0:
        return float(gamma + 1)
    return (1.0 - alpha ** (gamma + 1)) / (1.0 - alpha)


def alpha_of_tau(tau: float, gamma: int) -> float:
    """PAPER.md:L534 ("We compute alpha from the measured tau using the equation ..."); reading P4."""
    if tau <= 1.0:
        return 0.0
    if tau >= gamma + 1:
        return 1.0
    lo, hi = 0.0, 1.0
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if tau_of_alpha(mid, gamma) < tau:
            lo = mid
        else:
            hi = mid
    return 0.5 * (lo + hi)


def roofline_times(m: RooflineModel, B: float, S: float, gamma: int):
    """M_T = (W_T + kappa_eff B S) / BW_eff, M_D = (eta_D W_D + kappa_eff B S) / BW_eff,
    C = B (C_dense + S C_attn) / F_eff; L115: T_p = max{M_T, C} + c_T B, T_q = max{M_D, C} + c_D B,
    T_V = max{M_T, (gamma + 1) C} + c_V B; L473 Eq. 4: + c_comm on each."""
    kv = m.rho_kappa * m.kappa * B * S
    M_T = (m.W_T + kv) / m.BW_eff
    M_D = (m.eta_D * m.W_D + kv) / m.BW_eff
    C = B * (m.C_dense + S * m.C_attn) / m.F_eff
    T_p = max(M_T, C) + m.c_T * B + m.c_comm
    T_q = max(M_D, C) + m.c_D * B + m.c_comm
    T_V = max(M_T, (gamma + 1) * C) + m.c_V * B + m.c_comm
    return T_p, T_q, T_V


def sd_speedup(tau: float, T_p: float, T_q: float, T_V: float, gamma: int) -> float:
    """PAPER.md:L68 Eq. 1: Speedup_SD = tau T_p / (gamma T_q + T_V)."""
    return tau * T_p / (gamma * T_q + T_V)


def sd_toggle(m: RooflineModel, B: float, S: float, tau: float, gamma: int, eps: float):
    """PAPER.md:L119 Eq. 3: pi_SD = 1[ tau T_p^ / (gamma T_q^ + T_V^) >= 1 + eps ].  Returns (0 / 1, speedup)."""
    T_p, T_q, T_V = roofline_times(m, B, S, gamma)
    s = sd_speedup(tau, T_p, T_q, T_V, gamma)
    return (1 if s >= 1.0 + eps else 0), s


def gamma_next(Gamma, gamma_t: int, tau_hist, P: int, alpha_up: float, alpha_down: float) -> int:
    """PAPER.md:L168 (Alg. 1 lines 11-12): next_Gamma(gamma_t) if min over the last P tau >= 1 + gamma_t alpha_up and
    gamma_t < gamma_high; prev_Gamma(gamma_t) if max over the last P tau <= 1 + gamma_t alpha_down and
    gamma_t > gamma_low; else gamma_t.  Reading P3 for short histories."""
    Gamma = list(Gamma)
    i = Gamma.index(gamma_t)
    if len(tau_hist) < P:
        return gamma_t
    window = list(tau_hist)[-P:]
    if min(window) >= 1.0 + gamma_t * alpha_up and i + 1 < len(Gamma):
        return Gamma[i + 1]
    if max(window) <= 1.0 + gamma_t * alpha_down and i > 0:
        return Gamma[i - 1]
    return gamma_t


def _lstsq(rows, rhs):
    A = np.asarray(rows, dtype=np.float64)
    b = np.asarray(rhs, dtype=np.float64)
    keep = np.any(A != 0.0, axis=0)           # an unknown no sample touches stays 0
    x = np.zeros(A.shape[1])
    if keep.any():
        x[keep] = np.linalg.lstsq(A[:, keep], b, rcond=None)[0]
    return x


def calibrate(m: RooflineModel, target, drafter, verify, iters: int = 50) -> RooflineModel:
    """PAPER.md:L478-L484, two-step fit (readings P1, P2).  F_eff and the static terms of `m` are given (stage 1 and
    the architecture); returns a copy with BW_eff, rho_kappa, c_T (step 1, from the target sweep) and eta_D, c_D, c_V
    (step 2, from the drafter and verification sweeps) fitted.
      target   rows (B, S, T_p);  drafter  rows (B, S, T_q);  verify  rows (B, S, gamma, T_V)   [seconds]
    T_p - c_comm = max{a W_T + b kappa B S, C} + c_T B with a = 1 / BW_eff, b = rho_kappa / BW_eff is linear in
    (a, b, c_T) once every sample is classed as memory- or compute-bound; class and fit are iterated."""
    out = dataclasses.replace(m)
    C_of = lambda B, S: B * (m.C_dense + S * m.C_attn) / m.F_eff
    a, b, cT = 1.0 / m.BW_eff, m.rho_kappa / m.BW_eff, m.c_T
    mem = None
    for _ in range(iters):
        new = [a * m.W_T + b * m.kappa * B * S >= C_of(B, S) for B, S, _ in target]
        if new == mem:
            break
        mem = new
        rows = [[m.W_T, m.kappa * B * S, B] if k else [0.0, 0.0, B] for (B, S, _), k in zip(target, mem)]
        rhs = [T - m.c_comm - (0.0 if k else C_of(B, S)) for (B, S, T), k in zip(target, mem)]
        x = _lstsq(rows, rhs)
        if x[0] > 0.0:
            a = x[0]
        b, cT = x[1], x[2]
    out.BW_eff = 1.0 / a
    out.rho_kappa = b / a
    out.c_T = cT
    # step 2a: eta_D, c_D from the drafter sweep, BW_eff and rho_kappa fixed
    kv = lambda B, S: out.rho_kappa * m.kappa * B * S / out.BW_eff
    eta, cD = m.eta_D, m.c_D
    mem = None
    for _ in range(iters):
        new = [eta * m.W_D / out.BW_eff + kv(B, S) >= C_of(B, S) for B, S, _ in drafter]
        if new == mem:
            break
        mem = new
        rows = [[m.W_D / out.BW_eff, B] if k else [0.0, B] for (B, S, _), k in zip(drafter, mem)]
        rhs = [T - m.c_comm - (kv(B, S) if k else C_of(B, S)) for (B, S, T), k in zip(drafter, mem)]
        x = _lstsq(rows, rhs)
        if x[0] > 0.0:
            eta = x[0]
        cD = x[1]
    out.eta_D, out.c_D = eta, cD
    # step 2b: c_V from the verification sweep
    num = den = 0.0
    for B, S, gamma, T in verify:
        base = max(m.W_T / out.BW_eff + kv(B, S), (gamma + 1) * C_of(B, S))
        num += B * (T - m.c_comm - base)
        den += B * B
    out.c_V = num / den if den > 0.0 else m.c_V
    return out


def simulate_rollout(m: RooflineModel, lengths, S0: float, gamma: int, tau: float, eps: float, mode: int):
    """Reading P5 (our measurement driver for PAPER.md:L145-L160, Alg. 1 lines 4-10; the paper's rollouts are real):
    `lengths` response lengths in tokens; every active sequence advances one token per AR step (cost T_p^(B, S)) and tau
    tokens per SD block (cost gamma T_q^ + T_V^), B = #{lengths > position}, S = S0 + position.  mode 0: AR only;
    1: SD from the first step; 2: pi_SD decides, sticky once on.  Returns (seconds, steps, steps decoded
    autoregressively)."""
    L = np.sort(np.asarray(lengths, dtype=np.float64))
    pos, t, steps, ar_steps = 0.0, 0.0, 0, 0
    sd_on = mode == 1
    Lmax = float(L[-1]) if len(L) else 0.0
    while pos < Lmax:
        B = float(len(L) - np.searchsorted(L, pos, side="right"))
        S = S0 + pos
        if mode == 2 and not sd_on and sd_toggle(m, B, S, tau, gamma, eps)[0] == 1:
            sd_on = True
        T_p, T_q, T_V = roofline_times(m, B, S, gamma)
        if sd_on:
            t += gamma * T_q + T_V
            pos += tau
        else:
            t += T_p
            pos += 1.0
            ar_steps += 1
        steps += 1
    return t, steps, ar_steps
