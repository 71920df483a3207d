"""Pins for the oracle's speculative verification (V1-V12).  CPU only."""
import itertools
from fractions import Fraction

import numpy as np
import scipy.special

from oracle import er_oracle as O
from paper_2606_18967_b200 import inputs as I


def _probs(B, G, V, seed):
    rng = np.random.default_rng(seed)
    p = rng.random((B, G, V)).astype(np.float32)
    return (p / p.sum(-1, keepdims=True)).astype(np.float32)


def test_softmax_against_scipy():
    rng = np.random.default_rng(0)
    z = (rng.standard_normal((3, 1000)) * 2).astype(np.float32)
    for T in (1.0, 0.6):
        ref = scipy.special.softmax(z.astype(np.float64) / T, axis=-1)
        assert np.allclose(O.softmax64(z, T), ref, rtol=1e-13, atol=0)


def test_q_equals_p_accepts_everything():
    B, G, V = 6, 4, 50
    p = _probs(B, G + 1, V, 1)
    x = I.sample_draft_tokens(p[:, :G], seed=3)
    ua = I.uniforms((B, G), 4)
    us = I.uniforms((B,), 5)
    n, out = O.spec_verify(p, p[:, :G].copy(), x, ua, us, inputs_are_logits=False)
    assert np.all(n == G)
    assert np.array_equal(out[:, :G], x)
    # bonus token is the inverse CDF of p_{gamma+1} at r
    for b in range(B):
        C = np.cumsum(p[b, G].astype(np.float64))
        t = out[b, G]
        lo = C[t - 1] if t > 0 else 0.0
        assert lo <= us[b] * C[-1] < C[t]


def test_one_hot_target_and_zero_probability():
    V, G = 8, 2
    q = np.full((1, G, V), 1.0 / V, dtype=np.float32)
    x = np.array([[3, 5]], dtype=np.int32)
    p = np.zeros((1, G + 1, V), dtype=np.float32)
    p[0, 0, 3] = 1.0          # one-hot on x_1 -> accepted for any u < 1
    p[0, 1, 2] = 1.0          # p(x_2) = 0 -> rejected, resampled token != x_2 (must be 2)
    p[0, 2, 0] = 1.0
    n, out = O.spec_verify(p, q, x, np.array([[0.999999, 0.0]], np.float32), np.array([0.5], np.float32),
                           inputs_are_logits=False)
    assert n[0] == 1 and list(out[0]) == [3, 2, -1]


def test_strictness_and_u_zero():
    V = 4
    p = np.array([[[0.25, 0.25, 0.25, 0.25], [0.1, 0.2, 0.3, 0.4]]], np.float32)
    q = np.array([[[0.5, 0.25, 0.125, 0.125]]], np.float32)
    x = np.array([[0]], np.int32)
    # u*q == p exactly (0.5*0.5 = 0.25): strict '<' rejects
    n, _ = O.spec_verify(p, q, x, np.array([[0.5]], np.float32), np.array([0.0], np.float32), inputs_are_logits=False)
    assert n[0] == 0
    n, out = O.spec_verify(p, q, x, np.array([[0.0]], np.float32), np.array([0.0], np.float32), inputs_are_logits=False)
    assert n[0] == 1 and out[0, 1] == 0        # r = 0 -> first v with w > 0 (bonus row)


def test_zero_residual_falls_back_to_target():
    # artificial w == 0: p == q bitwise but the accept test is forced to fail via u*q == p ... impossible for u<1,
    # so drive the fallback directly with p(x)=q(x)=0 at the drafted token (accept iff 0 < 0 -> reject) and p == q.
    p = np.array([[[0.0, 0.5, 0.5], [1.0, 0.0, 0.0]]], np.float32)
    q = np.array([[[0.0, 0.5, 0.5]]], np.float32)
    n, out = O.spec_verify(p, q, np.array([[0]], np.int32), np.array([[0.3]], np.float32),
                           np.array([0.6], np.float32), inputs_are_logits=False)
    assert n[0] == 0 and out[0, 0] == 2       # R = 0 -> sample from p_1: C = (0, .5, 1), r = .6 -> token 2


def _exact_output_histogram(p16, q16, gamma):
    """Enumerate drafted tokens (weighted by q), u and r on midpoint grids fine enough that every threshold falls on a
    grid edge, run the ORACLE on each grid point, and return the exact distribution of the first emitted token."""
    V = len(p16[0])
    p = np.array([[Fraction(a, 16) for a in row] for row in p16], dtype=object)
    q = np.array([[Fraction(a, 16) for a in row] for row in q16], dtype=object)
    pf = np.array([[float(a) for a in row] for row in p], np.float32)[None]
    qf = np.array([[float(a) for a in row] for row in q], np.float32)[None]
    # u-grid: multiple of every q numerator so p/q thresholds are grid edges; r-grid: multiple of 16 R and of 16
    Gu = int(np.lcm.reduce([a for row in q16 for a in row if a > 0])) * 4
    res16 = [sum(max(0, a - b) for a, b in zip(p16[i], q16[i])) for i in range(gamma)]
    Gr = int(np.lcm.reduce([r for r in res16 if r > 0] + [16])) * 2
    hist = [Fraction(0)] * V
    for xs in itertools.product(range(V), repeat=gamma):
        wx = Fraction(1)
        for i, xv in enumerate(xs):
            wx *= q[i][xv]
        if wx == 0:
            continue
        for us_idx in itertools.product(range(Gu), repeat=gamma):
            ua = np.array([[(j + 0.5) / Gu for j in us_idx]], np.float32)
            for jr in range(Gr):
                r = np.array([(jr + 0.5) / Gr], np.float32)
                _, out = O.spec_verify(pf, qf, np.array([xs], np.int32), ua, r, inputs_are_logits=False)
                hist[int(out[0, 0])] += wx * Fraction(1, Gu ** gamma) * Fraction(1, Gr)
    return hist, [p[0][v] for v in range(V)]


def test_brute_force_output_distribution_equals_target_gamma1():
    # P(out = v) = min(p,q)(v) + (1 - sum min(p,q)) * max(0,p-q)(v)/R = p(v)   (ref. [29])
    p16 = [[1, 9, 4, 2], [4, 4, 4, 4]]
    q16 = [[6, 2, 3, 5]]
    hist, p1 = _exact_output_histogram(p16, q16, gamma=1)
    assert hist == p1


def test_brute_force_output_distribution_equals_target_gamma2_v3():
    p16 = [[2, 10, 4], [8, 4, 4], [4, 4, 8]]
    q16 = [[8, 4, 4], [4, 8, 4]]
    hist, p1 = _exact_output_histogram(p16, q16, gamma=2)
    assert hist == p1


def test_second_position_distribution_given_first_accepted():
    # conditional on accepting x_1, the token emitted at position 2 follows p_2 exactly
    p16 = [[8, 8], [3, 13], [8, 8]]
    q16 = [[8, 8], [12, 4]]
    pf = np.array(p16, np.float32)[None] / 16
    qf = np.array(q16, np.float32)[None] / 16
    Gu, Gr = 48, 32 * 9
    hist = [Fraction(0), Fraction(0)]
    for x2 in range(2):
        for j in range(Gu):
            for jr in range(Gr):
                ua = np.array([[0.25, (j + 0.5) / Gu]], np.float32)       # u_1 = .25 always accepts (p=q at pos 1)
                _, out = O.spec_verify(pf, qf, np.array([[0, x2]], np.int32), ua,
                                       np.array([(jr + 0.5) / Gr], np.float32), inputs_are_logits=False)
                assert out[0, 0] == 0
                hist[int(out[0, 1])] += Fraction(q16[1][x2], 16) * Fraction(1, Gu * Gr)
    assert hist == [Fraction(3, 16), Fraction(13, 16)]


def test_statistical_acceptance_rate_matches_sum_min():
    B, G, V = 400, 3, 64
    tgt, drf = I.verify_logits_f32(B, G, V, seed=9, std=1.0, draft_noise=0.5)
    p = O.softmax64(tgt)
    q = O.softmax64(drf)
    x = I.sample_draft_tokens(q, seed=10)
    n, out = O.spec_verify(tgt, drf, x, I.uniforms((B, G), 11), I.uniforms((B,), 12), inputs_are_logits=True)
    alpha1 = np.minimum(p[:, 0], q[:, 0]).sum(-1).mean()
    rate = np.mean(n >= 1)
    sigma = np.sqrt(alpha1 * (1 - alpha1) / B)
    assert abs(rate - alpha1) < 3.5 * sigma
    # tau = mean(n) + 1 matches (1 - a^(g+1)) / (1 - a) when alpha is nearly constant across positions
    alpha = np.minimum(p[:, :G], q).sum(-1).mean()
    assert abs((n.mean() + 1) - O.block_efficiency(alpha, G)) < 0.15
    assert np.all(out[np.arange(B), n] >= 0) and np.all((out >= 0).sum(1) == n + 1)


def test_block_efficiency_matches_paper_table2():
    for line in open(__file__.rsplit("/", 1)[0] + "/golden/tau_table2.txt"):
        if line.startswith("#") or not line.strip():
            continue
        a, g, tau, _ = line.split()
        assert abs(O.block_efficiency(float(a) / 100, float(g)) - float(tau)) <= 0.05 + 1e-9
    assert O.block_efficiency(1.0, 5) == 6.0


def test_widened_interval_rule():
    # Rule V10, pinned on a hand-built dyadic CDF with R != 1 -- every expectation below is arithmetic
    # done on paper, none of it comes from the function under test:
    #   w = (1/4, 0, 1/2, 1/8, 5/8), R = 3/2, C = (1/4, 1/4, 3/4, 7/8, 3/2), C/R = (1/6, 1/6, 1/2, 7/12, 1)
    # token intervals in units of R: 0:[0,1/6)  1:empty (w = 0)  2:[1/6,1/2)  3:[1/2,7/12)  4:[7/12,1)
    w = np.array([0.25, 0.0, 0.5, 0.125, 0.625])
    C = np.array([0.25, 0.25, 0.75, 0.875, 1.5])
    assert np.array_equal(np.cumsum(w), C)
    mk = lambda r: {"C": C, "R": 1.5, "w": w, "r": r, "margins": []}
    # r just above the upper edge of token 2 (the exact token is 3): 0.9e-5 inside the slack, 1.1e-5 outside
    assert O.token_in_widened_interval(mk(0.5 + 0.9e-5), 2)
    assert not O.token_in_widened_interval(mk(0.5 + 1.1e-5), 2)
    # r just below the lower edge of token 3 (the exact token is 2)
    assert O.token_in_widened_interval(mk(0.5 - 0.9e-5), 3)
    assert not O.token_in_widened_interval(mk(0.5 - 1.1e-5), 3)
    # (a missing division by R would put token 3's lower edge at 0.75 and fail the third line; a slack of 1e-1 or
    #  1e-4 would pass the second and fourth)
    # a token without mass never passes, even when r sits exactly on its (empty) interval
    assert not O.token_in_widened_interval(mk(1.0 / 6.0), 1)
    # the exact token always passes; neighbours far from r do not
    for r, t in ((0.1, 0), (0.3, 2), (0.55, 3), (0.9, 4)):
        assert O.token_in_widened_interval(mk(r), t)
        for other in range(5):
            if other != t:
                assert not O.token_in_widened_interval(mk(r), other), (r, t, other)
    # first token: lower edge is 0 (no C[-1] wrap-around to the total mass)
    assert O.token_in_widened_interval(mk(0.0), 0) and not O.token_in_widened_interval(mk(0.0), 4)
    # out-of-range ids
    assert not O.token_in_widened_interval(mk(0.3), -1) and not O.token_in_widened_interval(mk(0.3), 5)
    # and through spec_verify's own diagnostics: the oracle's token passes its own window
    p = _probs(1, 2, 10, 7)
    q = _probs(1, 1, 10, 8)
    x = np.array([[0]], np.int32)
    n, out, diag = O.spec_verify(p, q, x, np.array([[0.999]], np.float32), np.array([0.4], np.float32),
                                 inputs_are_logits=False, return_diag=True)
    assert O.token_in_widened_interval(diag[0], int(out[0, n[0]]))
