"""Pins of oracle/er_policy.py (roofline model, pi_SD, tau / alpha, adaptive gamma, calibration) against
what the paper prints and the mathematics fixes -- nothing here calls the product."""
import itertools
import os

import numpy as np
import pytest

from oracle import er_policy as P

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _model(**kw):
    base = dict(W_T=16e9, W_D=5e9, C_dense=2 * 7.6e9, C_attn=4 * 28 * 3584.0, kappa=28 * 2 * 4 * 128 * 2.0,
                F_eff=1.0e15, BW_eff=6.0e12, rho_kappa=0.5, eta_D=1.3, c_T=2e-6, c_D=3e-6, c_V=5e-6, c_comm=0.0)
    base.update(kw)
    return P.RooflineModel(**base)


# ---- tau / alpha ----------------------------------------------------------------------------
def test_tau_closed_forms():
    for a in (0.0, 0.3, 0.8, 0.981):
        assert P.tau_of_alpha(a, 1) == pytest.approx(1.0 + a, rel=1e-15)          # gamma = 1: 1 + alpha
        for g in (2, 5, 11):
            assert P.tau_of_alpha(a, g) == pytest.approx(sum(a ** i for i in range(g + 1)), rel=1e-13)   # the series
    assert P.tau_of_alpha(1.0, 7) == 8.0 and P.tau_of_alpha(0.0, 7) == 1.0
    assert P.tau_of_alpha(1.0 - 1e-9, 7) == pytest.approx(8.0, rel=1e-6)          # continuous at alpha = 1


def test_tau_is_expected_block_length_by_enumeration():
    # i.i.d. acceptance with probability alpha: tokens per block = accepted prefix + 1; exact expectation over all
    # 2^gamma accept / reject patterns
    a, g = 0.7, 4
    e = 0.0
    for pat in itertools.product((0, 1), repeat=g):
        pr = np.prod([a if x else 1 - a for x in pat])
        n = next((i for i, x in enumerate(pat) if not x), g)
        e += pr * (n + 1)
    assert P.tau_of_alpha(a, g) == pytest.approx(e, rel=1e-13)


def test_table2_rows_as_printed():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "table2_tau_alpha.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 6
    for *_, tau, g, a in rows:
        tau, g, a = float(tau), int(g), float(a) / 100.0
        assert abs(P.tau_of_alpha(a, g) - tau) <= 0.05 + 1e-9                    # tau printed to one decimal
        lo, hi = P.alpha_of_tau(tau - 0.05, g), P.alpha_of_tau(tau + 0.05, g)     # and alpha inverts it
        assert lo - 5e-4 <= a <= hi + 5e-4


def test_alpha_of_tau_inverts_and_clamps():
    for g in (1, 3, 7, 15):
        for a in (0.0, 0.05, 0.5, 0.9, 0.999):
            assert P.alpha_of_tau(P.tau_of_alpha(a, g), g) == pytest.approx(a, abs=1e-12)
        assert P.alpha_of_tau(0.5, g) == 0.0 and P.alpha_of_tau(g + 2.0, g) == 1.0


# ---- roofline times and Eq. 3 ------------------------------------------------------------------
def test_roofline_times_by_hand_memory_bound():
    # B = 1, S = 0: everything is weight traffic.  M_T = 16e9 / 6e12, M_D = 1.3 * 5e9 / 6e12, C = 15.2e9 / 1e15
    m = _model()
    T_p, T_q, T_V = P.roofline_times(m, 1, 0, 4)
    assert T_p == pytest.approx(16e9 / 6e12 + 2e-6, rel=1e-14)
    assert T_q == pytest.approx(6.5e9 / 6e12 + 3e-6, rel=1e-14)
    assert T_V == pytest.approx(16e9 / 6e12 + 5e-6, rel=1e-14)       # (gamma + 1) C = 7.6e-5 << M_T: verify is "free"


def test_roofline_times_by_hand_compute_bound_and_kv():
    # B = 512, S = 1000: C = 512 (15.2e9 + 1000 * 401408) / 1e15 = 7.98792...e-3;  kv = 0.5 * 57344 * 512 * 1000
    m = _model()
    B, S, g = 512.0, 1000.0, 4
    C = B * (15.2e9 + S * 4 * 28 * 3584.0) / 1e15
    kv = 0.5 * 57344.0 * B * S
    M_T, M_D = (16e9 + kv) / 6e12, (6.5e9 + kv) / 6e12
    assert C > M_T > M_D                                                 # the compute side of the crossover
    T_p, T_q, T_V = P.roofline_times(m, B, S, g)
    assert T_p == pytest.approx(C + 2e-6 * B, rel=1e-14)
    assert T_q == pytest.approx(C + 3e-6 * B, rel=1e-14)
    assert T_V == pytest.approx(5 * C + 5e-6 * B, rel=1e-14)
    # c_comm is added once to each (Eq. 4)
    T2 = P.roofline_times(_model(c_comm=1e-4), B, S, g)
    assert np.allclose(np.array(T2) - np.array((T_p, T_q, T_V)), 1e-4, rtol=0, atol=1e-15)


def test_eq1_and_toggle_threshold_by_hand():
    # T_p = 4, T_q = 1, T_V = 5, gamma = 3, tau = 2.1: speedup = 2.1 * 4 / (3 + 5) = 1.05
    assert P.sd_speedup(2.1, 4.0, 1.0, 5.0, 3) == pytest.approx(1.05, rel=1e-15)
    # a model whose times are exactly those: no kv, no compute, W_T / BW = 4, eta W_D / BW = 1, c_V B = 1 at B = 1
    m = _model(W_T=4.0, W_D=1.0, BW_eff=1.0, eta_D=1.0, C_dense=0.0, C_attn=0.0, kappa=0.0, c_T=0.0, c_D=0.0, c_V=1.0)
    assert P.roofline_times(m, 1, 0, 3) == (4.0, 1.0, 5.0)
    on, s = P.sd_toggle(m, 1, 0, 2.2, 3, 0.05)
    assert on == 1 and s == pytest.approx(1.1)
    assert P.sd_toggle(m, 1, 0, 2.0, 3, 0.05)[0] == 0                    # speedup 1.0 < 1.05
    assert P.sd_toggle(m, 1, 0, 2.0, 3, 0.0)[0] == 1                     # ">=": equality switches SD on
    # large batches are compute-bound: verification costs (gamma + 1) forward passes and SD loses
    big = _model()
    assert P.sd_toggle(big, 2048, 2000, 4.5, 4, 0.05)[0] == 0 and P.sd_toggle(big, 2, 2000, 4.5, 4, 0.05)[0] == 1


# ---- adaptive draft length --------------------------------------------------------------------
def test_gamma_controller_by_hand():
    G, up, dn = [5, 7, 9, 11], 0.94, 0.85                                # the paper's configuration, P = 2
    # gamma = 5: up needs min >= 1 + 5 * 0.94 = 5.7 ; down needs max <= 1 + 5 * 0.85 = 5.25
    assert P.gamma_next(G, 5, [5.8, 5.71], 2, up, dn) == 7
    assert P.gamma_next(G, 5, [5.8, 5.69], 2, up, dn) == 5               # one step of the window below: stays
    assert P.gamma_next(G, 5, [5.0, 5.8, 5.7], 2, up, dn) == 7           # only the last P count
    assert P.gamma_next(G, 5, [3.0, 3.0], 2, up, dn) == 5                # already gamma_low
    assert P.gamma_next(G, 5, [5.9], 2, up, dn) == 5                     # fewer than P steps recorded (reading P3)
    # gamma = 9: down needs max <= 1 + 9 * 0.85 = 8.65 ; up needs min >= 9.46
    assert P.gamma_next(G, 9, [8.64, 8.0], 2, up, dn) == 7
    assert P.gamma_next(G, 9, [8.66, 8.0], 2, up, dn) == 9
    assert P.gamma_next(G, 9, [9.47, 9.5], 2, up, dn) == 11
    assert P.gamma_next(G, 11, [11.9, 11.9], 2, up, dn) == 11            # already gamma_high
    assert P.gamma_next(G, 11, [10.0, 10.34], 2, up, dn) == 9            # 1 + 11 * 0.85 = 10.35
    # ">=" and "<=" include equality (thresholds that are exact in binary: 1 + 2 * 0.75 = 2.5, 1 + 4 * 0.5 = 3)
    assert P.gamma_next([2, 4], 2, [2.5, 2.5], 2, 0.75, 0.5) == 4
    assert P.gamma_next([2, 4], 4, [3.0, 3.0], 2, 0.75, 0.5) == 2


def test_gamma_controller_walks_the_set():
    G = [5, 7, 9, 11]
    g, hist, seen = 5, [], []
    for tau in [5.8, 5.8, 7.7, 7.7, 9.5, 9.5, 9.0, 9.0, 9.0, 6.0, 6.0]:
        hist.append(tau)
        g = P.gamma_next(G, g, hist, 2, 0.94, 0.85)
        seen.append(g)
    # by hand: [5.8] short; [5.8,5.8] >= 5.7 -> 7; [5.8,7.7] neither (7.58 / 6.95); [7.7,7.7] -> 9; [7.7,9.5] neither;
    # [9.5,9.5] >= 9.46 -> 11; [9.5,9.0] max <= 10.35 -> 9; [9,9], [9,9] neither (9.46 / 8.65); [9,6] max 9 > 8.65; [6,6] -> 7
    assert seen == [5, 7, 7, 9, 9, 11, 9, 9, 9, 9, 7]


# ---- calibration -------------------------------------------------------------------------------
def _sweeps(m, Bs, Ss, gammas=(3, 7, 11, 15)):
    tgt = [(B, S, P.roofline_times(m, B, S, 3)[0]) for B in Bs for S in Ss]
    drf = [(B, S, P.roofline_times(m, B, S, 3)[1]) for B in Bs for S in Ss]
    ver = [(B, S, g, P.roofline_times(m, B, S, g)[2]) for B in Bs for S in Ss for g in gammas]
    return tgt, drf, ver


@pytest.mark.parametrize("Bs", [(1, 2, 4, 8, 16), (1, 8, 64, 512, 2048), (512, 1024, 2048)])
def test_calibration_recovers_planted_parameters(Bs):
    # noise-free sweeps generated from known parameters: memory-bound only, mixed, (nearly) compute-bound only
    truth = _model(BW_eff=5.3e12, rho_kappa=0.62, c_T=4e-6, eta_D=1.41, c_D=6e-6, c_V=9e-6)
    start = _model(BW_eff=8.0e12, rho_kappa=1.0, c_T=0.0, eta_D=1.0, c_D=0.0, c_V=0.0)
    fit = P.calibrate(start, *_sweeps(truth, Bs, (128, 1024, 4096)))
    memory_points = any(P.roofline_times(truth, B, S, 3)[0] - truth.c_T * B > B * (truth.C_dense + S * truth.C_attn) / truth.F_eff * (1 + 1e-12)
                        for B in Bs for S in (128, 1024, 4096))
    assert fit.c_T == pytest.approx(truth.c_T, rel=1e-6) and fit.c_V == pytest.approx(truth.c_V, rel=1e-6)
    assert fit.c_D == pytest.approx(truth.c_D, rel=1e-6)
    if memory_points:
        assert fit.BW_eff == pytest.approx(truth.BW_eff, rel=1e-8)
        assert fit.rho_kappa == pytest.approx(truth.rho_kappa, rel=1e-8)
    if Bs[0] == 1:
        assert fit.eta_D == pytest.approx(truth.eta_D, rel=1e-8)
    # static terms are not touched
    assert (fit.W_T, fit.W_D, fit.F_eff, fit.kappa) == (truth.W_T, truth.W_D, truth.F_eff, truth.kappa)


def test_calibration_without_kv_sweep_leaves_rho_at_zero():
    # this repository's path has no attention / KV cache: S = 0 everywhere, the rho_kappa column is empty
    truth = _model(BW_eff=5.3e12, rho_kappa=0.0, kappa=0.0, C_attn=0.0)
    fit = P.calibrate(_model(BW_eff=8e12, rho_kappa=0.0, kappa=0.0, C_attn=0.0, c_T=0, c_D=0, c_V=0, eta_D=1.0),
                      *_sweeps(truth, (1, 4, 16, 64, 256), (0,), gammas=(2, 4, 8)))
    assert fit.rho_kappa == 0.0 and fit.BW_eff == pytest.approx(5.3e12, rel=1e-9)
    assert fit.eta_D == pytest.approx(truth.eta_D, rel=1e-9) and fit.c_V == pytest.approx(truth.c_V, rel=1e-9)


# ---- rollout driver (reading P5) ------------------------------------------------------------------------------------
def test_rollout_driver_closed_form_for_constant_costs():
    # no batch or length dependence: T_p = 4, T_q = 1, T_V = 5 as above; 10 sequences of 100 tokens
    m = _model(W_T=4.0, W_D=1.0, BW_eff=1.0, eta_D=1.0, C_dense=0.0, C_attn=0.0, kappa=0.0, c_T=0.0, c_D=0.0, c_V=0.0)
    m.c_comm = 0.0
    m_v = P.RooflineModel(**{**m.__dict__})
    lengths = [100] * 10
    t_ar, steps_ar, ar = P.simulate_rollout(m_v, lengths, 0, 3, 2.5, 0.05, 0)
    assert (t_ar, steps_ar, ar) == (400.0, 100, 100)
    t_sd, steps_sd, ar = P.simulate_rollout(m_v, lengths, 0, 3, 2.5, 0.05, 1)
    assert steps_sd == 40 and ar == 0 and t_sd == pytest.approx(40 * (3 * 1.0 + 4.0))     # T_V = M_T = 4 here
    t_pi, steps_pi, ar = P.simulate_rollout(m_v, lengths, 0, 3, 2.5, 0.05, 2)
    assert (t_pi, steps_pi, ar) == (t_sd, steps_sd, 0)                    # speedup 2.5 * 4 / 7 > 1.05 from step one


def test_rollout_driver_toggle_beats_both_on_a_long_tail():
    # a long-tailed batch on a model with a compute-bound head: AR early, SD in the tail
    m = _model()
    rng = np.random.default_rng(0)
    lengths = np.minimum(8192, rng.lognormal(6.5, 0.9, size=1024)).astype(int) + 1
    tau = P.tau_of_alpha(0.9, 5)
    t_ar = P.simulate_rollout(m, lengths, 512, 5, tau, 0.05, 0)[0]
    t_sd = P.simulate_rollout(m, lengths, 512, 5, tau, 0.05, 1)[0]
    t_pi, steps, ar_steps = P.simulate_rollout(m, lengths, 512, 5, tau, 0.05, 2)
    assert t_pi <= min(t_ar, t_sd) * (1 + 1e-12) and 0 < ar_steps < steps
