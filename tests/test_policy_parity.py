"""Parity of the host policy entry points of include/er.h (csrc/sd_policy.cu) against
oracle/er_policy.py, through the C ABI.  Host scalars only: these run without a GPU.  Decisions (toggle, next draft
length, step counts) are compared exactly; fp64 values to 1e-12 relative (two independent implementations of the same
formulas; the calibration solves its least-squares problems by Householder QR here and by LAPACK in the oracle)."""
import dataclasses

import numpy as np
import pytest

from oracle import er_policy as P
from paper_2606_18967_b200 import er

FIELDS = [f.name for f in dataclasses.fields(P.RooflineModel)]


def _pair(**kw):
    base = dict(W_T=15.2e9, W_D=5.5e9, C_dense=2 * 7.6e9, C_attn=4 * 28 * 3584.0, kappa=28 * 2 * 4 * 128 * 2.0,
                F_eff=1.4e15, BW_eff=6.4e12, rho_kappa=0.55, eta_D=1.35, c_T=2.5e-6, c_D=3.5e-6, c_V=6e-6, c_comm=0.0)
    base.update(kw)
    c = er.RooflineModel(**base)
    return P.RooflineModel(**base), c


def test_tau_and_alpha():
    rng = np.random.default_rng(1)
    for g in (1, 2, 5, 7, 11, 16):
        for a in list(rng.random(20)) + [0.0, 1.0, 0.981]:
            assert er.tau_of_alpha(a, g) == pytest.approx(P.tau_of_alpha(a, g), rel=1e-13)
        for tau in list(1.0 + rng.random(20) * g) + [0.3, 1.0, g + 1.0, g + 5.0]:
            assert er.alpha_of_tau(tau, g) == pytest.approx(P.alpha_of_tau(tau, g), abs=1e-13)
    with pytest.raises(er.ErError):
        er.tau_of_alpha(0.5, 0)


def test_roofline_times_and_toggle_grid():
    o, c = _pair()
    rng = np.random.default_rng(2)
    n_on = 0
    for B in (1, 2, 8, 32, 128, 512, 2048):
        for S in (0, 256, 2048, 8192):
            for g in (2, 5, 7, 11, 15):
                t_o, t_c = P.roofline_times(o, B, S, g), er.roofline_times(c, B, S, g)
                assert np.allclose(t_o, t_c, rtol=1e-14, atol=0)
                tau = 1.0 + rng.random() * g
                on_o, s_o = P.sd_toggle(o, B, S, tau, g, 0.05)
                on_c, s_c = er.sd_toggle(c, B, S, tau, g, 0.05)
                assert s_c == pytest.approx(s_o, rel=1e-14)
                if abs(s_o - 1.05) > 1e-9:
                    assert on_c == on_o
                n_on += on_o
    assert 0 < n_on < 7 * 4 * 5          # both outcomes occur
    o2, c2 = _pair(c_comm=2e-5)          # Eq. 4
    assert np.allclose(P.roofline_times(o2, 64, 1024, 7), er.roofline_times(c2, 64, 1024, 7), rtol=1e-14)


def test_gamma_next_random_histories():
    rng = np.random.default_rng(3)
    G = [5, 7, 9, 11]
    moves = set()
    for _ in range(2000):
        g = int(rng.choice(G))
        n = int(rng.integers(0, 6))
        hist = list(1.0 + g * (0.8 + 0.2 * rng.random(n)))
        Pw = int(rng.integers(1, 4))
        want = P.gamma_next(G, g, hist, Pw, 0.94, 0.85)
        assert er.gamma_next(G, g, hist, Pw, 0.94, 0.85) == want
        moves.add(int(np.sign(want - g)))
    assert moves == {-1, 0, 1}
    with pytest.raises(er.ErError):
        er.gamma_next(G, 6, [6.0, 6.0], 2, 0.94, 0.85)        # gamma_t not in Gamma
    with pytest.raises(er.ErError):
        er.gamma_next([5, 5, 7], 5, [6.0, 6.0], 2, 0.94, 0.85)   # not ascending


def _sweeps(m, Bs, Ss, gammas, noise=0.0, seed=0):
    rng = np.random.default_rng(seed)
    j = lambda: 1.0 + noise * rng.standard_normal()
    tgt = [(B, S, P.roofline_times(m, B, S, 3)[0] * j()) for B in Bs for S in Ss]
    drf = [(B, S, P.roofline_times(m, B, S, 3)[1] * j()) for B in Bs for S in Ss]
    ver = [(B, S, g, P.roofline_times(m, B, S, g)[2] * j()) for B in Bs for S in Ss for g in gammas]
    return tgt, drf, ver


@pytest.mark.parametrize("noise", [0.0, 0.03])
@pytest.mark.parametrize("Bs,Ss", [((1, 2, 4, 8, 16), (128, 1024, 4096)), ((1, 8, 64, 512, 2048), (128, 1024, 4096)),
                                   ((1, 4, 16, 64, 256), (0,))])
def test_calibration(Bs, Ss, noise):
    truth, _ = _pair(BW_eff=5.3e12, rho_kappa=0.62, c_T=4e-6, eta_D=1.41, c_D=6e-6, c_V=9e-6)
    start_o, start_c = _pair(BW_eff=8.0e12, rho_kappa=1.0 if Ss != (0,) else 0.0, c_T=0.0, eta_D=1.0, c_D=0.0, c_V=0.0)
    sweeps = _sweeps(truth, Bs, Ss, (3, 7, 11, 15), noise, seed=len(Bs) + len(Ss))
    fit_o = P.calibrate(start_o, *sweeps)
    fit_c = er.roofline_calibrate(start_c, *sweeps)
    for f in FIELDS:
        assert getattr(fit_c, f) == pytest.approx(getattr(fit_o, f), rel=1e-9, abs=1e-18), f
    if noise == 0.0:
        assert fit_c.BW_eff == pytest.approx(truth.BW_eff, rel=1e-8) and fit_c.c_V == pytest.approx(truth.c_V, rel=1e-6)


def test_rollout_driver():
    o, c = _pair()
    rng = np.random.default_rng(5)
    lengths = (np.minimum(8192, rng.lognormal(6.5, 0.9, size=512)).astype(int) + 1).tolist()
    for g, a in ((5, 0.9), (7, 0.981), (11, 0.97)):
        tau = P.tau_of_alpha(a, g)
        for mode in (0, 1, 2):
            t_o, st_o, ar_o = P.simulate_rollout(o, lengths, 512, g, tau, 0.05, mode)
            t_c, st_c, ar_c = er.rollout_simulate(c, lengths, 512, g, tau, 0.05, mode)
            assert (st_c, ar_c) == (st_o, ar_o)
            assert t_c == pytest.approx(t_o, rel=1e-12)
    assert er.rollout_simulate(c, [], 0, 5, 3.0, 0.05, 2) == (0.0, 0, 0)
    with pytest.raises(er.ErError):
        er.rollout_simulate(c, lengths, 0, 5, 3.0, 0.05, 3)
