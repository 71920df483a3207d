"""GPU parity: er_spec_verify vs the oracle (V1-V12): accept counts and accepted-prefix tokens
exact, -1 padding exact, final token by rule V10 (exact, or inside its own fp64 CDF interval +-1e-5)."""
import numpy as np
import pytest
import torch

from oracle import er_oracle as O
from paper_2606_18967_b200 import er, inputs as I

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _run_and_check(tgt, drf, toks, ua, us, logits, dtype, temperature=1.0, min_margin=1e-5):
    """tgt/drf: float32 numpy (probs or logits).  dtype: torch dtype sent to the device."""
    t_dev = torch.from_numpy(tgt).to(DEV).to(dtype).contiguous()
    d_dev = torch.from_numpy(drf).to(DEV).to(dtype).contiguous()
    # the oracle sees exactly the values the device sees
    t_host = t_dev.float().cpu().numpy()
    d_host = d_dev.float().cpu().numpy()
    acc, out = er.spec_verify(t_dev, d_dev, torch.from_numpy(toks).to(DEV), torch.from_numpy(ua).to(DEV),
                              torch.from_numpy(us).to(DEV), logits, temperature)
    torch.cuda.synchronize()
    acc, out = acc.cpu().numpy(), out.cpu().numpy()
    acc_ref, out_ref, diag = O.spec_verify(t_host, d_host, toks, ua, us, inputs_are_logits=logits,
                                           temperature=temperature, return_diag=True)
    B, G1 = out.shape
    thin = [m for d in diag for m in d["margins"] if m < min_margin]
    assert not thin, f"accept tests with margin < {min_margin}: {thin} (listed, never re-seeded)"
    assert np.array_equal(acc, acc_ref)
    n_exact = 0
    for b in range(B):
        n = int(acc_ref[b])
        assert np.array_equal(out[b, :n], out_ref[b, :n])
        assert np.all(out[b, n + 1:] == -1)
        if out[b, n] == out_ref[b, n]:
            n_exact += 1
        else:
            assert O.token_in_widened_interval(diag[b], int(out[b, n])), (b, out[b, n], out_ref[b, n])
    return acc, out, n_exact


def _softmax(x):
    return O.softmax64(x).astype(np.float32)


def test_config0_probs_fp32():
    B, gamma, V = 4, 4, 32000
    lt, ld = I.verify_logits_f32(B, gamma, V, I.seed_of("cfg0", "verify"))
    p, q = _softmax(lt), _softmax(ld)
    toks = I.sample_draft_tokens(q, I.seed_of("cfg0", "x"))
    ua = I.uniforms((B, gamma), I.seed_of("cfg0", "ua"))
    us = I.uniforms((B,), I.seed_of("cfg0", "us"))
    _run_and_check(p, q, toks, ua, us, False, torch.float32)


def test_q_equals_p_accepts_everything():
    B, gamma, V = 3, 5, 5000
    lt, _ = I.verify_logits_f32(B, gamma, V, 11)
    p = _softmax(lt)
    q = p[:, :gamma].copy()
    toks = I.sample_draft_tokens(q, 12)
    ua = I.uniforms((B, gamma), 13)
    us = I.uniforms((B,), 14)
    acc, out, _ = _run_and_check(p, q, toks, ua, us, False, torch.float32, min_margin=0.0)
    assert np.all(acc == gamma) and np.all(out[:, gamma] >= 0)


@pytest.mark.parametrize("V", [1, 7, 255, 8192, 8193, 8200, 20011, 20012])
def test_ragged_vocab_sizes_logits_f32(V):
    B, gamma = 5, 3
    lt, ld = I.verify_logits_f32(B, gamma, V, I.seed_of("ragged", V), draft_noise=0.5)
    toks = I.sample_draft_tokens(_softmax(ld), V + 1)
    ua = I.uniforms((B, gamma), V + 2)
    us = I.uniforms((B,), V + 3)
    _run_and_check(lt, ld, toks, ua, us, True, torch.float32)


def test_forced_rejection_and_zero_probability():
    # p(x_1) = 0 -> rejected at once and the resampled token differs from x_1; one-hot p on x -> accepted
    B, gamma, V = 2, 2, 64
    p = np.full((B, gamma + 1, V), 1.0 / (V - 1), dtype=np.float32)
    q = np.full((B, gamma, V), 1.0 / V, dtype=np.float32)
    toks = np.array([[3, 4], [5, 6]], dtype=np.int32)
    p[0, 0, 3] = 0.0
    p[1, :, :] = 0.0
    p[1, 0, 5] = 1.0
    p[1, 1, 6] = 1.0
    p[1, 2, 9] = 1.0
    ua = np.full((B, gamma), 0.999, dtype=np.float32)
    us = np.array([0.5, 0.5], dtype=np.float32)
    acc, out, _ = _run_and_check(p, q, toks, ua, us, False, torch.float32, min_margin=0.0)
    assert acc[0] == 0 and out[0, 0] != 3
    assert acc[1] == 2 and out[1, 2] == 9


@pytest.mark.parametrize("gamma", [2, 4, 8])
def test_config4_bf16_logits(gamma):
    B, V = 8, 152064          # config 4 shape at a batch the oracle finishes in seconds
    lt, ld = I.verify_logits_f32(B, gamma, V, I.seed_of("cfg4", gamma), draft_noise=0.5)
    t_b = torch.from_numpy(lt).to(torch.bfloat16).float().numpy()
    d_b = torch.from_numpy(ld).to(torch.bfloat16).float().numpy()
    toks = I.sample_draft_tokens(_softmax(d_b), I.seed_of("cfg4", "x", gamma))
    ua = I.uniforms((B, gamma), I.seed_of("cfg4", "ua", gamma))
    us = I.uniforms((B,), I.seed_of("cfg4", "us", gamma))
    acc, out, n_exact = _run_and_check(t_b, d_b, toks, ua, us, True, torch.bfloat16)
    assert n_exact >= B // 2   # most tokens are exactly the oracle's; the rest passed the V10 window


def _device_workload(B, gamma, V, tag):
    """Config-4 verify inputs generated on the device (the numpy generators need minutes at B = 64-256); both sides
    see the same bf16 bytes."""
    tgt, drf = I.verify_logits_bf16_device(B, gamma, V, I.seed_of(tag, "logits", B, gamma), DEV)
    toks = I.sample_draft_tokens_gumbel(drf, I.seed_of(tag, "tok", B, gamma))
    ua = I.uniforms((B, gamma), I.seed_of(tag, "ua", B, gamma))
    us = I.uniforms((B,), I.seed_of(tag, "us", B, gamma))
    return tgt, drf, toks, ua, us


def _check_against_oracle(tgt, drf, toks, ua, us, acc, out, rows=None):
    """acc / out from the device for ALL sequences; the oracle on `rows` (default all)."""
    B, G1, V = tgt.shape
    rows = list(range(B)) if rows is None else rows
    acc, out = acc.cpu().numpy(), out.cpu().numpy()
    toks_h = toks.cpu().numpy()
    n_exact = 0
    for b in rows:
        a_ref, o_ref, diag = O.spec_verify(tgt[b:b + 1].float().cpu().numpy(), drf[b:b + 1].float().cpu().numpy(),
                                           toks_h[b:b + 1], ua[b:b + 1], us[b:b + 1], inputs_are_logits=True,
                                           return_diag=True)
        thin = [m for m in diag[0]["margins"] if m < 1e-5]
        assert not thin, f"sequence {b}: accept test with margin < 1e-5 (listed, never re-seeded): {thin}"
        n = int(a_ref[0])
        assert acc[b] == n, (b, acc[b], n)
        assert np.array_equal(out[b, :n], o_ref[0, :n]) and np.all(out[b, n + 1:] == -1)
        if out[b, n] == o_ref[0, n]:
            n_exact += 1
        else:
            assert O.token_in_widened_interval(diag[0], int(out[b, n])), (b, out[b, n], o_ref[0, n])
    return n_exact


@pytest.mark.parametrize("gamma", [2, 4, 8])
def test_config4_full_batch_64(gamma):
    # BASELINE.json configs[4] as stated: batch 64, vocab 152064, bf16 logits, draft = target + N(0, 0.5^2)
    B, V = 64, 152064
    tgt, drf, toks, ua, us = _device_workload(B, gamma, V, "cfg4full")
    acc, out = er.spec_verify(tgt, drf, toks, torch.from_numpy(ua).to(DEV), torch.from_numpy(us).to(DEV), True)
    torch.cuda.synchronize()
    n_exact = _check_against_oracle(tgt, drf, toks, ua, us, acc, out)
    assert n_exact >= B // 2
    # statistical sanity of the workload: mean(n) + 1 ~ tau(alpha ~ 0.80, gamma)
    a = acc.float()
    assert abs(float(a.mean()) + 1 - O.block_efficiency(0.80, gamma)) < 3.5 * float(a.std()) / np.sqrt(B) + 0.15


def test_config2_maximum_batch_256_gamma_8():
    # config 2's largest verify (B = M = 256, gamma = 8): 1024 CTAs in clusters of 4, seven residency waves; every
    # sequence's structural properties + the oracle on a seeded quarter of the sequences
    B, gamma, V = 256, 8, 152064
    tgt, drf, toks, ua, us = _device_workload(B, gamma, V, "cfg2max")
    acc, out = er.spec_verify(tgt, drf, toks, torch.from_numpy(ua).to(DEV), torch.from_numpy(us).to(DEV), True)
    torch.cuda.synchronize()
    a, o, t = acc.cpu().numpy(), out.cpu().numpy(), toks.cpu().numpy()
    for b in range(B):
        n = int(a[b])
        assert 0 <= n <= gamma and np.array_equal(o[b, :n], t[b, :n]) and 0 <= o[b, n] < V and np.all(o[b, n + 1:] == -1)
    rows = sorted(np.random.default_rng(2).choice(B, size=64, replace=False).tolist())
    _check_against_oracle(tgt, drf, toks, ua, us, acc, out, rows=rows)


@pytest.mark.parametrize("dtype", [torch.float32, torch.bfloat16])
@pytest.mark.parametrize("V", [20011, 20012, 20016, 5001])
def test_masked_logits_minus_infinity(V, dtype):
    # logits after top-k style masking: everything outside the top 50 of the TARGET row is -inf in both rows (also whole
    # 8-element chunks, whole segments and the ragged tail chunk, whose positions beyond V are filled by the kernel);
    # the kernel must not produce NaN / inf statistics (a finite fill value once became a lane's softmax
    # reference there).  V = 20011 / 5001: scalar loads; 20012: fp32 rows through the ring with a clipped tail; 20016:
    # both dtypes through the ring
    B, gamma = 6, 3
    lt, ld = I.verify_logits_f32(B, gamma, V, 4242, draft_noise=0.5)
    for b in range(B):
        for i in range(gamma + 1):
            keep = np.argsort(lt[b, i])[-50:]
            m = np.ones(V, bool)
            m[keep] = False
            lt[b, i, m] = -np.inf
            if i < gamma:
                ld[b, i, m] = -np.inf
    lt = torch.from_numpy(lt).to(dtype).float().numpy()
    ld = torch.from_numpy(ld).to(dtype).float().numpy()
    toks = I.sample_draft_tokens(_softmax(ld), 4243)
    for T in (1.0, 0.6):
        acc, out, _ = _run_and_check(lt, ld, toks, I.uniforms((B, gamma), 4244), I.uniforms((B,), 4245), True, dtype,
                                     temperature=T)
        assert np.all(out[np.arange(B), acc] >= 0)
        for b in range(B):
            assert np.isfinite(lt[b, acc[b], out[b, acc[b]]])        # the drawn token is never a masked one


def test_temperature():
    B, gamma, V = 4, 3, 4096
    lt, ld = I.verify_logits_f32(B, gamma, V, 77, draft_noise=0.5)
    toks = I.sample_draft_tokens(O.softmax64(ld, 0.6).astype(np.float32), 78)
    _run_and_check(lt, ld, toks, I.uniforms((B, gamma), 79), I.uniforms((B,), 80), True, torch.float32, temperature=0.6)


def test_deterministic():
    B, gamma, V = 4, 4, 32000
    lt, ld = I.verify_logits_f32(B, gamma, V, 5, draft_noise=0.5)
    t = torch.from_numpy(lt).to(DEV).to(torch.bfloat16)
    d = torch.from_numpy(ld).to(DEV).to(torch.bfloat16)
    toks = torch.from_numpy(I.sample_draft_tokens(_softmax(ld), 6)).to(DEV)
    ua = torch.from_numpy(I.uniforms((B, gamma), 7)).to(DEV)
    us = torch.from_numpy(I.uniforms((B,), 8)).to(DEV)
    a1, o1 = er.spec_verify(t, d, toks, ua, us, True)
    a2, o2 = er.spec_verify(t, d, toks, ua, us, True)
    assert torch.equal(a1, a2) and torch.equal(o1, o2)


def test_max_gamma_and_high_acceptance():
    # gamma = 16 (the maximum), draft close to target: most tokens are accepted, several sequences reach the bonus
    # position (the paper's regime); vocabulary not a multiple of the tile
    B, gamma, V = 3, 16, 50001
    lt, ld = I.verify_logits_f32(B, gamma, V, 901, draft_noise=0.05)
    toks = I.sample_draft_tokens(_softmax(ld), 902)
    acc, out, _ = _run_and_check(lt, ld, toks, I.uniforms((B, gamma), 903), I.uniforms((B,), 904), True, torch.float32)
    assert acc.max() >= gamma // 2


@pytest.mark.parametrize("ring", [16, 17])
@pytest.mark.parametrize("cluster", [1, 2, 4, 8])
def test_every_cluster_size_gives_the_same_tokens(cluster, ring):
    # the per-sequence work may be split over 1-8 CTAs, and the rows may come through the shared-memory ring (16)
    # or through registers (17); decisions and accepted prefixes must not depend on either (the drawn token may
    # differ only inside the V10 window, which _run_and_check enforces)
    B, gamma, V = 6, 4, 152064
    lt, ld = I.verify_logits_f32(B, gamma, V, 911, draft_noise=0.5)
    toks = I.sample_draft_tokens(_softmax(ld), 912)
    ua, us = I.uniforms((B, gamma), 913), I.uniforms((B,), 914)
    with er.dev_library() as lib:
        assert lib.er_dev_verify_cluster(cluster) == 0 and lib.er_dev_verify_cluster(ring) == 0
        _run_and_check(lt, ld, toks, ua, us, True, torch.float32)


@pytest.mark.parametrize("V", [8, 264, 50001, 50008, 65536])
@pytest.mark.parametrize("ring", [16, 17])
def test_ragged_vocab_sizes_logits_bf16(V, ring):
    # bf16 rows that are 16-byte multiples take the ring kernel (unless 17 forces the register path), the others
    # (V = 50001) the register-path kernel with scalar loads
    B, gamma = 5, 3
    lt, ld = I.verify_logits_f32(B, gamma, V, I.seed_of("ragged16", V), draft_noise=0.5)
    t_b = torch.from_numpy(lt).to(torch.bfloat16).float().numpy()
    d_b = torch.from_numpy(ld).to(torch.bfloat16).float().numpy()
    toks = I.sample_draft_tokens(_softmax(d_b), V + 1)
    ua, us = I.uniforms((B, gamma), V + 2), I.uniforms((B,), V + 3)
    with er.dev_library() as lib:
        assert lib.er_dev_verify_cluster(ring) == 0
        _run_and_check(t_b, d_b, toks, ua, us, True, torch.bfloat16)


@pytest.mark.parametrize("cluster", [0, 1])
def test_maximum_vocabulary(cluster):
    # V = 2^20, the largest the call accepts: 4096 segments; with one CTA per sequence (cluster 1) the segment-sum
    # array and the fp64 blocked prefix are at their largest
    B, gamma, V = 2, 2, 1 << 20
    lt, ld = I.verify_logits_f32(B, gamma, V, 31337, draft_noise=0.5)
    t_b = torch.from_numpy(lt).to(torch.bfloat16).float().numpy()
    d_b = torch.from_numpy(ld).to(torch.bfloat16).float().numpy()
    toks = I.sample_draft_tokens(_softmax(d_b), 31338)
    ua, us = I.uniforms((B, gamma), 31339), I.uniforms((B,), 31340)
    with er.dev_library() as lib:
        assert lib.er_dev_verify_cluster(cluster) == 0
        _run_and_check(t_b, d_b, toks, ua, us, True, torch.bfloat16)
    lib = er.load()
    z = torch.zeros(16, device=DEV)
    assert lib.er_spec_verify(z.data_ptr(), z.data_ptr(), 0, 1, 1.0, z.data_ptr(), z.data_ptr(), z.data_ptr(), 1, 2,
                              (1 << 20) + 8, z.data_ptr(), z.data_ptr(), None) == 2       # ER_ERR_SHAPE


@pytest.mark.parametrize("dtype", [torch.float32, torch.bfloat16])
@pytest.mark.parametrize("ring", [16, 17])
def test_rising_logits_raise_the_softmax_reference_many_times(dtype, ring):
    # logits that climb along the vocabulary by far more than the 32-bit margin of the lazily raised reference (range
    # 600 / T = 0.5 -> ~1700 binades): every lane has to re-reference its sums again and again, in both kernels; the
    # statistics must still match the fp64 oracle (accept counts exact, token by rule V10)
    B, gamma, V = 4, 3, 40000
    rng = np.random.default_rng(99)
    ramp = np.linspace(-300.0, 300.0, V, dtype=np.float32)
    lt = (ramp[None, None, :] + rng.standard_normal((B, gamma + 1, V)).astype(np.float32)).astype(np.float32)
    ld = (lt[:, :gamma] + 0.3 * rng.standard_normal((B, gamma, V)).astype(np.float32)).astype(np.float32)
    lt[1], ld[1] = lt[1, :, ::-1].copy(), ld[1, :, ::-1].copy()          # one sequence falls instead of climbing
    t_h = torch.from_numpy(lt).to(dtype).float().numpy()
    d_h = torch.from_numpy(ld).to(dtype).float().numpy()
    toks = I.sample_draft_tokens(O.softmax64(d_h, 0.5).astype(np.float32), 100)
    ua, us = I.uniforms((B, gamma), 101), I.uniforms((B,), 102)
    with er.dev_library() as lib:
        assert lib.er_dev_verify_cluster(ring) == 0
        _run_and_check(t_h, d_h, toks, ua, us, True, dtype, temperature=0.5)
