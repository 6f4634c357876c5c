"""Pins for oracle.sampling: Gumbel-max == softmax sampling (closed form), greedy limit, ties."""
import numpy as np

from oracle import sampling
from oracle.transformer import softmax


def test_histogram_converges_to_softmax():
    rng = np.random.default_rng(0)
    V, N, T = 12, 30000, 0.7
    z = rng.normal(0, 1.5, V)
    p = softmax(z / T)
    counts = np.zeros(V)
    for n in range(N):                                   # vary prompt / sample / step / seed
        tok, _ = sampling.sample_token(z, T, seed=n // 1000, i=n % 7, j=n % 11, s=n)
        counts[tok] += 1
    chi2 = np.sum((counts - N * p) ** 2 / (N * p))
    assert chi2 < 40.0, chi2                             # 11 dof: P(chi2 > 40) ~ 4e-5
    # a dropped temperature would fail: chi2 against softmax(z) is huge
    q = softmax(z)
    assert np.sum((counts - N * q) ** 2 / (N * q)) > 200.0


def test_temperature_zero_is_argmax_and_low_temperature_limit():
    z = np.array([0.1, 2.0, -1.0, 1.99])
    assert sampling.sample_token(z, 0.0, 1, 0, 0, 0)[0] == 1
    assert abs(sampling.sample_token(z, 0.0, 1, 0, 0, 0)[1] - 0.01) < 1e-12
    for s in range(50):
        assert sampling.sample_token(z * 1000, 1e-3, 1, 0, 0, s)[0] == 1


def test_ties_go_to_lowest_index_and_margin_is_top1_minus_top2():
    z = np.array([1.0, 3.0, 3.0, 2.0])
    tok, margin = sampling.sample_token(z, 0.0, 0, 0, 0, 0)
    assert tok == 1 and margin == 0.0
    y = sampling.perturbed_logits(np.arange(9.0), 1.3, 4, 3, 2, 1)
    tok, margin = sampling.sample_token(np.arange(9.0), 1.3, 4, 3, 2, 1)
    srt = np.sort(y)
    assert y[tok] == srt[-1] and abs(margin - (srt[-1] - srt[-2])) < 1e-15


def test_same_key_same_token_other_key_other_stream():
    z = np.zeros(512)
    a = [sampling.sample_token(z, 1.0, 7, 2, 3, s)[0] for s in range(64)]
    b = [sampling.sample_token(z, 1.0, 7, 2, 3, s)[0] for s in range(64)]
    c = [sampling.sample_token(z, 1.0, 7, 2, 4, s)[0] for s in range(64)]
    assert a == b and a != c
    assert len(set(a)) > 32                              # uniform logits: tokens spread out


def test_token_logprob_against_the_library_closed_forms_and_invariants():
    """SURVEY.md 8(a) row 7 (optional log-prob): log softmax(z/T)[v]."""
    from scipy.special import log_softmax
    rng = np.random.default_rng(5)
    for V, T in ((7, 1.0), (513, 0.7), (4096, 1.3)):
        z = rng.standard_normal(V) * 4
        ref = log_softmax(z / T)
        lp = np.array([sampling.token_logprob(z, T, v) for v in range(V)])
        assert np.allclose(lp, ref, atol=1e-12)
        assert abs(np.exp(lp).sum() - 1.0) < 1e-12                       # a distribution
        assert abs(sampling.token_logprob(z + 123.0, T, 3) - lp[3]) < 1e-9   # shift invariance
        assert np.argmax(lp) == np.argmax(z)
    assert abs(sampling.token_logprob(np.full(100, 2.5), 0.3, 17) + np.log(100)) < 1e-12          # uniform: -ln V
    a, b, T = 1.7, -0.4, 0.5
    assert abs(sampling.token_logprob(np.array([a, b]), T, 0) + np.log1p(np.exp(-(a - b) / T))) < 1e-12   # log-sigmoid
    assert sampling.token_logprob(np.array([a, b]), 0, 0) == sampling.token_logprob(np.array([a, b]), 1.0, 0)  # T=0: temperature 1
    big = np.array([1000.0, 0.0, -1000.0])                                # no overflow; the dominated tokens get the gap
    assert abs(sampling.token_logprob(big, 1.0, 0)) < 1e-12 and abs(sampling.token_logprob(big, 1.0, 2) + 2000.0) < 1e-9


def test_rollout_reports_the_logprob_of_every_drawn_token():
    from oracle import rollout as orl
    from paper_2605_30859_b200 import workloads as wl
    cfg = dict(wl.CONFIGS["c1"]["model"])
    model = wl.host_model(wl.make_model(cfg, seed=3))
    prompts = wl.make_prompts(2, 8, cfg["vocab"], 3)
    out = orl.rollout_stepwise(model, list(prompts), np.array([3, 3]), 2, 6, 0.8, 11, forced_len=None, keep_logits=True)
    for (r, s), z in out["logits"].items():
        v = out["oracle_tokens"][r, s]
        assert abs(out["logprobs"][r, s] - sampling.token_logprob(z, 0.8, v)) < 1e-12
        assert out["logprobs"][r, s] <= 0.0
    assert np.isnan(out["logprobs"][out["tokens"] < 0]).all()          # nothing beyond a row's length
