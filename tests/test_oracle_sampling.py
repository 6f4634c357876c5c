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
