"""Temperature + Gumbel-max sampling (oracle; test infrastructure only).

north_star: "a fused logits kernel applies temperature and Gumbel-max sampling
from counter-based Philox keyed on (seed, prompt, sample, step)".  The paper
only requires that the M'_i trajectories of a prompt be independent samples
(§4.1.1); temperature is never stated (R14: API parameter).

    y_v   = z_v / T + g_v          g_v from oracle.philox.gumbel_noise(V, seed, i, j, s)
    token = argmax_v y_v           ties -> lowest v
    margin = y_(1) - y_(2)         (top-1 minus top-2; the near-tie measure)
    T == 0  ->  y = z (greedy)
    logprob = log softmax(z / T)[token]   (T == 0: log softmax(z)[token]) — SURVEY.md 8(a) row 7 "optionally log-prob":
              the sampling policy's log-probability of the token it drew, written out as its definition

argmax_v (z_v/T + g_v) with i.i.d. standard Gumbel g is an exact sample from
softmax(z/T) (the Gumbel-max trick) — that closed form is the pin
(tests/test_oracle_sampling.py, chi-square against softmax).  token_logprob is pinned there against
scipy.special.log_softmax, the closed forms (uniform logits: -ln V; two logits: log-sigmoid of their difference / T),
normalisation (sum_v exp = 1) and shift invariance.
"""
import numpy as np

from .philox import gumbel_noise


def perturbed_logits(z, T, seed, i, j, s):
    z = np.asarray(z, dtype=np.float64)
    if T == 0:
        return z.copy()
    return z / T + gumbel_noise(z.shape[0], seed, i, j, s)


def top2(y):
    """(argmax with lowest-index tie-break, top-1 value, top-2 value)."""
    v1 = int(np.argmax(y))                 # numpy returns the first maximal index
    y1 = y[v1]
    if y.shape[0] == 1:
        return v1, y1, -np.inf
    rest = np.delete(y, v1)
    return v1, y1, np.max(rest)


def sample_token(z, T, seed, i, j, s):
    """Returns (token, margin)."""
    y = perturbed_logits(z, T, seed, i, j, s)
    v1, y1, y2 = top2(y)
    return v1, float(y1 - y2)


def token_logprob(z, T, v):
    """log softmax(z / T)[v] in fp64 (T == 0: temperature 1), by the definition with the maximum subtracted."""
    zt = np.asarray(z, dtype=np.float64)
    if T != 0:
        zt = zt / T
    m = np.max(zt)
    return float(zt[v] - (m + np.log(np.sum(np.exp(zt - m)))))
