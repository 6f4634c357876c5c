"""Adaptive redundancy allocation (oracle; test infrastructure only).  SURVEY.md 8(f) row f1.

The step immediately upstream of the rollout: it turns the per-prompt length variances a rollout reports into the
per-prompt redundancy M'_i (= Kp[i]) of the next rollout.

  ema_update      smoothed historical variance  sigma~^2_L(q_i)  "maintained via a moving average over preceding
                  epochs", "updated via an Exponential Moving Average" (:415).  The factor is not given
                  numerically: parameter beta, new = (1 - beta) * old + beta * observed; a prompt with no
                  history (old < 0) takes the observed value.
  norm_minmax     Norm(.) = min-max normalisation over the prompt batch.  All-equal input is not
                  covered by the paper (R21): every weight is 1 (uniform need).
  budget          Eq. 8-9:  M* = rho_t / (lambda k),  M_total = clip(floor(M*), M N, 2 M N).
  greedy_allocate Alg. 1: start from M_low, give the remaining budget one unit at a time to the
                  prompt with the largest marginal gain  w_i (1/M'_i - 1/(M'_i + 1))  among those below M_up
                  (R18 for the garbled subscript; ties -> smallest i).
  objective       sum_i w_i / M'_i  (Eq. 5 / Eq. 10).
Pins (tests/test_oracle_allocation.py): the greedy result attains the brute-force minimum of Eq. 5 over ALL feasible
integer allocations (N <= 5) — "the objective function is convex ... can be efficiently solved using a greedy
algorithm"; sum M'_i = M_total and M_low <= M'_i <= M_up always; Eq. 8 is the stationary point of
U(M) = rho ln M - lambda (k M + c); Eq. 9's clip bounds.
"""
import math

import numpy as np


def ema_update(old, observed, beta):
    old, observed = np.asarray(old, dtype=np.float64), np.asarray(observed, dtype=np.float64)
    return np.where(old < 0, observed, (1.0 - beta) * old + beta * observed)


def norm_minmax(x):
    x = np.asarray(x, dtype=np.float64)
    lo, hi = np.min(x), np.max(x)
    if hi == lo:
        return np.ones_like(x)
    return (x - lo) / (hi - lo)


def budget(rho, lam, k, N, M):
    m_star = rho / (lam * k)                                   # Eq. 8
    return int(min(max(math.floor(m_star), M * N), 2 * M * N))  # Eq. 9


def objective(w, alloc):
    return float(np.sum(np.asarray(w, dtype=np.float64) / np.asarray(alloc, dtype=np.float64)))


def greedy_allocate(var_ema, M_total, M_low, M_up):
    """var_ema [N]: smoothed length variances sigma~^2_L(q_i).  Returns M'_i [N] int32."""
    w = norm_minmax(np.sqrt(np.asarray(var_ema, dtype=np.float64)))     # Alg. 1 line 1: w_i = Norm(sigma~_L(q_i))
    N = len(w)
    alloc = np.full(N, M_low, dtype=np.int64)
    remain = int(M_total) - N * M_low                           # line 2
    while remain > 0:                                           # line 3
        best, k = -1.0, -1
        for i in range(N):                                      # line 4: valid candidates only
            if alloc[i] < M_up:
                gain = w[i] * (1.0 / alloc[i] - 1.0 / (alloc[i] + 1))
                if gain > best:                                 # strict: ties -> smallest i
                    best, k = gain, i
        if k < 0:                                               # every prompt saturated: budget cannot be spent
            break
        alloc[k] += 1                                           # line 6
        remain -= 1
    return alloc.astype(np.int32)
