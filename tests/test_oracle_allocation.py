"""Pins of oracle.allocation against what the paper and the mathematics fix."""
import itertools

import numpy as np
import pytest

from oracle import allocation as al


@pytest.mark.parametrize("seed", range(6))
def test_greedy_attains_the_brute_force_minimum_of_eq5(seed):
    rng = np.random.default_rng(seed)
    N = int(rng.integers(2, 6))
    M_low, M_up = 2, 5
    var = rng.uniform(0.0, 100.0, size=N) ** 2
    M_total = int(rng.integers(N * M_low, N * M_up + 1))
    got = al.greedy_allocate(var, M_total, M_low, M_up)
    assert got.sum() == M_total and got.min() >= M_low and got.max() <= M_up
    w = al.norm_minmax(np.sqrt(var))
    best = min(al.objective(w, a) for a in itertools.product(range(M_low, M_up + 1), repeat=N) if sum(a) == M_total)
    assert abs(al.objective(w, got) - best) < 1e-12        # convex => greedy is optimal


def test_budget_is_the_stationary_point_and_is_clipped():
    rho, lam, k, c = 0.9, 0.002, 0.7, 3.0
    m_star = rho / (lam * k)
    U = lambda m: rho * np.log(m) - lam * (k * m + c)        # U = E - lambda T, Eq. 6-7
    assert U(m_star) > U(m_star * 1.01) and U(m_star) > U(m_star * 0.99)
    N, M = 64, 8
    assert al.budget(rho, lam, k, N, M) == int(np.floor(m_star))          # 642 lies inside [512, 1024]
    assert al.budget(rho, lam * 10, k, N, M) == M * N                      # too costly: lower clip
    assert al.budget(rho, lam / 10, k, N, M) == 2 * M * N                  # upper clip


def test_saturation_ties_and_degenerate_inputs():
    # equal variances: uniform weights, ties -> smallest index first, so the extra units go round-robin from prompt 0
    assert al.greedy_allocate([4.0, 4.0, 4.0], 3 * 8 + 4, 8, 16).tolist() == [10, 9, 9]
    # the least-variance prompt has weight 0 and never receives more than M_low while others are below M_up
    a = al.greedy_allocate([1.0, 100.0, 25.0], 3 * 8 + 6, 8, 16)
    assert a[0] == 8 and a.sum() == 30 and a[1] >= a[2]
    # budget larger than N * M_up cannot be spent
    assert al.greedy_allocate([1.0, 2.0], 100, 8, 16).tolist() == [16, 16]


def test_ema():
    out = al.ema_update([-1.0, 10.0], [4.0, 20.0], 0.25)
    assert out.tolist() == [4.0, 12.5]
