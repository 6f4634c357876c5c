"""CPU checks of the PTL(b) tooling: the 3-stage piecewise-linear fit (App. A) and
the rollout time of Eq. 4 against closed forms."""
import numpy as np

from paper_2605_30859_b200.ptl import eq4_rollout_time, fit_piecewise3


def test_fit_recovers_an_exact_three_segment_curve():
    b = np.array([1, 8, 16, 32, 64, 96, 128, 192, 256, 384, 512], float)
    knots, vals = [1, 64, 256, 512], [2.0, 2.5, 6.0, 14.0]
    t = np.interp(b, knots, vals)
    k, v, rmse = fit_piecewise3(b, t)
    assert rmse < 1e-9
    assert k == [1.0, 64.0, 256.0, 512.0]
    assert np.allclose(v, vals)


def test_eq4_constant_ptl_is_the_longest_trajectory():
    # PTL independent of the batch size: T = sum_m (l_(m) - l_(m-1)) * c = c * max length  ("the longest response blocks the batch")
    lens = [5, 17, 3, 9, 17, 40]
    assert eq4_rollout_time(lens, lambda b: 2.0) == 2.0 * 40


def test_eq4_linear_ptl_is_total_tokens():
    # PTL(b) = a*b: T = a * sum_m (l_(m) - l_(m-1)) * (n - m + 1) = a * sum of lengths (every token costs a)
    lens = [5, 17, 3, 9, 17, 40]
    assert abs(eq4_rollout_time(lens, lambda b: 0.5 * b) - 0.5 * sum(lens)) < 1e-12


def test_eq4_matches_a_step_by_step_simulation():
    rng = np.random.default_rng(0)
    lens = rng.integers(1, 50, size=12)
    ptl = lambda b: 1.0 + 0.1 * b + 0.01 * b * b
    T = 0.0
    for step in range(int(lens.max())):
        T += ptl(int((lens > step).sum()))
    assert abs(eq4_rollout_time(lens, ptl) - T) < 1e-9


def test_ctx_slope_recovers_the_second_axis_and_eq6_k_is_its_marginal_cost():
    """step(b, t) = PTL(b) + c_kv b t: the least-squares slope recovers c_kv from a synthetic table, and Eq. 6's k is the
    time one more trajectory costs: mean_len x dPTL/db for the batch it widens + c_kv x mean_len^2 / 2 for its own KV."""
    from paper_2605_30859_b200.ptl import eq6_k, fit_ctx_slope
    ptl = lambda b: 3.0 + 0.01 * b
    pts = [dict(rows=b, ctx=t, ms_median=ptl(b) + 2.5e-5 * b * t) for b in (16, 64, 256) for t in (0, 1024, 4096)]
    c, resid = fit_ctx_slope(pts)
    assert abs(c - 2.5e-5) < 1e-12 and resid < 1e-9
    b = np.array([16.0, 64.0, 256.0])
    k = eq6_k(b, ptl(b), c, mean_len=1000.0, b_at=100.0)
    assert abs(k - (1000.0 * 0.01 + 2.5e-5 * 1000.0 ** 2 / 2)) < 1e-9
    # brute force: total time of n lock-step trajectories of equal length L, one more trajectory added
    L, n = 1000, 100
    T = lambda m: sum(ptl(m) + c * m * s for s in range(L))
    assert abs((T(n + 1) - T(n)) - k) / k < 0.01
