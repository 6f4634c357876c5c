"""The library's host-side redundancy allocation (include/darts.h) against oracle.allocation:
integer plans bit-exact, on random batches and the edge cases (runs on CPU: these entry points do no GPU work)."""
import numpy as np
import pytest

from oracle import allocation as al


@pytest.mark.parametrize("seed", range(8))
def test_plan_matches_oracle_bit_exact(seed):
    from paper_2605_30859_b200 import api
    rng = np.random.default_rng(seed)
    G, K = int(rng.integers(1, 65)), 8
    var = (rng.lognormal(6.0, 1.0, size=G) ** 2).astype(np.float32)
    if seed == 0:
        var[:] = var[0]                                   # all equal: uniform weights
    M_total = int(rng.integers(G * K, 2 * G * K + 1))
    got = api.allocate_redundancy(var, M_total, K, 2 * K)
    ref = al.greedy_allocate(var.astype(np.float64), M_total, K, 2 * K)
    assert np.array_equal(got, ref)
    assert got.sum() == M_total and got.min() >= K and got.max() <= 2 * K


def test_budget_and_ema_match_oracle_and_reject_bad_arguments():
    from paper_2605_30859_b200 import api
    for rho, lam, k in [(0.9, 0.002, 0.7), (0.1, 0.5, 2.0), (3.0, 1e-5, 1.0), (0.75, 0.001, 1.0)]:
        assert api.redundancy_budget(rho, lam, k, 64, 8) == al.budget(rho, lam, k, 64, 8)
    ema = np.array([-1.0, 10.0, 0.0], np.float32)
    api.update_variance_ema(ema, np.array([4.0, 20.0, 8.0], np.float32), 0.25)
    assert np.allclose(ema, al.ema_update([-1.0, 10.0, 0.0], [4.0, 20.0, 8.0], 0.25))
    with pytest.raises(api.DartsError):
        api.allocate_redundancy(np.array([1.0, -2.0], np.float32), 16, 8, 16)
    with pytest.raises(api.DartsError):
        api.allocate_redundancy(np.array([1.0, 2.0], np.float32), 15, 8, 16)     # budget below G * M_low
    with pytest.raises(api.DartsError):
        api.redundancy_budget(1.0, 0.0, 1.0, 4, 8)
