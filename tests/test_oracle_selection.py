"""Pins for oracle.selection: exhaustive enumeration of tiny pools against an independent
brute-force statement of the rule (subset search with pairwise precedence, no sorting)."""
import itertools

import numpy as np

from oracle import ACTIVE, VALID, TRUNC, PRUNED, MODE_AUTO, MODE_DUAL_END, MODE_SHORTEST_EARLY_STOP
from oracle import selection as sel

CLS = {VALID: 0, TRUNC: 1, PRUNED: 2}


def brute_first_k(items, K, before):
    """The unique K-subset whose members all precede every non-member (strict total order)."""
    hits = []
    for sub in itertools.combinations(items, K):
        rest = [x for x in items if x not in sub]
        if all(before(a, b) for a in sub for b in rest):
            hits.append(set(sub))
    assert len(hits) == 1
    return hits[0]


def brute_early(lens, status, K):
    def before(a, b):
        if CLS[status[a]] != CLS[status[b]]:
            return CLS[status[a]] < CLS[status[b]]
        if lens[a] != lens[b]:
            return lens[a] < lens[b]
        return a < b
    return brute_first_k(list(range(len(lens))), K, before)


def brute_dual(lens, status, K, L):
    n = len(lens)
    asc = lambda a, b: (lens[a] < lens[b]) or (lens[a] == lens[b] and a < b)
    short = brute_first_k(list(range(n)), K - L, asc) if K - L > 0 else set()
    rest = [j for j in range(n) if j not in short]
    valid = [j for j in rest if status[j] == VALID]
    desc = lambda a, b: (lens[a] > lens[b]) or (lens[a] == lens[b] and a < b)
    take = min(L, len(valid))
    longest = brute_first_k(valid, take, desc) if take > 0 else set()
    others = [j for j in rest if j not in longest]
    fill = brute_first_k(others, L - take, asc) if L - take > 0 else set()
    return short, longest | fill


def test_select_early_exhaustive():
    n_cases = 0
    for n in range(1, 6):
        for lens in itertools.product(range(1, 4), repeat=n):
            for status in itertools.product((VALID, TRUNC, PRUNED), repeat=n):
                for K in range(1, n + 1):
                    got = sel.select_early(lens, status, K)
                    assert len(got) == K and len(set(got)) == K
                    assert set(got) == brute_early(lens, status, K)
                    keys = [(CLS[status[j]], lens[j], j) for j in got]
                    assert keys == sorted(keys)                       # emitted in rule order
                    n_cases += 1
    assert n_cases > 50000


def test_select_dual_exhaustive():
    for n in range(1, 6):
        for lens in itertools.product(range(1, 4), repeat=n):
            for status in itertools.product((VALID, TRUNC), repeat=n):
                for K in range(1, n + 1):
                    for L in range(0, K):
                        got = sel.select_dual(lens, status, K, L)
                        assert len(got) == K and len(set(got)) == K and all(0 <= j < n for j in got)
                        short, longs = brute_dual(lens, status, K, L)
                        assert set(got[: K - L]) == short and set(got[K - L:]) == longs
                        for part in (got[: K - L], got[K - L:]):
                            keys = [(lens[j], j) for j in part]
                            assert keys == sorted(keys)


def test_dual_special_cases():
    lens, st = [5, 3, 9, 3, 7, 9], [VALID] * 6
    assert sel.select_dual(lens, st, 6, 1) == [1, 3, 0, 4, 2, 5]            # K' = K: everything
    assert sel.select_dual(lens, st, 3, 0) == sel.select_early(lens, st, 3)  # L_long = 0: shortest only
    assert sel.select_dual(lens, st, 4, 1) == [1, 3, 0, 2]                  # longest: tie 9,9 -> j=2
    st2 = [VALID, VALID, TRUNC, VALID, VALID, TRUNC]                          # limit-hitting rows excluded (:140)
    assert sel.select_dual(lens, st2, 4, 1) == [1, 3, 0, 4]
    # no VALID left for the long end: filled in ascending order (R8)
    assert sel.select_dual([2, 9, 9], [VALID, TRUNC, TRUNC], 2, 1) == [0, 1]


def test_apply_stop_rule_order():
    eos, mx = 99, 8
    assert sel.apply_stop(5, 3, 3, eos, mx) == (eos, VALID)                 # forced EOS overwrites the token
    assert sel.apply_stop(eos, 2, 5, eos, mx) == (eos, VALID)               # natural EOS
    assert sel.apply_stop(5, 8, None, eos, mx) == (5, TRUNC)                # length limit
    assert sel.apply_stop(eos, 8, None, eos, mx) == (eos, VALID)            # EOS exactly at the limit is VALID (R9)
    assert sel.apply_stop(5, 8, 8, eos, mx) == (eos, VALID)                 # forced_len == max_new is VALID (R11)
    assert sel.apply_stop(5, 7, 9, eos, mx) == (5, ACTIVE)
    assert sel.apply_stop(5, 3, None, -1, mx) == (5, ACTIVE)                # eos_id < 0: natural EOS off


def test_group_mode_threshold():
    assert sel.group_mode(16, 8, 16, MODE_AUTO) == "EARLY"                  # M'_i >= M_up (:432)
    assert sel.group_mode(15, 8, 16, MODE_AUTO) == "DUAL"
    assert sel.group_mode(8, 8, 16, MODE_SHORTEST_EARLY_STOP) == "EARLY"
    assert sel.group_mode(16, 8, 16, MODE_DUAL_END) == "DUAL"


def lockstep(nat_len, nat_status, K, L, M_up, mode):
    """Lock-step simulation on lengths alone: row j ends at step nat_len[j] with nat_status[j]."""
    n = len(nat_len)
    lens, status = np.zeros(n, dtype=np.int32), np.full(n, ACTIVE, dtype=np.uint8)
    t = 0
    while True:
        t += 1
        for j in range(n):
            if status[j] == ACTIVE:
                lens[j] = t
                if nat_len[j] == t:
                    status[j] = nat_status[j]
        got = sel.group_rule(lens, status, n, K, L, M_up, mode)
        if got is not None:
            return got, lens.copy(), status.copy(), t


def test_early_stop_equals_full_rollout_then_sort_exhaustive():
    """EARLY result == K smallest (len, j) among VALID of the fully rolled-out pool (SURVEY §8(c) ii)."""
    mx = 4
    for n in range(2, 6):
        for nat in itertools.product(range(1, mx + 1), repeat=n):
            for trunc_bits in range(1 << n):
                st = [TRUNC if (nat[j] == mx and trunc_bits >> j & 1) else VALID for j in range(n)]
                if any((trunc_bits >> j & 1) and nat[j] != mx for j in range(n)):
                    continue
                for K in range(1, n + 1):
                    got, lens, status, t = lockstep(nat, st, K, 1, 0, MODE_SHORTEST_EARLY_STOP)
                    valid = sorted((nat[j], j) for j in range(n) if st[j] == VALID)
                    if len(valid) >= K:
                        assert got == [j for _, j in valid[:K]]
                        assert t == valid[K - 1][0]                              # closes when the K-th valid ends
                        for j in range(n):
                            if nat[j] > t:
                                assert status[j] == PRUNED and lens[j] == t
                            else:
                                assert status[j] == st[j] and lens[j] == nat[j]
                    else:
                        trunc = sorted((nat[j], j) for j in range(n) if st[j] == TRUNC)
                        assert got == [j for _, j in (valid + trunc)[:K]]
                        assert not np.any(status == PRUNED)
                    # DUAL never prunes and waits for the whole pool (:224)
                    got_d, lens_d, status_d, t_d = lockstep(nat, st, K, min(1, K - 1), 10 ** 9, MODE_AUTO)
                    assert t_d == max(nat) and list(lens_d) == list(nat) and not np.any(status_d == PRUNED)
                    assert got_d == sel.select_dual(nat, st, K, min(1, K - 1))


def test_compact_is_stable_partition_and_mask():
    rows = [4, 7, 1, 9, 3]
    status = {4: ACTIVE, 7: VALID, 1: ACTIVE, 9: PRUNED, 3: ACTIVE}
    assert sel.compact(rows, status) == [4, 1, 3]
    assert sel.sel_mask([0, 3, 15]) == (1 | 8 | 1 << 15)


def test_length_stats_closed_form():
    m, v = sel.length_stats([2, 4, 4, 4, 5, 5, 7, 9])
    assert m == 5.0 and v == 4.0
