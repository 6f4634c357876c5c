"""CPU checks of bench.py's algorithmic-byte counters (the numerators of the roofline fractions) against hand-computed cases."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def test_attention_bytes_prefix_once_per_open_group():
    # 2 groups x 2 rows, P = 10, kvB = 1; lengths: group 0 -> (3, 1), group 1 -> (2, 2)
    total, per_step = bench.rollout_algo_attention_bytes([3, 1, 2, 2], np.array([2, 2]), 10, 1)
    # decode step s feeds token s-1 of every row with len > s: its suffix holds s tokens
    # s=1: rows 0, 2, 3 active (3 rows x 1 token) + 2 open groups x 10;  s=2: row 0 only (2 tokens) + 1 group x 10
    assert per_step == [3 * 1 + 2 * 10, 1 * 2 + 1 * 10]
    assert total == sum(per_step)


def test_step_bytes_dense_closed_form():
    cfg = dict(n_layers=2, d_model=8, head_dim=4, n_q_heads=2, n_kv_heads=1, vocab=16, ffn=12, n_experts=0, top_k=0, expert_ffn=0)
    attn_w = (2 + 2) * 4 * 8 + 2 * 4 * 8
    params = 2 * (attn_w + 3 * 8 * 12) + 16 * 8
    kvb = 2 * 1 * 4 * 2 * 2                                  # K+V x Hkv x hd x bf16 x layers
    got = bench.rollout_algo_step_bytes(cfg, [3, 1], np.array([2]), 5)
    # s=1: 1 row active (len 3 > 1): weights + (1 row x 1 token + 1 group x 5 + 1 append) x kvb;  s=2: (1 x 2 + 5 + 1) x kvb
    want = (params * 2 + (1 + 5 + 1) * kvb) + (params * 2 + (2 + 5 + 1) * kvb)
    assert got == want


def test_step_bytes_moe_counts_expected_distinct_experts():
    cfg = dict(n_layers=1, d_model=4, head_dim=4, n_q_heads=1, n_kv_heads=1, vocab=8, ffn=0, n_experts=4, top_k=2, expert_ffn=4)
    got = bench.rollout_algo_step_bytes(cfg, [2], np.array([1]), 3)
    attn_w = 3 * 4 * 4 + 4 * 4
    fixed = (attn_w + 4 * 4 * 2) + 8 * 4                     # attention + router (counted as E x d x 2 elements of bf16-equivalents) + LM head
    experts = 4 * (1 - (1 - 2 / 4) ** 1) * (3 * 4 * 4)       # one active row: E (1 - (1 - k/E)^1) = k distinct experts
    kvb = 2 * 1 * 4 * 2
    assert abs(got - ((fixed + experts) * 2 + (1 + 3 + 1) * kvb)) < 1e-9
