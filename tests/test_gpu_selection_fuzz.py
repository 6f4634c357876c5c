"""-m gpu: randomised rule / compaction parity: many small rollouts with random pool sizes, keep counts, dual-end
long counts, saturation thresholds, modes, length limits and forced-EOS patterns (including truncated rows, groups with fewer than K
valid rows, equal lengths) — lengths, statuses, selected indices, masks and closing steps must equal the oracle's bit for bit."""
import numpy as np
import pytest

from oracle import MODE_AUTO, MODE_DUAL_END, MODE_SHORTEST_EARLY_STOP
from oracle import rollout as ro
from paper_2605_30859_b200 import workloads as wl
from tests.gpu_util import make_ctx

pytestmark = pytest.mark.gpu


BF16 = dict(n_layers=2, d_model=256, n_q_heads=4, n_kv_heads=2, head_dim=128, ffn=512, vocab=1024, n_experts=0, top_k=0, expert_ffn=0,
            qk_norm=False, rope_theta=1.0e6, rms_eps=1.0e-6, dtype="bf16")
BF16_MOE = dict(BF16, ffn=0, n_experts=8, top_k=2, expert_ffn=128)


@pytest.mark.parametrize("seed,kind", [(s, "f32") for s in range(24)] + [(s, "bf16") for s in range(24, 30)] + [(s, "moe") for s in range(30, 34)])
def test_random_policies_match_oracle_bit_exact(seed, kind):
    rng = np.random.default_rng(100 + seed)
    if kind == "f32":
        cfg = dict(wl.CONFIGS["c1"]["model"], vocab=int(rng.choice([64, 512])))   # vocab 64: natural EOS fires now and then
    else:
        cfg = dict(BF16 if kind == "bf16" else BF16_MOE)                          # tensor-core path: stream-K GEMMs, tuned attention
    G = int(rng.integers(1, 6))
    K = int(rng.integers(1, 7))
    Kp = rng.integers(K, min(32, 3 * K) + 1, size=G).astype(np.int32)
    L_long = int(rng.integers(0, K))
    M_up = int(rng.integers(K, 2 * K + 2))
    mode = int(rng.choice([MODE_AUTO, MODE_AUTO, MODE_DUAL_END, MODE_SHORTEST_EARLY_STOP]))
    max_new = int(rng.integers(3, 20))
    P = 12
    prompts = [rng.integers(0, cfg["vocab"] - 1, size=int(rng.integers(1, P + 1))).astype(np.int32) for _ in range(G)]
    forced = np.zeros((G, int(Kp.max())), np.int32)
    for i in range(G):
        pat = rng.integers(0, 4)                              # (not `kind`: that is the test's dtype parameter, used below)
        if pat == 0:      # long tail, some beyond the limit (TRUNC)
            forced[i, :Kp[i]] = np.clip(np.round(rng.lognormal(1.6, 0.9, size=Kp[i])), 1, 4 * max_new)
        elif pat == 1:    # many equal lengths: tie-breaks by sample index
            forced[i, :Kp[i]] = rng.choice([2, 3, max_new], size=Kp[i])
        elif pat == 2:    # nobody is forced: natural EOS or the length limit only
            forced[i, :Kp[i]] = 0
        else:              # fewer than K valid rows
            forced[i, :Kp[i]] = np.where(rng.random(Kp[i]) < 0.3, rng.integers(1, max_new + 1, size=Kp[i]), 10 * max_new)
    d, host = make_ctx(cfg, seed, G, int(Kp.max()), P, max_new, page=8 if kind == "f32" else 64, std=0.3 if kind == "f32" else 0.05)
    d.prefill(prompts, Kp, K, temperature=1.0, seed=seed, forced_len=forced, L_long=L_long, M_up=M_up, mode=mode)
    d.run_to_completion()
    gpu = d.results()
    orc = ro.rollout_stepwise(host, prompts, Kp, K, max_new, 1.0, seed, forced_len=forced, L_long=L_long, M_up=M_up, mode=mode,
                              teacher=gpu["tokens"])
    for key in ("len", "status", "sel", "sel_mask", "close_step"):
        assert np.array_equal(gpu[key], orc[key]), (key, dict(G=G, K=K, Kp=Kp.tolist(), L_long=L_long, M_up=M_up, mode=mode, max_new=max_new))
    cnt = d.counters()
    assert cnt["n_steps"] == orc["n_steps"] and cnt["n_generated_tokens"] == orc["n_generated_tokens"] and cnt["n_kept_tokens"] == orc["n_kept_tokens"]
    for i in range(G):
        assert len(set(gpu["sel"][i].tolist())) == K and gpu["sel"][i].max() < Kp[i]
    d.close()
