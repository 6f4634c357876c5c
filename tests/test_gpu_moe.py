"""-m gpu parity of the mixture-of-experts path (router, top-k, expert MLPs, gated combine) against the oracle:
fp32 through the generic kernels (1e-4), bf16 through the grouped tcgen05 GEMMs (2e-2), teacher-forced.
Rows whose discrete expert choice is a near-tie in the oracle (R13) are set aside and counted."""
import numpy as np
import pytest

from oracle import rollout as ro
from paper_2605_30859_b200 import workloads as wl
from tests.gpu_util import make_ctx, rel_inf
from tests.test_gpu_bf16 import run_stepwise

pytestmark = pytest.mark.gpu

MOE_F32 = dict(n_layers=2, d_model=128, n_q_heads=4, n_kv_heads=2, head_dim=32, ffn=0, vocab=512, n_experts=8, top_k=2,
               expert_ffn=64, qk_norm=False, rope_theta=1.0e6, rms_eps=1.0e-6, dtype="f32")
MOE_BF16 = dict(n_layers=3, d_model=256, n_q_heads=4, n_kv_heads=2, head_dim=128, ffn=0, vocab=1024, n_experts=16, top_k=4,
                expert_ffn=128, qk_norm=False, rope_theta=1.0e6, rms_eps=1.0e-6, dtype="bf16")


def _case(cfg, seed, page, tol, gap_tol, std):
    from paper_2605_30859_b200 import api
    G, P, max_new, K, T = 3, 40, 24, 2, 1.0
    rng = np.random.default_rng(seed)
    prompts = [rng.integers(0, cfg["vocab"] - 1, size=n).astype(np.int32) for n in (40, 17, 33)]
    Kp = np.asarray([4, 5, 3], dtype=np.int32)
    forced = wl.make_forced_len(Kp, dict(kind="lognormal", mu=2.5, sigma=0.6, lo=2, hi=40), seed)
    d, host = make_ctx(cfg, seed, G, 5, P, max_new, page=page, flags=api.FLAG_DUMP_LOGITS, std=std)
    gpu, glog = run_stepwise(d, prompts, Kp, K, T, seed, forced)
    orc = ro.rollout_stepwise(host, prompts, Kp, K, max_new, T, seed, forced_len=forced, teacher=gpu["tokens"], keep_logits=True)
    for k in ("len", "status", "sel", "sel_mask", "close_step"):
        assert np.array_equal(gpu[k], orc[k]), k
    assert set(glog.keys()) == set(orc["logits"].keys())
    errs = {k: rel_inf(glog[k], orc["logits"][k]) for k in glog}
    clear = [k for k in glog if orc["router_gap"][k] > gap_tol]
    assert len(clear) >= len(glog) // 2, (len(clear), len(glog))
    worst = max(errs[k] for k in clear)
    assert worst < tol, worst
    cnt = d.counters()
    assert cnt["n_generated_tokens"] == orc["n_generated_tokens"]
    d.close()
    return len(glog) - len(clear), worst


def test_moe_fp32_generic_path_matches_oracle():
    near, worst = _case(MOE_F32, seed=1, page=16, tol=1e-4, gap_tol=1e-5, std=0.05)
    print("fp32 MoE: near-tie routings set aside", near, "worst rel logit err", worst)


def test_moe_bf16_tensor_core_path_matches_oracle():
    # the router sees the fp32 residual stream, whose bf16-induced error (~1e-2 relative) moves router probabilities by
    # ~1e-3: decisions with a smaller gap are not comparable
    near, worst = _case(MOE_BF16, seed=2, page=64, tol=2e-2, gap_tol=2e-3, std=0.05)
    print("bf16 MoE: near-tie routings set aside", near, "worst rel logit err", worst)


def test_moe_rollout_is_deterministic_and_loop_equals_stepwise():
    from paper_2605_30859_b200 import api
    cfg = dict(MOE_BF16)
    seed, G, P, max_new, K = 4, 4, 64, 32, 2
    prompts = wl.make_prompts(G, P, cfg["vocab"], seed)
    Kp = np.full(G, 4, dtype=np.int32)
    forced = wl.make_forced_len(Kp, dict(kind="lognormal", mu=2.8, sigma=0.6, lo=2, hi=32), seed)
    d, _ = make_ctx(cfg, seed, G, 4, P, max_new, page=64, flags=api.FLAG_DUMP_LOGITS, std=0.05)
    a, _ = run_stepwise(d, list(prompts), Kp, K, 1.0, 3, forced)
    b = d.rollout_host(prompts, Kp, K, max_new, 1.0, 3, forced_len=forced)
    c = d.rollout_host(prompts, Kp, K, max_new, 1.0, 3, forced_len=forced)
    for k in ("tokens", "len", "status", "sel", "sel_mask"):
        assert np.array_equal(a[k], b[k]), k
        assert np.array_equal(b[k], c[k]), k
    d.close()
