"""-m gpu edge cases of the rollout against the oracle: greedy decoding (T = 0), the largest pool a group may have (K' = 32), a single
prompt with a single token, max_new = 1, every row stopping at its first token, every row running into the length limit, natural EOS
disabled — on the fp32 (generic kernels) and the bf16 (tensor-core kernels) paths."""
import numpy as np
import pytest

from oracle import TRUNC, VALID, PRUNED, MODE_AUTO, MODE_DUAL_END
from oracle import rollout as ro
from paper_2605_30859_b200 import workloads as wl
from tests.gpu_util import make_ctx

pytestmark = pytest.mark.gpu

F32 = dict(wl.CONFIGS["c1"]["model"])
BF16 = dict(n_layers=2, d_model=256, n_q_heads=4, n_kv_heads=2, head_dim=128, ffn=512, vocab=1024, n_experts=0, top_k=0, expert_ffn=0,
            qk_norm=False, rope_theta=1.0e6, rms_eps=1.0e-6, dtype="bf16")


def check(cfg, prompts, Kp, K, max_new, T, seed, forced, page, margin_tol, **kw):
    G, P = len(prompts), max(len(p) for p in prompts)
    Kp = np.asarray(Kp, np.int32)
    d, host = make_ctx(cfg, seed, G, int(Kp.max()), P, max_new, page=page, std=0.05)
    d.prefill(prompts, Kp, K, temperature=T, seed=seed, forced_len=forced, **kw)
    d.run_to_completion()
    gpu = d.results()
    bf16 = cfg["dtype"] == "bf16"
    orc = ro.rollout_stepwise(host, prompts, Kp, K, max_new, T, seed, forced_len=forced, teacher=gpu["tokens"], keep_logits=bf16, **kw)
    for key in ("len", "status", "sel", "sel_mask", "close_step"):
        assert np.array_equal(gpu[key], orc[key]), key
    near = total = 0
    for r in range(len(orc["len"])):
        for s in range(orc["len"][r]):
            # fp32: north_star's 1e-3.  bf16 (R12): a token may differ only where the oracle's margin is within twice the logit
            # error the bf16 tolerance allows at this position, 2 x 2e-2 x |z|_inf / T (T = 0: greedy on z itself)
            tol = 2 * 2e-2 * float(np.max(np.abs(orc["logits"][(r, s)]))) / (T if T else 1.0) + 1e-3 if bf16 else margin_tol
            total += 1
            if orc["margins"][r, s] > tol:
                if not (s + 1 == orc["len"][r] and gpu["status"][r] == VALID):
                    assert orc["oracle_tokens"][r, s] == gpu["tokens"][r, s], (r, s)
            else:
                near += 1
    if total:
        print(f"{cfg['dtype']}: {near}/{total} sampled tokens inside the near-tie band (not compared)")
        assert near <= 0.5 * total, (near, total)          # greedy on 1024 near-Gaussian logits: the top two are often closer than the band
    cnt = d.counters()
    assert cnt["n_generated_tokens"] == orc["n_generated_tokens"] and cnt["n_kept_tokens"] == orc["n_kept_tokens"]
    d.close()
    return gpu


@pytest.mark.parametrize("cfg,page,tol", [(F32, 16, 1e-3), (BF16, 64, None)])
def test_greedy_temperature_zero(cfg, page, tol):
    rng = np.random.default_rng(1)
    prompts = [rng.integers(0, cfg["vocab"] - 1, size=n).astype(np.int32) for n in (9, 20)]
    forced = np.array([[5, 9, 3, 12], [7, 2, 30, 30]], np.int32)
    g = check(cfg, prompts, [4, 4], 2, 16, 0.0, 4, forced, page, tol, mode=MODE_DUAL_END)
    # greedy: the samples of a prompt are identical until a forced stop cuts them
    assert np.array_equal(g["tokens"][0, :2], g["tokens"][1, :2])


@pytest.mark.parametrize("cfg,page,tol", [(F32, 16, 1e-3), (BF16, 64, None)])
def test_maximum_pool_of_32_samples(cfg, page, tol):
    rng = np.random.default_rng(2)
    prompts = [rng.integers(0, cfg["vocab"] - 1, size=33).astype(np.int32)]
    forced = np.clip(np.round(rng.lognormal(2.3, 0.6, size=(1, 32))), 2, 40).astype(np.int32)
    g = check(cfg, prompts, [32], 16, 24, 1.0, 7, forced, page, tol, mode=MODE_AUTO)          # K' = 32 = 2K: early stop
    assert np.any(g["status"] == PRUNED) and len(set(g["sel"][0].tolist())) == 16


def test_one_token_prompt_and_max_new_one():
    rng = np.random.default_rng(3)
    prompts = [np.array([5], np.int32), rng.integers(0, 500, size=3).astype(np.int32)]
    g = check(F32, prompts, [3, 2], 2, 1, 1.0, 9, None, 16, 1e-3, mode=MODE_DUAL_END)
    assert np.all(g["len"] == 1) and set(np.unique(g["status"]).tolist()) <= {VALID, TRUNC}


@pytest.mark.parametrize("cfg,page,tol", [(F32, 16, 1e-3), (BF16, 64, None)])
def test_all_rows_stop_at_their_first_token_and_all_rows_truncate(cfg, page, tol):
    rng = np.random.default_rng(4)
    prompts = [rng.integers(0, cfg["vocab"] - 1, size=n).astype(np.int32) for n in (6, 17, 11)]
    g = check(cfg, prompts, [4, 4, 4], 2, 8, 1.0, 5, np.ones((3, 4), np.int32), page, tol)     # forced EOS at len 1: no decode step runs
    assert np.all(g["len"] == 1) and np.all(g["status"] == VALID)
    # natural EOS off, no forced stop: every row hits the length limit (TRUNC) and the selection falls back to rule R8
    G, P = len(prompts), 17
    d, host = make_ctx(cfg, 5, G, 4, P, 6, page=page, std=0.05)
    d.close()
    from paper_2605_30859_b200 import api
    model_cpu = wl.make_model(cfg, seed=5, std=0.05)
    model_gpu = dict(cfg=model_cpu["cfg"], layers=[{k: v.cuda() for k, v in L.items()} for L in model_cpu["layers"]],
                     **{k: model_cpu[k].cuda() for k in ("embed", "lm_head", "final_norm")})
    d = api.Darts(model_gpu, page_size=page, n_pages=64, max_rows=12, max_prompts=3, max_prompt_len=P, max_new=6, eos_id=-1)
    d.prefill(prompts, np.full(3, 4, np.int32), 2, temperature=1.0, seed=5, forced_len=None)
    d.run_to_completion()
    g = d.results()
    orc = ro.rollout_stepwise(wl.host_model(model_cpu), prompts, [4, 4, 4], 2, 6, 1.0, 5, forced_len=None, eos_id=-1, teacher=g["tokens"])
    assert np.all(g["status"] == TRUNC) and np.all(g["len"] == 6)
    for key in ("len", "status", "sel", "sel_mask", "close_step"):
        assert np.array_equal(g[key], orc[key]), key
    d.close()


def test_stepwise_api_is_not_limited_by_an_earlier_shorter_rollout():
    """darts_rollout* take max_len per call; a later darts_prefill + darts_run_to_completion must run to the context's own limit."""
    c = wl.CONFIGS["c1"]
    x = wl.rollout_inputs("c1", seed=2)
    d, host = make_ctx(c["model"], 2, c["G"], c["Kp"], c["P"], c["max_new"], page=16)
    short = d.rollout_host(x["prompts"], x["Kp"], x["K"], 6, 1.0, 4, forced_len=None, mode=MODE_DUAL_END)
    assert short["len"].max() <= 6 and np.any(short["status"] == TRUNC)
    d.prefill(list(x["prompts"]), x["Kp"], x["K"], temperature=1.0, seed=4, forced_len=x["forced_len"], mode=MODE_DUAL_END)
    d.run_to_completion()
    full = d.results()
    orc = ro.rollout_stepwise(host, x["prompts"], x["Kp"], x["K"], c["max_new"], 1.0, 4, forced_len=x["forced_len"], mode=MODE_DUAL_END,
                              teacher=full["tokens"])
    assert full["len"].max() > 6
    for key in ("len", "status", "sel"):
        assert np.array_equal(full[key], orc[key]), key
    d.close()
