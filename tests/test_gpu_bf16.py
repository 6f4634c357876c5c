"""-m gpu parity of the bf16 tensor-core path (tcgen05 GEMMs, tuned attention, fused LM-head sampling) against the oracle,
teacher-forced (R12): the oracle consumes the GPU's tokens, logits must agree within 2e-2 relative
(north_star), tokens must agree wherever the oracle's margin exceeds twice the measured logit error."""
import numpy as np
import pytest
from oracle.sampling import token_logprob

from oracle import PRUNED, MODE_DUAL_END
from oracle import rollout as ro
from paper_2605_30859_b200 import workloads as wl
from tests.gpu_util import make_ctx, rel_inf

pytestmark = pytest.mark.gpu

LOGIT_TOL_BF16 = 2e-2

SMALL = dict(n_layers=2, d_model=256, n_q_heads=4, n_kv_heads=2, head_dim=128, ffn=512, vocab=1024, n_experts=0, top_k=0,
             expert_ffn=0, qk_norm=False, rope_theta=1.0e6, rms_eps=1.0e-6, dtype="bf16")


def run_stepwise(d, prompts, Kp, K, T, seed, forced, routing=False, **kw):
    """Drive the C-ABI step by step, keeping the fp32 logits of every (row, step).  routing=True (MoE): also the expert ids every
    layer's router chose, keyed the way oracle.rollout.rollout_stepwise(routing=...) takes them; returns (results, logits, routing)."""
    d.prefill(prompts, Kp, K, temperature=T, seed=seed, forced_len=forced, **kw)
    R = int(np.sum(Kp))
    route = {}
    if routing:
        offs = np.concatenate([[0], np.cumsum([len(p) for p in prompts])])
        assert offs[-1] <= 4096                                  # one prefill pass: slot = index of the prompt token
        ids = d.debug_routing(0, int(offs[-1]))
        for i in range(len(prompts)):
            route[("prefill", i)] = ids[:, offs[i]:offs[i + 1], :].copy()
    glog = {(r, 0): d.debug_logits(r) for r in range(R)}
    d.select_and_compact()
    s = 0
    while d.n_active() > 0:
        s += 1
        d.decode_step()
        res = d.results()
        if routing:
            slot, step = d.debug_row_slots()
            ids = d.debug_routing(0, int(slot[step == s].max()) + 1)
        for r in range(R):
            if res["len"][r] == s + 1:
                glog[(r, s)] = d.debug_logits(r)
                if routing:
                    assert step[r] == s
                    route[(r, s)] = ids[:, slot[r], :].copy()
        d.select_and_compact()
    return (d.results(), glog, route) if routing else (d.results(), glog)


# std 0.02 is the configs' init recipe (tolerance: north_star's 2e-2).  std 0.08 is a stress case outside the recipe:
# sharper softmaxes amplify the bf16 rounding of q, k, P and the activations, so it gets twice the tolerance.
# vocab 1000: the last 128-id tile of the LM head holds 104 ids and its last warp quadrant 8 (ragged tail of the sampling epilogue).
@pytest.mark.parametrize("qk_norm,std,tol,vocab,pairs", [(False, 0.02, LOGIT_TOL_BF16, 1024, False), (True, 0.02, LOGIT_TOL_BF16, 1024, False),
                                                         (False, 0.08, 2 * LOGIT_TOL_BF16, 1024, False), (False, 0.02, LOGIT_TOL_BF16, 1000, False),
                                                         (True, 0.02, LOGIT_TOL_BF16, 1000, True)])      # projections on the CTA-pair kernel
def test_small_bf16_model_matches_oracle(qk_norm, std, tol, vocab, pairs):
    from paper_2605_30859_b200 import api
    cfg = dict(SMALL, qk_norm=qk_norm, vocab=vocab)
    seed, G, P, max_new, K, T = 5, 3, 70, 40, 2, 1.0
    rng = np.random.default_rng(seed)
    prompts = [rng.integers(0, cfg["vocab"] - 1, size=n).astype(np.int32) for n in (70, 33, 64)]
    Kp = np.asarray([4, 5, 3], dtype=np.int32)
    forced = wl.make_forced_len(Kp, dict(kind="lognormal", mu=2.8, sigma=0.7, lo=2, hi=60), seed)
    d, host = make_ctx(cfg, seed, G, 5, P, max_new, page=64, flags=api.FLAG_DUMP_LOGITS | (api.FLAG_CTA_PAIRS if pairs else 0), std=std)
    gpu, glog = run_stepwise(d, prompts, Kp, K, T, seed, forced)
    orc = ro.rollout_stepwise(host, prompts, Kp, K, max_new, T, seed, forced_len=forced, teacher=gpu["tokens"], keep_logits=True)
    for k in ("len", "status", "sel", "sel_mask", "close_step"):
        assert np.array_equal(gpu[k], orc[k]), k
    assert set(glog.keys()) == set(orc["logits"].keys())
    worst = max(rel_inf(glog[k], orc["logits"][k]) for k in glog)
    assert worst < tol, worst
    near = 0
    for (r, s), zg in glog.items():
        err = float(np.max(np.abs(zg - orc["logits"][(r, s)]))) / T
        if orc["margins"][r, s] > 2 * err + 1e-3:
            forced_here = s + 1 == orc["len"][r] and gpu["tokens"][r, s] == cfg["vocab"] - 1
            assert forced_here or orc["oracle_tokens"][r, s] == gpu["tokens"][r, s], (r, s)
            # log-probability of the drawn token: |d logprob| <= 2 max|d z| / T
            assert abs(gpu["logprob"][r, s] - orc["logprobs"][r, s]) <= 2 * err + 1e-3, (r, s)
            if not forced_here:                             # and tightly against the definition on the GPU's own fp32 logits
                lp = token_logprob(zg, T, int(gpu["tokens"][r, s]))
                assert abs(gpu["logprob"][r, s] - lp) < 1e-4 * (1 + abs(lp)), (r, s, gpu["logprob"][r, s], lp)
        else:
            near += 1
    assert near <= len(glog) // 10, (near, len(glog))
    cnt = d.counters()
    assert cnt["n_generated_tokens"] == orc["n_generated_tokens"] and cnt["n_steps"] == orc["n_steps"]
    d.close()


def test_bf16_rollout_loop_equals_stepwise_and_is_deterministic():
    """darts_rollout_host (async loop, stale row-count upper bounds) gives the same result as the step-by-step calls."""
    from paper_2605_30859_b200 import api
    cfg = dict(SMALL)
    seed, G, P, max_new, K = 8, 4, 64, 48, 2
    prompts = wl.make_prompts(G, P, cfg["vocab"], seed)
    Kp = np.full(G, 4, dtype=np.int32)
    forced = wl.make_forced_len(Kp, dict(kind="lognormal", mu=3.0, sigma=0.6, lo=2, hi=48), seed)
    d, _ = make_ctx(cfg, seed, G, 4, P, max_new, page=64, flags=api.FLAG_DUMP_LOGITS, std=0.08)
    a, _ = run_stepwise(d, list(prompts), Kp, K, 1.0, 3, forced)
    b = d.rollout_host(prompts, Kp, K, max_new, 1.0, 3, forced_len=forced)
    c = d.rollout_host(prompts, Kp, K, max_new, 1.0, 3, forced_len=forced)
    for k in ("tokens", "len", "status", "sel", "sel_mask"):
        assert np.array_equal(a[k], b[k]), k
        assert np.array_equal(b[k], c[k]), k
    assert np.any(b["status"] == PRUNED)
    d.close()


@pytest.mark.parametrize("vocab,G,kp", [(1024, 4, 5), (1000, 4, 5), (1000, 17, 16), (1024, 33, 8)])   # 20 rows; 272 = 256 + 16 and 264 = 256 + 8 rows
def test_both_lm_head_kernels_sample_the_same_tokens(vocab, G, kp):
    """The decode LM head runs on the persistent swap-AB kernel; DARTS_FLAG_LM_HEAD_TILES selects the 128 x 128 tile kernel instead.
    Same logits (same k order), same Philox stream, same y = z / T + g: the rollouts must be identical, the log-probabilities equal
    up to the merge order of the per-tile log-sum-exps."""
    from paper_2605_30859_b200 import api
    cfg = dict(SMALL, vocab=vocab)
    seed, P, max_new, K = 11, 64, 40, 2
    prompts = wl.make_prompts(G, P, cfg["vocab"], seed)
    Kp = np.full(G, kp, dtype=np.int32)
    forced = wl.make_forced_len(Kp, dict(kind="lognormal", mu=3.0, sigma=0.6, lo=2, hi=40), seed)
    out = []
    for flags in (0, api.FLAG_LM_HEAD_TILES):
        d, _ = make_ctx(cfg, seed, G, kp, P, max_new, page=64, flags=flags)
        out.append(d.rollout_host(prompts, Kp, K, max_new, 1.0, 3, forced_len=forced))
        d.close()
    a, b = out
    for k in ("tokens", "len", "status", "sel", "sel_mask", "margin"):
        assert np.array_equal(a[k], b[k]), k
    assert np.max(np.abs(a["logprob"] - b["logprob"])) < 1e-5


def test_a_rows_bits_do_not_depend_on_the_other_rows_below_256_rows():
    """Batch invariance inside one row-count bucket: the same 64 trajectories decoded alone and next to 128 others give the
    same logits TO THE BIT.  At d_model 1024 the two runs also take different residual-add + RMSNorm kernels (one float4 per thread up to a
    row bound of 128, 256 threads walking the row above), which are chosen on the host's row bound and therefore must agree exactly."""
    from paper_2605_30859_b200 import api
    cfg = dict(SMALL, d_model=1024, n_q_heads=8, n_kv_heads=2, ffn=1024, qk_norm=True)
    seed, P, max_new, K, T = 5, 20, 12, 8, 1.0
    rng = np.random.default_rng(seed)                           # <= 240 prompt tokens: the prefill passes share a bucket too
    prompts = [rng.integers(0, cfg["vocab"] - 1, size=int(n)).astype(np.int32) for n in rng.integers(10, P + 1, size=12)]
    logs = []
    for G in (4, 12):
        d, _ = make_ctx(cfg, seed, G, 16, P, max_new, page=64, flags=api.FLAG_DUMP_LOGITS, norm_std=0.2)
        Kp = np.full(G, 16, dtype=np.int32)
        res, glog = run_stepwise(d, prompts[:G], Kp, K, T, seed, None, mode=MODE_DUAL_END)
        logs.append((res, glog))
        d.close()
    (ra, la), (rb, lb) = logs
    assert np.array_equal(ra["tokens"][:64], rb["tokens"][:64]) and np.array_equal(ra["len"][:64], rb["len"][:64])
    keys = [k for k in la if k[0] < 64]
    assert set(keys) == {k for k in lb if k[0] < 64} and len(keys) > 64 * max_new // 2
    for k in keys:
        assert np.array_equal(la[k], lb[k]), k
