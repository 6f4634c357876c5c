"""-m gpu: the CONSUMER half of token-level streaming (§4.3.2, App. E :481-489):
darts_score_begin / darts_score_chunk run a chunked teacher-forced forward over streamed token chunks on a second context (its own
KV cache) and return the log-probability of every given token.  Checked against the oracle's definition (forward over the token
history, log softmax(z / T) at the given token), against the rollout's own sampling log-probabilities, for several chunk lengths,
and inside a live streaming rollout."""
import numpy as np
import pytest

from oracle import rollout as ro
from oracle.sampling import token_logprob
from paper_2605_30859_b200 import workloads as wl
from tests.gpu_util import make_ctx
from tests.test_gpu_bf16 import SMALL
from tests.test_gpu_moe import MOE_BF16

pytestmark = pytest.mark.gpu


def _chunks(tokens, lens, n):
    """The token columns of a finished rollout cut the way darts_chunk_fn delivers them: [R, n] blocks, -1 from a row's end on."""
    steps = int(lens.max())
    for s0 in range(0, steps, n):
        s1 = min(steps, s0 + n)
        t = tokens[:, s0:s1].copy()
        t[np.arange(s0, s1)[None, :] >= lens[:, None]] = -1
        yield s0, s1, t


def _score_all(d, tokens, lens, n, max_new):
    out = np.zeros((len(lens), max_new), np.float32)
    for s0, s1, t in _chunks(tokens, lens, n):
        out[:, s0:s1] = d.score_chunk(s0, s1, t)
    return out


def _oracle_given_logprobs(host, prompts, Kp, K, max_new, T, seed, forced, gpu, mode=0):
    orc = ro.rollout_stepwise(host, prompts, Kp, K, max_new, T, seed, forced_len=forced, teacher=gpu["tokens"], keep_logits=True, mode=mode)
    assert np.array_equal(orc["len"], gpu["len"])
    lp = np.zeros((len(gpu["len"]), max_new))
    zmax = np.zeros((len(gpu["len"]), max_new))
    for (r, s), z in orc["logits"].items():
        lp[r, s] = token_logprob(z, T, int(gpu["tokens"][r, s]))
        zmax[r, s] = np.max(np.abs(z))
    return orc, lp, zmax


@pytest.mark.parametrize("T", [1.0, 0.7])
def test_fp32_chunk_scoring_matches_oracle_and_rollout(T):
    c = wl.CONFIGS["c1"]
    seed = 3
    x = wl.rollout_inputs("c1", seed=seed)
    a, host = make_ctx(c["model"], seed, c["G"], c["Kp"], c["P"], c["max_new"], page=16, norm_std=0.2)
    gpu = a.rollout_host(x["prompts"], x["Kp"], x["K"], x["max_new"], T, seed, forced_len=x["forced_len"])
    a.close()
    orc, lp_ref, _ = _oracle_given_logprobs(host, x["prompts"], x["Kp"], x["K"], x["max_new"], T, seed, x["forced_len"], gpu)
    lens, R = gpu["len"], len(gpu["len"])
    valid = np.arange(c["max_new"])[None, :] < lens[:, None]
    forced_here = np.zeros_like(valid)
    fl = np.concatenate([x["forced_len"][i, :x["Kp"][i]] for i in range(c["G"])])
    forced_here[np.arange(R), lens - 1] = fl == lens            # the rollout recorded the DRAWN token's log-prob there, the scorer scores the EOS
    b, _ = make_ctx(c["model"], seed, c["G"], c["Kp"], c["P"], c["max_new"], page=16, norm_std=0.2)
    for n in (1, 5, 16):                                        # 16-step chunks: 32 rows x 17 LM-head rows > max_rows = 32 -> one row per pass
        b.score_begin(x["prompts"], x["Kp"], temperature=T)
        lp = _score_all(b, gpu["tokens"], lens, n, c["max_new"])
        assert np.max(np.abs(lp[valid] - lp_ref[valid])) < 2e-4, (n, np.max(np.abs(lp[valid] - lp_ref[valid])))
        same = valid & ~forced_here
        assert np.max(np.abs(lp[same] - gpu["logprob"][same])) < 2e-4, n
        assert np.all(lp[~valid] == 0.0)
    from paper_2605_30859_b200 import api
    b.score_begin(x["prompts"], x["Kp"], temperature=T)
    with pytest.raises(api.DartsError) as e:                    # 40 steps + the pending row do not fit 32 LM-head rows
        b.score_chunk(0, 40, np.zeros((R, 40), np.int32))
    assert e.value.code == api.ERR_WORKSPACE_TOO_SMALL
    b.score_chunk(0, 4, np.ascontiguousarray(gpu["tokens"][:, :4]))
    with pytest.raises(api.DartsError) as e:                    # chunks must arrive in step order
        b.score_chunk(8, 12, np.ascontiguousarray(gpu["tokens"][:, 8:12]))
    assert e.value.code == api.ERR_BAD_STATE
    with pytest.raises(api.DartsError) as e:
        b.decode_step()
    assert e.value.code == api.ERR_BAD_STATE
    b.close()


@pytest.mark.parametrize("qk_norm", [False, True])
def test_bf16_chunk_scoring_matches_oracle_and_rollout(qk_norm):
    """Tensor-core path: the chunk runs through the decode step's kernels with rows = (trajectory, step) pairs; the LM-head epilogue
    keeps the target's z / T and the running log-sum-exp instead of drawing."""
    cfg = dict(SMALL, n_layers=3, qk_norm=qk_norm)
    seed, G, P, max_new, K, T = 9, 4, 70, 150, 2, 1.0
    rng = np.random.default_rng(seed)
    prompts = [rng.integers(0, cfg["vocab"] - 1, size=n).astype(np.int32) for n in (70, 33, 64, 9)]
    Kp = np.asarray([4, 6, 3, 5], dtype=np.int32)
    forced = wl.make_forced_len(Kp, dict(kind="lognormal", mu=3.6, sigma=0.8, lo=2, hi=300), seed)
    a, host = make_ctx(cfg, seed, G, 6, P, max_new, page=64, norm_std=0.2)
    a.prefill(prompts, Kp, K, temperature=T, seed=seed, forced_len=forced, mode=1)    # dual-end: nobody is pruned, long rows cross two pages
    a.run_to_completion()
    gpu = a.results()
    a.close()
    orc, lp_ref, zmax = _oracle_given_logprobs(host, prompts, Kp, K, max_new, T, seed, forced, gpu, mode=1)
    lens, R = gpu["len"], len(gpu["len"])
    assert lens.max() > 130
    valid = np.arange(max_new)[None, :] < lens[:, None]
    fl = np.concatenate([forced[i, :Kp[i]] for i in range(G)])
    forced_here = np.zeros_like(valid)
    forced_here[np.arange(R), lens - 1] = fl == lens
    b, _ = make_ctx(cfg, seed, G, 6, P, max_new, page=64, norm_std=0.2)
    worst = {}
    for n in (1, 5, 16):
        b.score_begin(prompts, Kp, temperature=T)
        lp = _score_all(b, gpu["tokens"], lens, n, max_new)
        # |d logprob| <= 2 max|dz| / T with max|dz| <= 2e-2 |z|_inf (north_star's bf16 logit tolerance)
        bound = 2 * 2e-2 * zmax / T + 1e-3
        assert np.all(np.abs(lp - lp_ref)[valid] <= bound[valid]), (n, float(np.max((np.abs(lp - lp_ref) - bound)[valid])))
        same = valid & ~forced_here
        worst[n] = (float(np.max(np.abs(lp - lp_ref)[valid])), float(np.max(np.abs(lp - gpu["logprob"])[same])))
        assert worst[n][1] < 3e-2, (n, worst[n])                 # the rollout's own values (decode path, other summation orders)
    print("bf16 chunk scoring, max |d logprob| vs (oracle, rollout) per chunk length:", worst)
    b.close()


def test_scoring_inside_a_live_streaming_rollout_and_moe():
    """The pipeline of PAPER.md §4.3.2: the rollout context streams token chunks (darts_run_to_completion_streaming), the callback hands
    each chunk to a scoring context while the rollout keeps decoding; the scorer's log-probabilities equal the sampler's own."""
    cfg = dict(MOE_BF16)
    seed, G, P, max_new, K = 4, 4, 64, 48, 2
    prompts = wl.make_prompts(G, P, cfg["vocab"], seed)
    Kp = np.full(G, 4, dtype=np.int32)
    forced = wl.make_forced_len(Kp, dict(kind="lognormal", mu=3.0, sigma=0.6, lo=2, hi=48), seed)
    a, _ = make_ctx(cfg, seed, G, 4, P, max_new, page=64, std=0.05)
    b, _ = make_ctx(cfg, seed, G, 4, P, max_new, page=64, std=0.05)
    b.score_begin(list(prompts), Kp, temperature=1.0)
    got = {}

    def on_chunk(s0, s1, tokens, logprob):
        got[(s0, s1)] = (tokens, logprob, b.score_chunk(s0, s1, tokens))

    a.prefill(list(prompts), Kp, K, temperature=1.0, seed=seed, forced_len=forced)
    a.run_to_completion_streaming(7, on_chunk)
    res = a.results()
    assert sum(s1 - s0 for s0, s1 in got) >= int(res["len"].max())
    fl = np.concatenate([forced[i, :Kp[i]] for i in range(G)])
    diffs = []
    for (s0, s1), (tok, lp_roll, lp_score) in got.items():
        for r in range(len(fl)):
            for k in range(s1 - s0):
                if tok[r, k] >= 0 and not (fl[r] == s0 + k + 1):     # a forced EOS is scored as the EOS it is, the sampler logged its draw
                    diffs.append(abs(float(lp_score[r, k]) - float(lp_roll[r, k])))
                if tok[r, k] < 0:
                    assert lp_score[r, k] == 0.0
    diffs = np.asarray(diffs)
    # MoE: a near-tie expert choice may fall differently in the batched pass (R13); everything else is bf16 summation order
    assert np.median(diffs) < 5e-3 and np.mean(diffs < 3e-2) > 0.9, (float(np.median(diffs)), float(np.mean(diffs < 3e-2)), float(diffs.max()))
    print(f"streaming + scoring (bf16 MoE): {len(diffs)} tokens, median |d logprob| {np.median(diffs):.1e}, max {diffs.max():.1e}")
    a.close()
    b.close()
