"""-m gpu parity of the CUDA path (through the C-ABI) against the oracle on config 1 (fp32) and variants."""
import numpy as np
import pytest

from oracle import ACTIVE, VALID, TRUNC, PRUNED, MODE_AUTO, MODE_DUAL_END, MODE_SHORTEST_EARLY_STOP
from oracle import rollout as ro
from paper_2605_30859_b200 import workloads as wl
from tests.gpu_util import make_ctx, rel_inf

pytestmark = pytest.mark.gpu

LOGIT_TOL_F32 = 1e-4        # north_star: "logits within 1e-4 relative in fp32"
MARGIN = 1e-3               # north_star: tokens bit-exact wherever the Gumbel-max margin exceeds 1e-3


def compare_rollout(gpu, orc, G, K):
    """`orc` ran teacher-forced on the GPU's tokens: everything integer must agree exactly; the oracle's own
    argmax must equal the GPU token wherever its margin exceeds MARGIN."""
    assert np.array_equal(gpu["len"], orc["len"])
    assert np.array_equal(gpu["status"], orc["status"])
    assert np.array_equal(gpu["sel"], orc["sel"])
    assert np.array_equal(gpu["sel_mask"], orc["sel_mask"])
    assert np.array_equal(gpu["close_step"], orc["close_step"])
    mn = orc["tokens"].shape[1]
    assert np.array_equal(gpu["tokens"][:, :mn], orc["tokens"])
    near = 0
    R = len(orc["len"])
    for r in range(R):
        for s in range(orc["len"][r]):
            forced_or_same = orc["oracle_tokens"][r, s] == gpu["tokens"][r, s]
            if orc["margins"][r, s] > MARGIN:
                # a forced EOS overwrites the sampled token: only then may they differ
                if not forced_or_same:
                    assert gpu["tokens"][r, s] == orc["tokens"][r, s] and s + 1 == orc["len"][r], (r, s)
            else:
                near += 1
            if orc["margins"][r, s] > MARGIN and forced_or_same:
                assert abs(gpu["margin"][r, s] - orc["margins"][r, s]) < 1e-3
            if orc["margins"][r, s] > MARGIN:               # both sides drew the same token (a forced EOS replaces it afterwards)
                assert abs(gpu["logprob"][r, s] - orc["logprobs"][r, s]) < 2e-4, (r, s, gpu["logprob"][r, s], orc["logprobs"][r, s])
        assert np.all(gpu["logprob"][r, orc["len"][r]:] == 0.0)
    return near


@pytest.mark.parametrize("seed", [0, 1])
def test_config1_rollout_matches_oracle(seed):
    c = wl.CONFIGS["c1"]
    x = wl.rollout_inputs("c1", seed=seed)
    d, host = make_ctx(c["model"], seed, c["G"], c["Kp"], c["P"], c["max_new"], page=16)
    gpu = d.rollout_host(x["prompts"], x["Kp"], x["K"], x["max_new"], x["temperature"], seed, forced_len=x["forced_len"])
    cnt = d.counters()
    orc = ro.rollout_stepwise(host, x["prompts"], x["Kp"], x["K"], x["max_new"], x["temperature"], seed,
                              forced_len=x["forced_len"], teacher=gpu["tokens"])
    near = compare_rollout(gpu, orc, c["G"], x["K"])
    assert near <= 5, near
    assert cnt["n_steps"] == orc["n_steps"]
    assert cnt["n_generated_tokens"] == orc["n_generated_tokens"] and cnt["n_kept_tokens"] == orc["n_kept_tokens"]
    assert cnt["kernel_launches"] > 0
    assert np.any(gpu["status"] == PRUNED)          # K'=8 >= M_up=8: early stop really happened
    d.close()


@pytest.mark.parametrize("mode,Kp,K,L_long", [(MODE_DUAL_END, (5, 8, 6), 4, 1), (MODE_AUTO, (4, 8, 7), 4, 2),
                                              (MODE_SHORTEST_EARLY_STOP, (6, 6, 3), 3, 1)])
def test_modes_ragged_prompts_and_natural_eos(mode, Kp, K, L_long):
    """Ragged prompt lengths, per-prompt K', no forced EOS on some rows (natural EOS / TRUNC paths), small vocab so
    natural EOS fires."""
    cfg = dict(wl.CONFIGS["c1"]["model"], vocab=48)
    seed, G, max_new = 3, 3, 24
    rng = np.random.default_rng(seed)
    prompts = [rng.integers(0, 47, size=n).astype(np.int32) for n in (7, 32, 19)]
    Kp = np.asarray(Kp, dtype=np.int32)
    forced = wl.make_forced_len(Kp, dict(kind="lognormal", mu=2.5, sigma=0.8, lo=2, hi=40), seed)
    d, host = make_ctx(cfg, seed, G, 8, 32, max_new, page=8, std=0.3)
    d.prefill(prompts, Kp, K, temperature=0.9, seed=11, forced_len=forced, L_long=L_long, mode=mode)
    d.run_to_completion()
    gpu = d.results()
    orc = ro.rollout_stepwise(host, prompts, Kp, K, max_new, 0.9, 11, forced_len=forced, L_long=L_long, mode=mode,
                              teacher=gpu["tokens"])
    compare_rollout(gpu, orc, G, K)
    assert set(np.unique(gpu["status"]).tolist()) <= {VALID, TRUNC, PRUNED}
    d.close()


def test_logits_step_by_step_within_1e4():
    """fp32 logits of prefill and of every decode step, every active row, against the oracle (teacher-forced)."""
    c = wl.CONFIGS["c1"]
    seed = 2
    x = wl.rollout_inputs("c1", seed=seed)
    d, host = make_ctx(c["model"], seed, c["G"], c["Kp"], c["P"], c["max_new"], page=16)
    d.prefill(x["prompts"], x["Kp"], x["K"], temperature=1.0, seed=seed, forced_len=x["forced_len"])
    R = int(x["Kp"].sum())
    glog = {}
    for r in range(R):
        glog[(r, 0)] = d.debug_logits(r)
    d.select_and_compact()
    s = 0
    while d.n_active() > 0:
        s += 1
        d.decode_step()
        res = d.results()
        for r in range(R):
            if res["len"][r] == s + 1:               # took part in this step
                glog[(r, s)] = d.debug_logits(r)
        d.select_and_compact()
    gpu = d.results()
    orc = ro.rollout_stepwise(host, x["prompts"], x["Kp"], x["K"], x["max_new"], 1.0, seed, forced_len=x["forced_len"],
                              teacher=gpu["tokens"], keep_logits=True)
    assert set(glog.keys()) == set(orc["logits"].keys())
    worst = max(rel_inf(glog[k], orc["logits"][k]) for k in glog)
    assert worst < LOGIT_TOL_F32, worst
    d.close()


def test_identical_seed_identical_rollout_and_seed_matters():
    c = wl.CONFIGS["c1"]
    x = wl.rollout_inputs("c1", seed=0)
    d, _ = make_ctx(c["model"], 0, c["G"], c["Kp"], c["P"], c["max_new"], page=16)
    a = d.rollout_host(x["prompts"], x["Kp"], x["K"], x["max_new"], 1.0, 5, forced_len=x["forced_len"])
    b = d.rollout_host(x["prompts"], x["Kp"], x["K"], x["max_new"], 1.0, 5, forced_len=x["forced_len"])
    e = d.rollout_host(x["prompts"], x["Kp"], x["K"], x["max_new"], 1.0, 6, forced_len=x["forced_len"])
    for k in ("tokens", "len", "status", "sel"):
        assert np.array_equal(a[k], b[k])
    assert not np.array_equal(a["tokens"], e["tokens"])
    d.close()


def test_early_stop_equals_full_rollout_then_sort_on_gpu():
    """Batch invariance: the EARLY result equals rolling everything out (DUAL, nobody pruned) and sorting."""
    c = wl.CONFIGS["c1"]
    x = wl.rollout_inputs("c1", seed=4)
    d, _ = make_ctx(c["model"], 4, c["G"], c["Kp"], c["P"], c["max_new"], page=16)
    early = d.rollout_host(x["prompts"], x["Kp"], x["K"], x["max_new"], 1.0, 9, forced_len=x["forced_len"], mode=MODE_SHORTEST_EARLY_STOP)
    full = d.rollout_host(x["prompts"], x["Kp"], x["K"], x["max_new"], 1.0, 9, forced_len=x["forced_len"], mode=MODE_DUAL_END)
    assert not np.any(full["status"] == PRUNED)
    for i in range(c["G"]):
        rows = np.arange(i * 8, i * 8 + 8)
        valid = sorted((int(full["len"][r]), int(r - i * 8)) for r in rows if full["status"][r] == VALID)
        assert early["sel"][i].tolist() == [j for _, j in valid[: x["K"]]]
    for r in range(32):
        L = early["len"][r]
        assert np.array_equal(early["tokens"][r, :L], full["tokens"][r, :L])
    d.close()


def test_error_paths():
    from paper_2605_30859_b200 import api
    c = wl.CONFIGS["c1"]
    x = wl.rollout_inputs("c1", seed=0)
    d, _ = make_ctx(c["model"], 0, c["G"], c["Kp"], c["P"], c["max_new"], page=16)
    with pytest.raises(api.DartsError) as e:
        d.decode_step()
    assert e.value.code == api.ERR_BAD_STATE
    with pytest.raises(api.DartsError) as e:
        d.prefill(x["prompts"], np.full(4, 3, np.int32), 4)           # K > Kp
    assert e.value.code == api.ERR_INVALID_ARG
    with pytest.raises(api.DartsError) as e:
        d.prefill(x["prompts"], x["Kp"], 4, L_long=4)                  # L_long >= K
    assert e.value.code == api.ERR_INVALID_ARG
    d.close()
    # pool too small: reported, not corrupted
    d2, _ = make_ctx(c["model"], 0, c["G"], c["Kp"], c["P"], c["max_new"], page=16, n_pages=4 * 2 + 40)
    with pytest.raises(api.DartsError) as e:
        d2.rollout_host(x["prompts"], x["Kp"], x["K"], x["max_new"], 1.0, 0)   # no forced EOS: rows run long
    assert e.value.code == api.ERR_KV_POOL_EXHAUSTED
    d2.close()
