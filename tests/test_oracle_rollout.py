"""Pins for oracle.rollout on tiny random-init models: stepwise (early stop) == plain definition,
determinism, invariants.  (Trajectory content itself has no paper-printed value: see DESIGN.md.)"""
import numpy as np
import pytest

from oracle import ACTIVE, VALID, TRUNC, PRUNED, MODE_AUTO, MODE_DUAL_END, MODE_SHORTEST_EARLY_STOP
from oracle import rollout as ro
from paper_2605_30859_b200 import workloads as wl

CFG = dict(n_layers=1, d_model=16, n_q_heads=2, n_kv_heads=1, head_dim=8, ffn=24, vocab=24,
           n_experts=0, top_k=0, expert_ffn=0, qk_norm=False, rope_theta=1.0e4, rms_eps=1e-6, dtype="f32")


def setup(seed, G=3, P=5, Kp=(4, 6, 5), lo=2, hi=14):
    model = wl.host_model(wl.make_model(CFG, seed=seed, std=0.5))
    prompts = wl.make_prompts(G, P, CFG["vocab"], seed)
    Kp = np.asarray(Kp, dtype=np.int32)
    forced = wl.make_forced_len(Kp, dict(kind="lognormal", mu=1.8, sigma=0.7, lo=lo, hi=hi), seed)
    return model, prompts, Kp, forced


@pytest.mark.parametrize("seed", [0, 1, 2])
@pytest.mark.parametrize("mode,M_up", [(MODE_AUTO, 5), (MODE_SHORTEST_EARLY_STOP, None), (MODE_DUAL_END, None)])
def test_stepwise_equals_plain_definition(seed, mode, M_up):
    model, prompts, Kp, forced = setup(seed)
    kw = dict(K=3, max_new=10, T=1.0, seed=seed + 40, forced_len=forced, L_long=1, M_up=M_up, mode=mode)
    a = ro.rollout_stepwise(model, prompts, Kp, **kw)
    b = ro.rollout_plain(model, prompts, Kp, **kw)
    for key in ("tokens", "len", "status", "sel", "sel_mask", "close_step"):
        assert np.array_equal(a[key], b[key]), key
    assert a["n_steps"] == b["n_steps"]
    assert a["n_generated_tokens"] == b["n_generated_tokens"] and a["n_kept_tokens"] == b["n_kept_tokens"]
    # invariants
    offs = np.concatenate([[0], np.cumsum(Kp)])
    assert not np.any(a["status"] == ACTIVE)
    for i in range(len(Kp)):
        s = a["sel"][i]
        assert len(set(s.tolist())) == 3 and np.all((0 <= s) & (s < Kp[i]))
        assert bin(int(a["sel_mask"][i])).count("1") == 3
    for r in range(offs[-1]):
        L = a["len"][r]
        assert np.all(a["tokens"][r, :L] >= 0) and np.all(a["tokens"][r, L:] == -1)
        if a["status"][r] == VALID:
            assert a["tokens"][r, L - 1] == CFG["vocab"] - 1
        if a["status"][r] == TRUNC:
            assert L == 10
    assert a["n_active_hist"][0] == offs[-1] and np.all(np.diff(a["n_active_hist"]) <= 0)


def test_early_mode_prunes_and_saves_steps():
    model, prompts, Kp, forced = setup(3, Kp=(6, 6, 6), hi=30)
    kw = dict(K=3, max_new=30, T=1.0, seed=9, forced_len=forced)
    early = ro.rollout_stepwise(model, prompts, Kp, mode=MODE_SHORTEST_EARLY_STOP, **kw)
    dual = ro.rollout_stepwise(model, prompts, Kp, mode=MODE_DUAL_END, **kw)
    assert np.any(early["status"] == PRUNED) and not np.any(dual["status"] == PRUNED)
    assert early["n_generated_tokens"] < dual["n_generated_tokens"] and early["n_steps"] <= dual["n_steps"]
    # un-pruned rows are identical token for token (a trajectory does not depend on its batch)
    keep = early["status"] != PRUNED
    assert np.array_equal(early["tokens"][keep], dual["tokens"][keep])
    pr = np.where(~keep)[0]
    for r in pr:
        L = early["len"][r]
        assert np.array_equal(early["tokens"][r, :L], dual["tokens"][r, :L])


def test_identical_seed_identical_trajectories_and_seed_matters():
    model, prompts, Kp, forced = setup(4)
    kw = dict(K=3, max_new=10, T=1.0, forced_len=None)
    a = ro.rollout_stepwise(model, prompts, Kp, seed=5, **kw)
    b = ro.rollout_stepwise(model, prompts, Kp, seed=5, **kw)
    c = ro.rollout_stepwise(model, prompts, Kp, seed=6, **kw)
    assert np.array_equal(a["tokens"], b["tokens"]) and not np.array_equal(a["tokens"], c["tokens"])
    # samples of one prompt are distinct draws ("independent trajectories")
    assert not np.array_equal(a["tokens"][0], a["tokens"][1])


def test_greedy_temperature_zero_makes_all_samples_equal():
    model, prompts, Kp, _ = setup(5)
    a = ro.rollout_stepwise(model, prompts, Kp, K=3, max_new=6, T=0.0, seed=1)
    offs = np.concatenate([[0], np.cumsum(Kp)])
    for i in range(len(Kp)):
        for r in range(offs[i], offs[i + 1]):
            assert np.array_equal(a["tokens"][r], a["tokens"][offs[i]])


def test_teacher_forcing_reproduces_and_reports_own_choice():
    model, prompts, Kp, forced = setup(6)
    kw = dict(K=3, max_new=10, T=1.0, seed=2, forced_len=forced)
    a = ro.rollout_stepwise(model, prompts, Kp, **kw)
    b = ro.rollout_stepwise(model, prompts, Kp, teacher=a["tokens"], **kw)
    assert np.array_equal(a["tokens"], b["tokens"]) and np.array_equal(a["oracle_tokens"], b["oracle_tokens"])
    assert np.nanmin(a["margins"]) >= 0.0


def test_config1_runs_in_seconds_and_matches_its_description():
    c = wl.CONFIGS["c1"]
    model = wl.host_model(wl.make_model(c["model"], seed=0))
    x = wl.rollout_inputs("c1", seed=0)
    assert x["prompts"].shape == (4, 32) and x["prompts"].max() <= 510
    assert x["forced_len"].min() >= 4 and x["forced_len"].max() <= 64
    out = ro.rollout_stepwise(model, x["prompts"], x["Kp"], x["K"], x["max_new"], x["temperature"], 0,
                              forced_len=x["forced_len"])
    # K'=8 >= M_up=2K=8 -> shortest-only with early stop (paper rule): stragglers are PRUNED
    assert set(np.unique(out["status"]).tolist()) <= {VALID, TRUNC, PRUNED} and np.any(out["status"] == PRUNED)
    assert out["n_steps"] == int(out["len"].max())
    for i in range(4):
        kept = out["len"][i * 8 + out["sel"][i]]
        assert np.all(out["status"][i * 8 + out["sel"][i]] == VALID) and np.all(np.diff(kept) >= 0)
