"""-m gpu parity cases that close the gaps of the round-1 suite (VERDICT r1 "parity tests — gaps"):
  (a) random RMSNorm weights (attn / mlp / final / q / k norm): a kernel that drops or mis-indexes a norm weight fails;
  (b) FULL depth at full width: c3 at 36 layers, c5 at 48 layers, logits of a sampled row within north_star's 2e-2;
  (c) a LATE step: c3 width, context > three 512-token split-KV chunks + a ragged tail, ~30 rows left alive;
  (d) freed KV pages handed out again (pool sized at the rollout's own peak): bit-identical to a roomy pool and equal to the oracle;
  (e) darts_rollout itself (north_star's signature: device prompts, scalar K', L_long = 1, M_up = 2K).
All through the C-ABI; the oracle runs teacher-forced on the GPU's tokens (R12)."""
import numpy as np
import pytest

from oracle import MODE_AUTO, MODE_DUAL_END, PRUNED, TRUNC, VALID
from oracle import rollout as ro
from oracle import transformer as otf
from oracle.sampling import sample_token, token_logprob
from paper_2605_30859_b200 import workloads as wl
from tests.gpu_util import make_ctx, rel_inf
from tests.test_gpu_bf16 import SMALL, run_stepwise
from tests.test_gpu_c1 import compare_rollout
from tests.test_gpu_moe import MOE_BF16, MOE_F32
from tests.test_gpu_moe import _case as moe_case

pytestmark = pytest.mark.gpu

NORM_STD = 0.2


# ------------------------------------------------------------------------------------------------ (a) norm weights
def _teacher_forced(cfg, seed, page, tol, std, gap_tol=None, plens=(40, 17, 33), max_new=24):
    """Small model, every (row, step) logit vector against the oracle; returns (worst rel error, set aside, compared)."""
    from paper_2605_30859_b200 import api
    G, K, T = 3, 2, 1.0
    rng = np.random.default_rng(seed)
    prompts = [rng.integers(0, cfg["vocab"] - 1, size=n).astype(np.int32) for n in plens]
    Kp = np.asarray([4, 5, 3], dtype=np.int32)
    forced = wl.make_forced_len(Kp, dict(kind="lognormal", mu=2.5, sigma=0.6, lo=2, hi=40), seed)
    d, host = make_ctx(cfg, seed, G, 5, max(plens), max_new, page=page, flags=api.FLAG_DUMP_LOGITS, std=std, norm_std=NORM_STD)
    for L in host["layers"]:                                 # the weights really are not 1, and differ per layer and tensor
        assert np.std(np.asarray(L["attn_norm"])) > 0.1 and not np.array_equal(np.asarray(L["attn_norm"]), np.asarray(L["mlp_norm"]))
    gpu, glog = run_stepwise(d, prompts, Kp, K, T, seed, forced)
    orc = ro.rollout_stepwise(host, prompts, Kp, K, max_new, T, seed, forced_len=forced, teacher=gpu["tokens"], keep_logits=True)
    for k in ("len", "status", "sel", "sel_mask", "close_step"):
        assert np.array_equal(gpu[k], orc[k]), k
    assert set(glog.keys()) == set(orc["logits"].keys())
    clear = [k for k in glog if gap_tol is None or orc["router_gap"][k] > gap_tol]
    worst = max(rel_inf(glog[k], orc["logits"][k]) for k in clear)
    assert worst < tol, worst
    for (r, s) in clear:
        err = float(np.max(np.abs(glog[(r, s)] - orc["logits"][(r, s)]))) / T
        if orc["margins"][r, s] > 2 * err + 1e-3:
            forced_here = s + 1 == orc["len"][r] and gpu["tokens"][r, s] == cfg["vocab"] - 1
            assert forced_here or orc["oracle_tokens"][r, s] == gpu["tokens"][r, s], (r, s)
    d.close()
    return worst, len(glog) - len(clear), len(glog)


def test_fp32_random_norm_weights_match_oracle():
    worst, _, n = _teacher_forced(dict(wl.CONFIGS["c1"]["model"]), seed=21, page=8, tol=1e-4, std=0.3, plens=(32, 7, 19))
    print(f"fp32, random norm weights: worst rel logit err {worst:.2e} over {n} (row, step) pairs")


def test_fp32_qk_norm_random_norm_weights_match_oracle():
    worst, _, n = _teacher_forced(dict(wl.CONFIGS["c1"]["model"], qk_norm=True, n_layers=3), seed=22, page=8, tol=1e-4, std=0.3, plens=(32, 7, 19))
    print(f"fp32 + qk_norm, random norm weights: worst rel logit err {worst:.2e} over {n}")


@pytest.mark.parametrize("qk_norm", [False, True])
def test_bf16_random_norm_weights_match_oracle(qk_norm):
    # three layers: attn_norm[l + 1] (fused behind the down projection of layer l) and final_norm (behind the last one) are all different vectors
    worst, _, n = _teacher_forced(dict(SMALL, n_layers=3, qk_norm=qk_norm), seed=23, page=64, tol=2e-2, std=0.02, plens=(70, 33, 64), max_new=40)
    print(f"bf16 qk_norm={qk_norm}, random norm weights: worst rel logit err {worst:.2e} over {n}")


def test_moe_fp32_random_norm_weights_match_oracle():
    swapped, n, regret, worst = moe_case(MOE_F32, seed=24, page=16, tol=1e-4, regret_tol=1e-5, std=0.05, norm_std=NORM_STD, max_swapped=0.02)
    print(f"fp32 MoE, random norm weights: worst {worst:.2e}, {swapped}/{n} near-tie expert swaps (max regret {regret:.1e})")


def test_moe_bf16_random_norm_weights_match_oracle():
    swapped, n, regret, worst = moe_case(MOE_BF16, seed=25, page=64, tol=2e-2, regret_tol=1e-3, std=0.05, norm_std=NORM_STD)
    print(f"bf16 MoE, random norm weights: worst {worst:.2e}, {swapped}/{n} near-tie expert swaps (max regret {regret:.1e})")


# ------------------------------------------------------------------------------------------------ (b) full depth
def _bf16(name, x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).to(torch.bfloat16).to(torch.float64).numpy()


def _full_depth(name, P, sampled_prompt, steps, ideal=False):
    """The config's full layer count, width, vocab, G x K' rows and page size; a short prompt so the fp64 oracle finishes in minutes.
    The oracle reads the weights through lazy device-backed views (a host copy of c5 would be 60 GB).  MoE: the oracle follows the
    GPU's expert choices (teacher-forced routing, R13) — over 48 layers x top-8-of-128 some near-tie is a certainty — and
    every choice must be within 1e-3 (probability) of the oracle's own top-k.
    ideal=True also runs the oracle's matched-rounding mode (oracle.transformer.ROUND = bf16 at the documented rounding points), i.e.
    an ideal bf16 pipeline in fp64: on the random-init dense c3 model rounding errors are amplified layer after layer and that ideal
    pipeline ALONE is 2.3e-2 away from the definition at 36 layers (R24, profiles/r2_rounding_probe.md), so no bf16 kernel
    can meet 2e-2 there; the test then requires the GPU to be no worse than that ideal pipeline by more than a third and no further from
    it than it is from the definition.  The tight check at full depth is the layer-by-layer one below."""
    import torch
    from paper_2605_30859_b200 import api
    c = wl.CONFIGS[name]
    cfg = dict(c["model"])
    G, K, seed, T = c["G"], c["K"], 4, 1.0
    model = wl.make_model(cfg, seed=seed, device="cuda", norm_std=NORM_STD)
    x = wl.rollout_inputs(name, seed=seed, max_new=64)
    Kp = x["Kp"]
    prompts = x["prompts"][:, :P]
    R, offs = int(Kp.sum()), np.concatenate([[0], np.cumsum(Kp)])
    d = api.Darts(model, page_size=64, n_pages=G * ((P + 63) // 64) + R * 2 + 8, max_rows=R, max_prompts=G, max_prompt_len=P, max_new=64,
                  flags=api.FLAG_DUMP_LOGITS | api.FLAG_DUMP_HIDDEN)
    d.prefill(list(prompts), Kp, K, temperature=T, seed=seed, forced_len=None)
    i = sampled_prompt
    j = (7 * i + 3) % int(Kp[i])
    r = int(offs[i] + j)
    moe = cfg["n_experts"] > 0
    glog = {0: d.debug_logits(r)}
    route = {0: d.debug_routing(i * P, P)} if moe else {}    # [L][P][top_k] of the sampled prompt's positions
    hidden = [d.debug_hidden(i * P, P)]                      # [L + 1][P][d]: the residual stream at every layer boundary
    d.select_and_compact()
    for s in range(1, steps + 1):
        d.decode_step()
        glog[s] = d.debug_logits(r)
        slot, step = d.debug_row_slots()
        assert step[r] == s
        hidden.append(d.debug_hidden(int(slot[r]), 1))
        if moe:
            route[s] = d.debug_routing(int(slot[r]), 1)
        d.select_and_compact()
    gpu = d.results()
    assert np.all(gpu["len"] == steps + 1)
    host = wl.host_model(model, lazy=True)
    worst, errs, regrets, kv, kv_m, e_ideal, d_gm = 0.0, [], [], None, None, [], []
    for s in range(steps + 1):
        if moe:
            otf.ROUTE_OVERRIDE, otf.ROUTE_REGRET = iter(route[s].reshape(-1, cfg["top_k"])), []
        try:
            if s == 0:
                z, kv = otf.prefill(host, prompts[i])
                kv = [(a.copy(), b.copy()) for a, b in kv]
            else:
                z = otf.decode_one(host, kv, int(gpu["tokens"][r, s - 1]), P + s - 1)
            if moe:
                regrets += otf.ROUTE_REGRET
        finally:
            otf.ROUTE_OVERRIDE = otf.ROUTE_REGRET = None
        zg = glog[s].astype(np.float64)
        e = rel_inf(zg, z)
        errs.append(e)
        worst = max(worst, e)
        tok, margin = sample_token(z, T, seed, i, j, s)
        err = float(np.max(np.abs(zg - z))) / T
        if margin > 2 * err + 1e-3:
            assert tok == gpu["tokens"][r, s], (s, margin, err)
            assert abs(gpu["logprob"][r, s] - token_logprob(z, T, tok)) <= 2 * err + 1e-3, s
        if ideal:
            otf.ROUND = _bf16
            try:
                if s == 0:
                    zm, kv_m = otf.prefill(host, prompts[i])
                    kv_m = [(a.copy(), b.copy()) for a, b in kv_m]
                else:
                    zm = otf.decode_one(host, kv_m, int(gpu["tokens"][r, s - 1]), P + s - 1)
            finally:
                otf.ROUND = None
            e_ideal.append(rel_inf(zm, z))
            d_gm.append(rel_inf(zg, zm))
    # Layer by layer, free of the amplification: layer l of the oracle is fed the GPU's own fp32 residual stream entering layer l (all
    # P + steps positions of the row, causal) and must reproduce the stream leaving it; one layer's worth of bf16 rounding, every layer.
    Hs = np.concatenate(hidden, axis=1).astype(np.float64)   # [L + 1][P + steps][d]
    RT = np.concatenate([route[s] for s in range(steps + 1)], axis=1) if moe else None
    pos = np.arange(P + steps)
    layer_err, layer_regret = [], []
    for l, layer in enumerate(host["layers"]):
        if moe:
            otf.ROUTE_OVERRIDE, otf.ROUTE_REGRET = iter(RT[l]), []
        try:
            h_out, _, _ = otf.layer_forward(layer, cfg, Hs[l], pos)
            if moe:
                layer_regret += otf.ROUTE_REGRET
        finally:
            otf.ROUTE_OVERRIDE = otf.ROUTE_REGRET = None
        layer_err.append(max(rel_inf(Hs[l + 1][t], h_out[t]) for t in range(P + steps)))
    zL = otf.logits_from_hidden(host, Hs[-1][P - 1:])        # final norm + LM head on the GPU's last residual stream
    head_err = max(rel_inf(glog[s].astype(np.float64), zL[s]) for s in range(steps + 1))
    print(f"   layer by layer on the GPU's own residual stream: worst layer {max(layer_err):.2e} (layer {int(np.argmax(layer_err))}), "
          f"median {np.median(layer_err):.2e}; final norm + LM head {head_err:.2e}")
    assert max(layer_err) < 1e-2 and head_err < 1e-2, (layer_err, head_err)
    if moe:
        assert max(layer_regret) < 1e-3, max(layer_regret)
    swaps = f", {int(np.sum(np.asarray(regrets) > 0))}/{len(regrets)} routing decisions swapped a near-tie expert (max regret {max(regrets):.1e})" if moe else ""
    print(f"{name} at FULL depth ({cfg['n_layers']} layers), row {r}: rel logit err per step {['%.2e' % e for e in errs]}{swaps}")
    assert len(errs) == steps + 1
    if ideal:
        print(f"   ideal bf16 pipeline (matched-rounding oracle) vs the definition {['%.2e' % e for e in e_ideal]}; GPU vs that pipeline {['%.2e' % e for e in d_gm]}")
        for e, ei, dg in zip(errs, e_ideal, d_gm):
            assert e < max(2e-2, 4.0 / 3.0 * ei) and dg < max(ei, 2e-2), (e, ei, dg)
    else:
        assert worst < 2e-2, worst                           # north_star: logits within 2e-2 relative in bf16
    if moe:
        assert max(regrets) < 1e-3 and np.sum(np.asarray(regrets) > 0) <= 0.05 * len(regrets), (max(regrets), np.sum(np.asarray(regrets) > 0))
    d.close()
    del model, host
    torch.cuda.empty_cache()


def test_c3_full_depth_36_layers_sampled_row_matches_oracle():
    _full_depth("c3", P=64, sampled_prompt=13, steps=1, ideal=True)


def test_c5_full_depth_48_layers_sampled_row_matches_oracle():
    _full_depth("c5", P=16, sampled_prompt=5, steps=1)


# ------------------------------------------------------------------------------------------------ (c) late step
def test_c3_width_late_step_long_context_matches_oracle():
    """c3 width (2 layers), 512 rows at the start; forced lengths leave 30 rows alive beyond step 1150: the sampled row's context
    is 512 prompt tokens + ~1200 of its own = one prefix chunk + three 512-token suffix chunks with a ragged tail, merged from
    4 split-KV partials, inside the full model, on pages handed out over a thousand steps."""
    import torch
    from paper_2605_30859_b200 import api
    c = wl.CONFIGS["c3"]
    cfg = dict(c["model"], n_layers=2)
    G, P, K, seed, T, V = c["G"], c["P"], c["K"], 6, 1.0, c["model"]["vocab"]
    max_new = 1280
    model = wl.make_model(cfg, seed=seed, device="cuda", norm_std=NORM_STD)
    x = wl.rollout_inputs("c3", seed=seed, max_new=max_new)
    Kp = x["Kp"]
    R = int(Kp.sum())
    forced = wl.make_forced_len(Kp, dict(kind="lognormal", mu=4.0, sigma=0.8, lo=2, hi=300), seed)
    rng = np.random.default_rng(seed)
    late = rng.choice(R, size=30, replace=False)
    forced.reshape(-1)[late] = rng.integers(1160, 1216, size=30)
    target = int(late[np.argmin(forced.reshape(-1)[late])])   # the first of the late rows to stop: the other 29 are alive at its last steps
    d = api.Darts(model, page_size=64, n_pages=G * (P // 64) + 30 * 21 + R * 6, max_rows=R, max_prompts=G, max_prompt_len=P, max_new=max_new,
                  flags=api.FLAG_DUMP_LOGITS)
    d.prefill(list(x["prompts"]), Kp, K, temperature=T, seed=seed, forced_len=forced, mode=api.MODE_DUAL_END)
    d.select_and_compact()
    glog, n_act, s = {}, {}, 0
    while True:
        na = d.n_active()
        if na == 0:
            break
        s += 1
        d.decode_step()
        n_act[s] = na
        if s >= 1150 and d.results()["len"][target] == s + 1:
            glog[s] = d.debug_logits(target)
        d.select_and_compact()
    gpu = d.results()
    eos = V - 1
    for r in range(R):                                       # lengths: the forced stop, or an earlier natural EOS the row really sampled
        L = int(gpu["len"][r])
        assert gpu["status"][r] == VALID and gpu["tokens"][r, L - 1] == eos and not np.any(gpu["tokens"][r, :L - 1] == eos)
        assert L == forced.reshape(-1)[r] or L < forced.reshape(-1)[r]
    Lt = int(gpu["len"][target])
    assert Lt >= 1160 and 25 <= n_act[Lt - 1] <= 30, (Lt, n_act.get(Lt - 1))
    steps = [Lt - 2, Lt - 1]                                 # the row's last two decode steps
    i = int(np.searchsorted(np.cumsum(Kp), target, side="right"))
    j = target - int(np.concatenate([[0], np.cumsum(Kp)])[i])
    host = wl.host_model(model, lazy=True)
    hist = np.concatenate([x["prompts"][i], gpu["tokens"][target, :steps[-1]]])
    z2 = otf.forward_full(host, hist, last=2)                # logits of steps Lt-2 and Lt-1 (each from the token history before it)
    for z, s_ in zip(z2, steps):
        zg = glog[s_].astype(np.float64)
        e = rel_inf(zg, z)
        print(f"late step {s_} (context {P + s_} tokens, {n_act[s_]} rows alive): rel logit err {e:.2e}")
        assert e < 2e-2, (s_, e)
        tok, margin = sample_token(z, T, seed, i, j, s_)
        err = float(np.max(np.abs(zg - z))) / T
        if margin > 2 * err + 1e-3 and s_ + 1 != Lt:         # the last token is the forced EOS
            assert tok == gpu["tokens"][target, s_], (s_, margin, err)
    d.close()
    del model, host
    torch.cuda.empty_cache()


# ------------------------------------------------------------------------------------------------ (d) freed pages handed out again
def _reuse_case(cfg, page, std, max_new, mu, Kp, K, mode, seed, P):
    Kp = np.asarray(Kp, dtype=np.int32)
    G = len(Kp)
    rng = np.random.default_rng(seed)
    prompts = [rng.integers(0, cfg["vocab"] - 1, size=int(rng.integers(P // 2, P + 1))).astype(np.int32) for _ in range(G)]
    forced = wl.make_forced_len(Kp, dict(kind="lognormal", mu=mu, sigma=1.0, lo=2, hi=2 * max_new), seed)   # long tail
    forced[2, 0] = 10 * max_new                              # never fires: this row of the dual-end group runs into the length limit
    # roomy pool first: its peak is what the tight pool gets
    d, host = make_ctx(cfg, seed, G, int(Kp.max()), P, max_new, page=page, std=std, norm_std=NORM_STD)
    worst_case = d.rt.n_pages
    d.prefill(prompts, Kp, K, temperature=1.0, seed=seed, forced_len=forced, mode=mode)
    d.run_to_completion()
    roomy, c0 = d.results(), d.counters()
    d.close()
    n_pages = int(c0["peak_pages"])
    assert n_pages <= 0.6 * worst_case, (n_pages, worst_case)
    d, _ = make_ctx(cfg, seed, G, int(Kp.max()), P, max_new, page=page, std=std, norm_std=NORM_STD, n_pages=n_pages)
    d.prefill(prompts, Kp, K, temperature=1.0, seed=seed, forced_len=forced, mode=mode)
    d.run_to_completion()
    tight, c1 = d.results(), d.counters()
    d.close()
    assert c1["pages_allocated"] == c0["pages_allocated"] and c1["peak_pages"] == n_pages
    assert c1["pages_allocated"] > 1.15 * n_pages, (c1["pages_allocated"], n_pages)    # freed pages really were handed out again
    for k in ("tokens", "len", "status", "sel", "sel_mask", "close_step", "margin", "logprob"):
        assert np.array_equal(roomy[k], tight[k]), k          # nothing a row computes depends on which physical page it got
    orc = ro.rollout_stepwise(host, prompts, Kp, K, max_new, 1.0, seed, forced_len=forced, mode=mode, teacher=tight["tokens"])
    return tight, orc, G, c1, n_pages, worst_case


@pytest.mark.parametrize("mode", [MODE_AUTO, MODE_DUAL_END])
def test_fp32_rollout_on_recycled_pages_matches_oracle(mode):
    cfg = dict(wl.CONFIGS["c1"]["model"])
    gpu, orc, G, cnt, n_pages, worst = _reuse_case(cfg, page=8, std=0.3, max_new=96, mu=2.8, Kp=(8, 8, 5, 8, 6), K=4, mode=mode, seed=31, P=20)
    near = compare_rollout(gpu, orc, G, 4)
    print(f"fp32 recycled pages (mode {mode}): pool {n_pages} of worst-case {worst}, {cnt['pages_allocated']} allocations, near-ties {near}")
    assert np.any(gpu["status"] == TRUNC) and (mode != MODE_AUTO or np.any(gpu["status"] == PRUNED))


@pytest.mark.parametrize("mode", [MODE_AUTO, MODE_DUAL_END])
def test_bf16_rollout_on_recycled_pages_matches_oracle(mode):
    cfg = dict(SMALL, n_layers=2)
    gpu, orc, G, cnt, n_pages, worst = _reuse_case(cfg, page=64, std=0.02, max_new=400, mu=4.8, Kp=(8, 8, 5, 8), K=4, mode=mode, seed=32, P=70)
    for k in ("len", "status", "sel", "sel_mask", "close_step"):
        assert np.array_equal(gpu[k], orc[k]), k
    # bf16: tokens must agree wherever the oracle's margin clears the bf16 logit error bound (2e-2 of |z|_inf <~ 0.5 here: 2e-2 absolute)
    sure = (orc["oracle_tokens"] >= 0) & (orc["margins"] > 5e-2) & (np.arange(orc["tokens"].shape[1])[None, :] != orc["len"][:, None] - 1)
    agree = orc["oracle_tokens"][sure] == gpu["tokens"][:, :orc["tokens"].shape[1]][sure]
    assert agree.all(), (int((~agree).sum()), int(sure.sum()))
    assert np.max(np.abs(gpu["logprob"][:, :orc["tokens"].shape[1]][sure] - orc["logprobs"][sure])) < 5e-2
    print(f"bf16 recycled pages (mode {mode}): pool {n_pages} of worst-case {worst}, {cnt['pages_allocated']} allocations, "
          f"{int(sure.sum())} tokens compared, {int((orc['oracle_tokens'] >= 0).sum() - sure.sum())} near-ties / final tokens set aside")


# ------------------------------------------------------------------------------------------------ (e) darts_rollout itself
@pytest.mark.parametrize("Kp,K,max_len", [(8, 4, 64), (6, 4, 64), (3, 1, 64), (8, 4, 40), (6, 4, 24)])
def test_darts_rollout_north_star_signature_matches_oracle(Kp, K, max_len):
    """darts_rollout(prompts, G, K', K, max_len, temperature, seed): device prompts [G][P], scalar K', device forced_len [G][K'];
    policy L_long = 1 (0 when K = 1), M_up = 2K, mode AUTO (Alg. 2).  K'=8, K=4: early stop; K'=6: dual-end;
    max_len below the context's max_new: rows reaching it are TRUNC."""
    import torch
    c = wl.CONFIGS["c1"]
    seed, G, P = 7, c["G"], c["P"]
    d, host = make_ctx(c["model"], seed, G, Kp, P, c["max_new"], page=16, norm_std=NORM_STD)
    prompts = wl.make_prompts(G, P, c["model"]["vocab"], seed)
    kp = np.full(G, Kp, dtype=np.int32)
    forced = wl.make_forced_len(kp, dict(c["forced"], hi=80), seed)
    pd, fd = torch.from_numpy(prompts).cuda(), torch.from_numpy(forced).cuda()
    gpu = d.rollout(pd, G, Kp, K, max_len, 0.8, seed, forced_len_dev=fd)
    cnt = d.counters()
    orc = ro.rollout_stepwise(host, prompts, kp, K, max_len, 0.8, seed, forced_len=forced, L_long=1 if K > 1 else 0, M_up=2 * K,
                              mode=MODE_AUTO, teacher=gpu["tokens"])
    compare_rollout(gpu, orc, G, K)
    assert np.all(gpu["tokens"][:, max_len:] == -1)
    assert cnt["n_steps"] == orc["n_steps"] and cnt["n_generated_tokens"] == orc["n_generated_tokens"] and cnt["n_kept_tokens"] == orc["n_kept_tokens"]
    assert np.any(gpu["status"] == PRUNED) == (Kp >= 2 * K)
    assert np.array_equal(gpu["n_pruned"], (orc["status"].reshape(G, Kp) == PRUNED).sum(axis=1))   # which groups' sigma_L^2 is censored (R25)
    if max_len == 24:                                        # dual-end pool (nobody is pruned) with a limit below the forced lengths' tail
        assert np.any(gpu["status"] == TRUNC)
    # out = NULL, results fetched afterwards, and the host-buffer entry point with the same policy spelled out: same bits
    assert d.rollout(pd, G, Kp, K, max_len, 0.8, seed, forced_len_dev=fd, fetch=False) is None
    again = d.results()
    host_api = d.rollout_host(prompts, kp, K, max_len, 0.8, seed, forced_len=forced, L_long=1 if K > 1 else 0, M_up=2 * K, mode=MODE_AUTO)
    for k in ("tokens", "len", "status", "sel", "sel_mask", "close_step", "margin", "logprob", "len_mean", "len_var", "n_pruned"):
        assert np.array_equal(gpu[k], again[k]), k
        assert np.array_equal(gpu[k], host_api[k]), k
    d.close()
