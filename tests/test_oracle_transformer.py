"""Pins for oracle.transformer / oracle.attention against library routines, closed forms and invariants."""
import numpy as np
import torch
import torch.nn.functional as F

from oracle import attention, transformer as tr
from paper_2605_30859_b200 import workloads as wl


def tiny_cfg(**kw):
    cfg = dict(n_layers=2, d_model=32, n_q_heads=4, n_kv_heads=2, head_dim=8, ffn=48, vocab=40,
               n_experts=0, top_k=0, expert_ffn=0, qk_norm=False, rope_theta=1.0e4, rms_eps=1e-6, dtype="f32")
    cfg.update(kw)
    return cfg


def tiny_model(seed=0, std=0.3, norm_std=0.0, **kw):
    return wl.host_model(wl.make_model(tiny_cfg(**kw), seed=seed, std=std, norm_std=norm_std))


def test_softmax_rows_sum_to_one_and_shift_invariant():
    z = np.random.default_rng(0).normal(size=(5, 17)) * 30
    p = tr.softmax(z)
    assert np.allclose(p.sum(-1), 1.0, atol=1e-14)
    assert np.allclose(p, tr.softmax(z + 1234.5), atol=1e-13)


def test_rmsnorm_against_torch_and_invariants():
    rng = np.random.default_rng(1)
    x, w = rng.normal(size=(3, 16)), rng.normal(size=16)
    ref = F.rms_norm(torch.from_numpy(x), (16,), torch.from_numpy(w), eps=1e-6).numpy()
    assert np.allclose(tr.rmsnorm(x, w, 1e-6), ref, atol=1e-14)
    y = tr.rmsnorm(x, np.ones(16), 0.0)
    assert np.allclose(np.sqrt(np.mean(y * y, -1)), 1.0)
    assert np.allclose(tr.rmsnorm(7.0 * x, w, 0.0), tr.rmsnorm(x, w, 0.0))


def test_rope_closed_forms():
    # hd = 2: a plain 2-D rotation by angle pos (theta^0 = 1)
    x = np.array([[[1.0, 0.0]]])                                  # [T=1, H=1, hd=2]
    y = tr.rope(x, np.array([3]), 100.0)
    assert np.allclose(y[0, 0], [np.cos(3.0), np.sin(3.0)])
    # hd = 4: pairs are (0,2) at frequency 1 and (1,3) at frequency theta^(-1/2)
    x = np.array([[[1.0, 0.0, 0.0, 0.0]], [[0.0, 1.0, 0.0, 0.0]]])
    y = tr.rope(x, np.array([2, 5]), 100.0)
    assert np.allclose(y[0, 0], [np.cos(2.0), 0, np.sin(2.0), 0])
    assert np.allclose(y[1, 0], [0, np.cos(0.5), 0, np.sin(0.5)])
    # norm preserving
    z = np.random.default_rng(0).normal(size=(4, 3, 8))
    assert np.allclose(np.linalg.norm(tr.rope(z, np.arange(4), 1e4), axis=-1), np.linalg.norm(z, axis=-1))


def test_rope_scores_depend_on_relative_position_only():
    rng = np.random.default_rng(2)
    q, k = rng.normal(size=(1, 1, 16)), rng.normal(size=(1, 1, 16))
    def score(pq, pk):
        return float(np.sum(tr.rope(q, np.array([pq]), 1e6) * tr.rope(k, np.array([pk]), 1e6)))
    assert abs(score(10, 3) - score(1010, 1003)) < 1e-9
    assert abs(score(10, 3) - score(11, 3)) > 1e-6


def test_attention_against_torch_sdpa_with_gqa_mapping():
    rng = np.random.default_rng(3)
    T, Hq, Hkv, hd = 9, 4, 2, 8
    q, K, V = rng.normal(size=(Hq, hd)), rng.normal(size=(T, Hkv, hd)), rng.normal(size=(T, Hkv, hd))
    out = tr.attention_one(q, K, V, Hkv)
    tq = torch.from_numpy(q)[None, :, None, :]                                   # [1,Hq,1,hd]
    tk = torch.from_numpy(K).permute(1, 0, 2).repeat_interleave(Hq // Hkv, 0)[None]   # kv head h//rep
    tv = torch.from_numpy(V).permute(1, 0, 2).repeat_interleave(Hq // Hkv, 0)[None]
    ref = F.scaled_dot_product_attention(tq, tk, tv)[0, :, 0, :].numpy()
    assert np.allclose(out, ref, atol=1e-13)


def test_prefix_shared_equals_unshared_and_split_kv_merge_equals_unsplit():
    rng = np.random.default_rng(4)
    P, t, Hq, Hkv, hd = 13, 7, 4, 2, 8
    Kp_, Vp = rng.normal(size=(P, Hkv, hd)), rng.normal(size=(P, Hkv, hd))
    Ks, Vs = rng.normal(size=(t, Hkv, hd)), rng.normal(size=(t, Hkv, hd))
    q = rng.normal(size=(Hq, hd)) * 3
    whole = attention.attention_row(q, Kp_, Vp, Ks, Vs)
    K, V = np.concatenate([Kp_, Ks]), np.concatenate([Vp, Vs])
    for cuts in ([P], [5, P, P + 3], [1, 2, 3, 19]):
        edges = [0] + cuts + [P + t]
        for h in range(Hq):
            g = h // (Hq // Hkv)
            parts = [attention.partial(q[h], K[a:b, g], V[a:b, g]) for a, b in zip(edges[:-1], edges[1:])]
            assert np.allclose(attention.merge_partials(parts), whole[h], atol=1e-13)


def torch_forward(model, tokens):
    """The same decoder built from torch library routines (rms_norm, SDPA, silu, linear); RoPE has no
    library routine and is pinned separately above, so the oracle's own rope is applied here."""
    cfg = model["cfg"]
    t64 = lambda a: torch.from_numpy(np.asarray(a, dtype=np.float64))
    Hq, Hkv, hd, d = cfg["n_q_heads"], cfg["n_kv_heads"], cfg["head_dim"], cfg["d_model"]
    T = len(tokens)
    h = F.embedding(torch.as_tensor(tokens, dtype=torch.long), t64(model["embed"]))
    for L in model["layers"]:
        a = F.rms_norm(h, (d,), t64(L["attn_norm"]), eps=cfg["rms_eps"])
        qkv = F.linear(a, t64(L["wqkv"]))
        q, k, v = qkv.split([Hq * hd, Hkv * hd, Hkv * hd], dim=-1)
        q, k = q.reshape(T, Hq, hd), k.reshape(T, Hkv, hd)
        if cfg.get("qk_norm"):                              # per-head RMSNorm over head_dim BEFORE RoPE (R5)
            q = F.rms_norm(q, (hd,), t64(L["q_norm"]), eps=cfg["rms_eps"])
            k = F.rms_norm(k, (hd,), t64(L["k_norm"]), eps=cfg["rms_eps"])
        q = t64(tr.rope(q.numpy(), np.arange(T), cfg["rope_theta"])).permute(1, 0, 2)[None]
        k = t64(tr.rope(k.numpy(), np.arange(T), cfg["rope_theta"])).permute(1, 0, 2)[None]
        v = v.reshape(T, Hkv, hd).permute(1, 0, 2)[None]
        o = F.scaled_dot_product_attention(q, k, v, is_causal=True, enable_gqa=True)[0].permute(1, 0, 2).reshape(T, -1)
        h = h + F.linear(o, t64(L["wo"]))
        b = F.rms_norm(h, (d,), t64(L["mlp_norm"]), eps=cfg["rms_eps"])
        g, u = F.linear(b, t64(L["wgu"])).chunk(2, dim=-1)
        h = h + F.linear(F.silu(g) * u, t64(L["wd"]))
    return F.linear(F.rms_norm(h, (d,), t64(model["final_norm"]), eps=cfg["rms_eps"]), t64(model["lm_head"])).numpy()


def test_forward_full_against_torch_library_decoder():
    tokens = np.array([3, 17, 0, 39, 22, 8, 8, 1, 30, 11])
    # unit norm weights (the configs' recipe), then random ones, then random ones with the per-head QK-norm
    for kw in (dict(), dict(norm_std=0.3), dict(norm_std=0.3, qk_norm=True)):
        model = tiny_model(seed=5, **kw)
        assert np.allclose(tr.forward_full(model, tokens), torch_forward(model, tokens), atol=1e-11), kw


def test_qk_norm_branch_against_torch_rms_norm_per_head_before_rope():
    """Pins oracle.transformer.qkv_project's qk_norm branch (random q_norm / k_norm: with unit weights
    rmsnorm and rope commute and neither the order nor the weight indexing would be checked)."""
    model = tiny_model(seed=11, norm_std=0.5, qk_norm=True)
    cfg, L = model["cfg"], model["layers"][1]
    Hq, Hkv, hd = cfg["n_q_heads"], cfg["n_kv_heads"], cfg["head_dim"]
    rng = np.random.default_rng(0)
    a, pos = rng.normal(size=(3, cfg["d_model"])), np.array([0, 7, 19])
    q, k, v = tr.qkv_project(L, cfg, a, pos)
    qkv = torch.from_numpy(a) @ torch.from_numpy(np.asarray(L["wqkv"], dtype=np.float64)).T
    tq, tk, tv = qkv.split([Hq * hd, Hkv * hd, Hkv * hd], dim=-1)
    wq, wk = (torch.from_numpy(np.asarray(L[n], dtype=np.float64)) for n in ("q_norm", "k_norm"))
    assert not np.allclose(wq.numpy(), wk.numpy()) and not np.allclose(wq.numpy(), 1.0)
    nq = F.rms_norm(tq.reshape(3, Hq, hd), (hd,), wq, eps=cfg["rms_eps"]).numpy()
    nk = F.rms_norm(tk.reshape(3, Hkv, hd), (hd,), wk, eps=cfg["rms_eps"]).numpy()
    assert np.allclose(q, tr.rope(nq, pos, cfg["rope_theta"]), atol=1e-12)
    assert np.allclose(k, tr.rope(nk, pos, cfg["rope_theta"]), atol=1e-12)
    assert np.allclose(v, tv.reshape(3, Hkv, hd).numpy(), atol=1e-12)          # v: neither norm nor rotation
    # the other order (rotate, then normalise) is a different function once the weights are not 1
    wrong = F.rms_norm(torch.from_numpy(tr.rope(tq.reshape(3, Hq, hd).numpy(), pos, cfg["rope_theta"])), (hd,), wq, eps=cfg["rms_eps"]).numpy()
    assert np.max(np.abs(wrong - q)) > 1e-3


def test_incremental_decode_equals_full_causal_forward():
    for kw in (dict(), dict(qk_norm=True), dict(n_experts=4, top_k=2, expert_ffn=24, ffn=0)):
        model = tiny_model(seed=6, **kw)
        tokens = np.array([5, 1, 9, 33, 2, 2, 18, 7, 25, 12, 0, 3])
        P = 5
        full = tr.forward_full(model, tokens)
        z0, kv0 = tr.prefill(model, tokens[:P])
        assert np.allclose(z0, full[P - 1], atol=1e-11)
        kv = [(a.copy(), b.copy()) for a, b in kv0]
        for t in range(P, len(tokens)):
            z = tr.decode_one(model, kv, tokens[t], t)
            assert np.allclose(z, full[t], atol=1e-10), (kw, t)


def test_forward_full_last_n_is_a_slice_of_the_full_result():
    model = tiny_model(seed=13, norm_std=0.2)
    tokens = np.array([5, 1, 9, 33, 2, 2, 18])
    full = tr.forward_full(model, tokens)
    assert np.array_equal(tr.forward_full(model, tokens, last=2), full[-2:])
    assert np.array_equal(tr.forward_full(model, tokens, last=7), full)


def test_zero_weights_give_uniform_logits():
    model = tiny_model(seed=7)
    model["lm_head"] = np.zeros((40, 32))
    z = tr.forward_full(model, np.array([1, 2, 3]))
    assert np.all(z == 0.0)
    assert np.allclose(tr.softmax(z), 1.0 / 40)


def test_moe_single_expert_equals_dense_and_gates_sum_to_one():
    dense = tiny_model(seed=8)
    moe = tiny_model(seed=8, n_experts=1, top_k=1, expert_ffn=48, ffn=0)
    for Ld, Lm in zip(dense["layers"], moe["layers"]):
        Lm["wqkv"], Lm["wo"] = Ld["wqkv"], Ld["wo"]
        Lm["wgu_e"], Lm["wd_e"] = np.asarray(Ld["wgu"], dtype=np.float64)[None], np.asarray(Ld["wd"], dtype=np.float64)[None]
    moe["embed"], moe["lm_head"] = dense["embed"], dense["lm_head"]
    tokens = np.array([4, 4, 31, 7])
    assert np.allclose(tr.forward_full(moe, tokens), tr.forward_full(dense, tokens), atol=1e-12)
    m4 = tiny_model(seed=9, n_experts=6, top_k=3, expert_ffn=16, ffn=0)
    b = np.random.default_rng(0).normal(size=32)
    ids, w = tr.moe_route(m4["layers"][0], m4["cfg"], b)
    assert len(set(ids.tolist())) == 3 and abs(np.sum(w) - 1.0) < 1e-14 and np.all(np.diff(w) <= 0)
    p = tr.softmax(np.asarray(m4["layers"][0]["wr"], dtype=np.float64) @ b)
    assert set(ids.tolist()) == set(np.argsort(p)[-3:].tolist())


def test_moe_identical_experts_top3_equals_dense_and_scaled_experts_pin_the_gates():
    """Pins the gate-weighted combine of oracle.transformer.mlp for top_k > 1.
    (a) E identical experts, top-3: gates sum to 1, so the MoE block IS the dense MLP (a dropped gate gives 3x,
        un-renormalised probabilities give sum(p_top) x).
    (b) expert e's down-projection scaled by c_e: the block is dense(b) * sum_e w_e c_e with w from an independent
        softmax / top-k, so each gate must meet its OWN expert."""
    from scipy.special import softmax as sp_softmax
    E, k = 5, 3
    dense = tiny_model(seed=12, norm_std=0.2)
    moe = tiny_model(seed=12, norm_std=0.2, n_experts=E, top_k=k, expert_ffn=48, ffn=0)
    for Ld, Lm in zip(dense["layers"], moe["layers"]):
        Lm["wqkv"], Lm["wo"] = Ld["wqkv"], Ld["wo"]
        Lm["wgu_e"] = np.repeat(np.asarray(Ld["wgu"], dtype=np.float64)[None], E, axis=0)
        Lm["wd_e"] = np.repeat(np.asarray(Ld["wd"], dtype=np.float64)[None], E, axis=0)
    moe["embed"], moe["lm_head"] = dense["embed"], dense["lm_head"]
    tokens = np.array([4, 4, 31, 7, 19])
    assert np.allclose(tr.forward_full(moe, tokens), tr.forward_full(dense, tokens), atol=1e-11)
    Ld, Lm, cfg = dense["layers"][0], dict(moe["layers"][0]), moe["cfg"]
    c = np.array([1.0, -2.0, 0.5, 3.0, 7.0])
    Lm["wd_e"] = c[:, None, None] * Lm["wd_e"]
    b = np.random.default_rng(1).normal(size=(4, cfg["d_model"]))
    base = tr.mlp(Ld, dense["cfg"], b)
    p = sp_softmax(b @ np.asarray(Lm["wr"], dtype=np.float64).T, axis=-1)
    for t in range(4):
        top = np.argsort(p[t])[-k:]
        scale = float(np.sum(p[t, top] * c[top]) / np.sum(p[t, top]))
        assert np.allclose(tr.mlp(Lm, cfg, b[t:t + 1])[0], scale * base[t], atol=1e-11), t


def test_teacher_forced_routing_hook_is_neutral_on_own_choice_and_reports_the_regret():
    """oracle.transformer.ROUTE_OVERRIDE / ROUTE_REGRET (R13): forcing the oracle's OWN expert ids changes nothing and
    reports zero regret; forcing a swapped expert gives the gates of the forced set (independent softmax) and the probability
    difference of the swapped pair."""
    from scipy.special import softmax as sp_softmax
    model = tiny_model(seed=14, norm_std=0.2, n_experts=6, top_k=2, expert_ffn=16, ffn=0)
    tokens = np.array([3, 9, 27, 1])
    full = tr.forward_full(model, tokens)
    own = []
    orig = tr.moe_route
    try:
        tr.moe_route = lambda L, c, b: (lambda r: (own.append(r[0].copy()), r)[1])(orig(L, c, b))
        assert np.array_equal(tr.forward_full(model, tokens), full)
    finally:
        tr.moe_route = orig
    assert len(own) == 2 * 4
    tr.ROUTE_OVERRIDE, tr.ROUTE_REGRET = iter(own), []
    try:
        assert np.array_equal(tr.forward_full(model, tokens), full)
        assert tr.ROUTE_REGRET == [0.0] * 8
    finally:
        tr.ROUTE_OVERRIDE = tr.ROUTE_REGRET = None
    L, cfg = model["layers"][0], model["cfg"]
    b = np.random.default_rng(2).normal(size=cfg["d_model"])
    p = sp_softmax(np.asarray(L["wr"], dtype=np.float64) @ b)
    rank = np.argsort(-p)
    forced = np.array([rank[0], rank[2]])                    # second choice swapped for the third
    tr.ROUTE_OVERRIDE, tr.ROUTE_REGRET = iter([forced]), []
    try:
        ids, w = tr.moe_route(L, cfg, b)
        assert ids.tolist() == forced.tolist() and np.allclose(w, p[forced] / p[forced].sum(), atol=1e-15)
        assert abs(tr.ROUTE_REGRET[0] - (p[rank[1]] - p[rank[2]])) < 1e-15
    finally:
        tr.ROUTE_OVERRIDE = tr.ROUTE_REGRET = None


def test_matched_rounding_hook_is_neutral_when_off_visits_the_documented_points_and_stays_close():
    """oracle.transformer.ROUND: an identity hook reproduces the definition (to rounding order: the matched attention divides after
    P.V); every layer visits the documented rounding points; bf16 rounding moves the logits by O(2^-9), and incremental == full still
    holds under it."""
    for kw in (dict(), dict(qk_norm=True), dict(n_experts=4, top_k=2, expert_ffn=24, ffn=0)):
        model = tiny_model(seed=15, norm_std=0.2, **kw)
        tokens = np.array([5, 1, 9, 33, 2, 2, 18, 7])
        full = tr.forward_full(model, tokens)
        seen = []
        bf16 = lambda name, x: torch.from_numpy(np.ascontiguousarray(x)).to(torch.bfloat16).to(torch.float64).numpy()
        try:
            tr.ROUND = lambda name, x: (seen.append(name), x)[1]
            assert np.allclose(tr.forward_full(model, tokens), full, rtol=0, atol=1e-12), kw
            per_layer = {"xn", "q", "k", "v", "p", "ao", "xn2", "act"}
            assert set(seen) == per_layer | {"xnf"} and seen.count("xn") == 2 and seen.count("xnf") == 1
            tr.ROUND = bf16
            zr = tr.forward_full(model, tokens)
            err = np.max(np.abs(zr - full)) / np.max(np.abs(full))
            assert 1e-4 < err < 3e-2, err
            z0, kv0 = tr.prefill(model, tokens[:5])
            kv = [(a.copy(), b.copy()) for a, b in kv0]
            assert np.allclose(z0, zr[4], atol=1e-10)
            for t in range(5, len(tokens)):
                assert np.allclose(tr.decode_one(model, kv, tokens[t], t), zr[t], atol=1e-10), (kw, t)
        finally:
            tr.ROUND = None


def test_moe_route_tie_prefers_lower_expert_id():
    cfg = dict(top_k=2)
    layer = dict(wr=np.zeros((5, 3)))                       # all logits equal -> experts 0,1
    ids, w = tr.moe_route(layer, cfg, np.ones(3))
    assert ids.tolist() == [0, 1] and np.allclose(w, 0.5)


def test_linear_matches_written_out_sum():
    """oracle.linear: y[r,n] = sum_k x[r,k] W[n,k] (non-square W so a transposed operand cannot pass)."""
    from oracle.linear import linear, linear_loops
    rng = np.random.default_rng(0)
    x, W = rng.standard_normal((3, 5)), rng.standard_normal((4, 5))
    y = linear(x, W)
    assert y.shape == (3, 4)
    assert np.allclose(y, linear_loops(x, W), rtol=0, atol=1e-13)
    assert abs(y[1, 2] - sum(x[1, k] * W[2, k] for k in range(5))) < 1e-13
