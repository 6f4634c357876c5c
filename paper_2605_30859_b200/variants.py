"""Policy variants of the rollout on one synthetic workload: the decode-side analogue of the paper's
Table 4 (dual-end ratio L:S) and Table 3 (uniform vs adaptive redundancy, :264-269).

    python -m paper_2605_30859_b200.variants [--workload c3] [--max-new N] [--layers L] [--seed S]

Same model, prompts and per-trajectory forced-EOS draws for every variant (trajectory (i, j) has the same forced length
wherever it exists), so the rows differ only by the policy:
  no-redundancy   K' = K (plain group rollout: everything generated is kept)
  dual L:S        uniform K' = 1.5 K, dual-end selection with L in {1, 2, 4}  (generation is identical, the kept set differs)
  early-stop      uniform K' = 2 K, shortest-only sampling with proactive early stop (the saturated branch for every prompt)
  adaptive        K'_i from Alg. 1 on the length variances the dual 1:7 rollout reported, budget M_total = 1.5 K G
                  (the paper's average), rule AUTO (early stop only where K'_i reaches 2 K)
Long-tail severity is made prompt-dependent here (sigma of the forced-EOS lognormal drawn per prompt from U[0.3, 1.3]; the
BASELINE.json recipe uses one sigma for all prompts, under which "adaptive" would have nothing to adapt to) — the paper's
Fig. 5 observation that high-variance prompts carry the tail.  Prints one JSON object per variant and a markdown table.
"""
import argparse
import json

import numpy as np


def forced_lengths(G, Kmax, mu, seed, max_new):
    rng = np.random.default_rng(seed)
    sigma = rng.uniform(0.3, 1.3, size=G)
    z = rng.standard_normal((G, Kmax))                       # trajectory (i, j) keeps its draw across variants
    f = np.round(np.exp(mu + sigma[:, None] * z))
    return np.clip(f, 1, 1 << 30).astype(np.int32), sigma


def main():
    import torch
    from . import api, workloads as wl
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="c3")
    ap.add_argument("--max-new", type=int, default=None)
    ap.add_argument("--layers", type=int, default=None)
    ap.add_argument("--seed", type=int, default=0)
    a = ap.parse_args()
    c = wl.CONFIGS[a.workload]
    cfg = dict(c["model"])
    if a.layers:
        cfg["n_layers"] = a.layers
    G, P, K = c["G"], c["P"], c["K"]
    max_new = a.max_new or c["max_new"]
    mu = c["forced"]["mu"] if c["forced"]["kind"] == "lognormal" else c["forced"]["mu"][0]
    model = wl.make_model(cfg, seed=a.seed, device="cuda")
    R = G * 2 * K
    page = 64
    kv_page_bytes = cfg["n_layers"] * 2 * cfg["n_kv_heads"] * page * cfg["head_dim"] * 2
    n_pages = min(G * ((P + page - 1) // page) + R * (max_new // page + 1), int(120e9 // kv_page_bytes))
    d = api.Darts(model, page_size=page, n_pages=n_pages, max_rows=R, max_prompts=G, max_prompt_len=P, max_new=max_new)
    prompts = wl.make_prompts(G, P, cfg["vocab"], a.seed)
    forced_all, sigma = forced_lengths(G, 2 * K, mu, a.seed, max_new)
    toks = torch.from_numpy(prompts).cuda()

    def run(name, Kp, L_long, mode):
        Kp = np.ascontiguousarray(Kp, dtype=np.int32)
        f = forced_all[:, : int(Kp.max())].copy()
        for i in range(G):
            f[i, Kp[i]:] = 0
        f_dev = torch.from_numpy(f).cuda()
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        t0.record(d.stream)
        d.prefill_device(toks, P, Kp, K, temperature=1.0, seed=a.seed, forced_len_dev=f_dev, L_long=L_long, mode=mode)
        d.run_to_completion()
        t1.record(d.stream)
        torch.cuda.synchronize()
        res, cnt = d.results(), d.counters()
        offs = np.concatenate([[0], np.cumsum(Kp)])
        kept = np.concatenate([res["len"][offs[i] + res["sel"][i]] for i in range(G)])
        ms = t0.elapsed_time(t1)
        row = dict(variant=name, rows=int(Kp.sum()), decode_steps=int(cnt["n_steps"]), generated_tokens=int(cnt["n_generated_tokens"]),
                   kept_tokens=int(cnt["n_kept_tokens"]), kept_len_mean=float(kept.mean()), kept_len_max=int(kept.max()),
                   kept_truncated=int(np.sum(np.concatenate([res["status"][offs[i] + res["sel"][i]] for i in range(G)]) == api.ROW_TRUNC)),
                   seconds=ms / 1e3, generated_tokens_per_s=cnt["n_generated_tokens"] / (ms / 1e3))
        print(json.dumps(row), flush=True)
        return row, res

    rows = []
    r, _ = run("no-redundancy K'=K", np.full(G, K), 0 if K == 1 else 1, api.MODE_DUAL_END)
    rows.append(r)
    first = None
    for L in (1, 2, 4):
        if L < K:
            r, res = run(f"dual-end K'=1.5K L:S={L}:{K - L}", np.full(G, K + K // 2), L, api.MODE_DUAL_END)
            rows.append(r)
            first = first or res
    r, _ = run("shortest-only + early stop K'=2K", np.full(G, 2 * K), 1, api.MODE_SHORTEST_EARLY_STOP)
    rows.append(r)
    ema = np.full(G, -1.0, np.float32)
    api.update_variance_ema(ema, first["len_var"], 1.0)
    Kp = api.allocate_redundancy(ema, (3 * K * G) // 2, K, 2 * K)
    r, _ = run("adaptive K'_i (Alg. 1, M_total=1.5KG), rule AUTO", Kp, 1, api.MODE_AUTO)
    r["Kp_hist"] = {int(k): int(v) for k, v in zip(*np.unique(Kp, return_counts=True))}
    r["corr_Kp_sigma"] = float(np.corrcoef(Kp, sigma)[0, 1])
    rows.append(r)
    print(json.dumps(r), flush=True)
    print("\n| variant | rows | decode steps | generated tokens | kept tokens | kept len mean / max | kept TRUNC | s | generated tok/s |\n|---|---|---|---|---|---|---|---|---|")
    for r in rows:
        print(f"| {r['variant']} | {r['rows']} | {r['decode_steps']} | {r['generated_tokens']} | {r['kept_tokens']} | {r['kept_len_mean']:.0f} / {r['kept_len_max']} | "
              f"{r['kept_truncated']} | {r['seconds']:.1f} | {r['generated_tokens_per_s']:.0f} |")
    d.close()


if __name__ == "__main__":
    main()
