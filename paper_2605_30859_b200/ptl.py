"""PTL(b): per-token (= per lock-step decode step) latency as a function of the active batch size b on this GPU,
its 3-stage piecewise-linear fit, and the rollout time Eq. 4 predicts from it.

  PAPER.md:163-169 §4.2.1, Eq. 4:  T = sum_m (l_(m) - l_(m-1)) * PTL(d_TP, M' - m + 1)   (lengths sorted ascending)
  PAPER.md:372-382 App. A:         PTL is profiled per batch size and fitted with a 3-stage piecewise-linear curve.

    python -m paper_2605_30859_b200.ptl --workload c3 [--rows 16,32,...] [--ctx 0,1024,4096,8000] [--steps 24] [--P 512] [--predict]

Measurement only (CUDA events around darts_decode_step + darts_select_and_compact through the C-ABI); the fit is an
ordinary least-squares search over two breakpoints.  d_TP = 1 (one GPU).
The paper's PTL has one argument, the active batch size (Eq. 4); on this GPU a decode step also reads every active row's own KV,
so the cost has a second axis, the generated length t:  step(b, t) = PTL(b) + c_kv * b * t  (the attention term is linear in the
sum of the rows' contexts).  --ctx sweeps t with darts_debug_fast_forward (the rows jump to a generated length of t; only the step
TIME at that context is used), c_kv is the least-squares slope of step(b, t) - step(b, 0) over b * t, and --predict evaluates
Eq. 4 with that term on one rollout of the workload.  eq6_k() turns the fit into Eq. 6's k.
"""
import argparse
import json
import sys

import numpy as np


def fit_piecewise3(b, t):
    """Least-squares continuous 3-segment piecewise-linear fit t(b); returns (breakpoints, knot values, rmse)."""
    b, t = np.asarray(b, float), np.asarray(t, float)
    best = None
    for i in range(1, len(b) - 2):
        for j in range(i + 1, len(b) - 1):
            knots = np.array([b[0], b[i], b[j], b[-1]])
            A = np.stack([np.interp(b, knots, np.eye(4)[k]) for k in range(4)], axis=1)     # hat basis
            y, *_ = np.linalg.lstsq(A, t, rcond=None)
            rmse = float(np.sqrt(np.mean((A @ y - t) ** 2)))
            if best is None or rmse < best[2]:
                best = (knots.tolist(), y.tolist(), rmse)
    return best


def eq4_rollout_time(lengths, ptl):
    """Eq. 4 for one lock-step batch: lengths of all trajectories decoded together, ptl(b) in ms."""
    l = np.sort(np.asarray(lengths, float))
    n, prev, T = len(l), 0.0, 0.0
    for m in range(n):
        T += (l[m] - prev) * ptl(n - m)
        prev = l[m]
    return T


def fit_ctx_slope(points):
    """c_kv (ms per row-token) of step(b, t) = PTL(b) + c_kv b t: least squares through the origin of the excess over the t = 0 point of
    the same b.  points: dicts with rows, ctx, ms_median.  Returns (c_kv, worst relative residual of the two-term model)."""
    base = {p["rows"]: p["ms_median"] for p in points if p["ctx"] == 0}
    x = np.array([p["rows"] * p["ctx"] for p in points if p["ctx"] > 0], float)
    y = np.array([p["ms_median"] - base[p["rows"]] for p in points if p["ctx"] > 0], float)
    if len(x) == 0:
        return 0.0, 0.0
    c = float(x @ y / (x @ x))
    full = np.array([p["ms_median"] for p in points if p["ctx"] > 0], float)
    return c, float(np.max(np.abs(y - c * x) / full))


def eq6_k(b, t, c_kv, mean_len, b_at):
    """Eq. 6's k ("derived from the measured PTL"): the rollout time one more trajectory costs at a batch of b_at rows — it
    lengthens mean_len lock-step iterations by the PTL slope there, and its own KV is read once per iteration it lives
    (sum_{s < mean_len} c_kv s = c_kv mean_len^2 / 2).  ms per trajectory."""
    db = max(1.0, 0.05 * b_at)
    slope = (np.interp(b_at + db, b, t) - np.interp(b_at - db, b, t)) / (2 * db)
    return float(mean_len * slope + c_kv * mean_len ** 2 / 2.0)


def measure(workload="c3", rows=(16, 32, 64, 128, 192, 256, 384, 512), steps=24, P=None, seed=0, layers=None, ctxs=(0,), pool_bytes=100e9,
            attention=False):
    """`attention`: also time the attention launches of layer 0 in every step (CUDA events inside the library, DARTS_FLAG_PROFILE_ATTENTION)
    and report their median and the fraction of the measured HBM copy peak their algorithmic bytes reach."""
    import torch
    from . import api, workloads as wl
    c = wl.CONFIGS[workload]
    cfg = dict(c["model"])
    if layers:
        cfg["n_layers"] = layers
    P = c["P"] if P is None else P
    model = wl.make_model(cfg, seed=seed, device="cuda")
    Rmax = max(rows)
    page = cfg.get("page", 64 if cfg["dtype"] == "bf16" else 16)
    Kp = 16
    ctxs = sorted(set(int(t) for t in ctxs))
    max_new = max(ctxs) + (steps + 4) * len(ctxs) + 8
    # every (rows, t) pair whose KV fits the pool is timed; 512 rows x 8 K tokens (600 GB at c3) never occurs in a rollout and is skipped
    kv_page_bytes = cfg["n_layers"] * 2 * cfg["n_kv_heads"] * page * cfg["head_dim"] * (2 if cfg["dtype"] == "bf16" else 4)
    n_prefix = (Rmax // Kp + 1) * (P // page + 1)
    n_pages = min(n_prefix + Rmax * (max_new // page + 2) + 64, int(pool_bytes // kv_page_bytes))
    d = api.Darts(model, page_size=page, n_pages=n_pages, max_rows=Rmax,
                  max_prompts=Rmax // Kp + 1, max_prompt_len=P, max_new=max_new, eos_id=-1,
                  flags=api.FLAG_PROFILE_ATTENTION if attention else 0)
    kv_tok_bytes = 2 * cfg["n_kv_heads"] * cfg["head_dim"] * (2 if cfg["dtype"] == "bf16" else 4)     # K + V of one token in one layer
    out = []
    for R in rows:
        G = max(1, R // Kp)
        kp = np.full(G, R // G, dtype=np.int32)
        prompts = wl.make_prompts(G, P, cfg["vocab"], seed)
        d.prefill(list(prompts), kp, 1, temperature=1.0, seed=seed, forced_len=None, L_long=0, mode=api.MODE_DUAL_END)
        d.select_and_compact()
        done = 1
        for t in ctxs:
            if n_prefix + int(kp.sum()) * ((max(t, done) + steps + 4) // page + 2) > n_pages:
                continue
            if t > done:
                d.debug_fast_forward(t)                          # every row now has t generated tokens (profiling hook: only the time matters)
                done = t
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
            for a, b in ev:
                a.record(d.stream)
                d.decode_step()
                d.select_and_compact()
                b.record(d.stream)
            torch.cuda.synchronize()
            done += steps
            ms = np.array([a.elapsed_time(b) for a, b in ev][4:])
            assert d.n_active() == int(kp.sum())
            out.append(dict(rows=int(kp.sum()), ctx=int(t), ms_median=float(np.median(ms)), ms_min=float(ms.min()), ms_max=float(ms.max())))
            if attention:
                a_ms = float(np.median(np.asarray(d.attention_times())[-(steps - 4):]))
                # algorithmic bytes of one layer's attention in the middle of the timed steps: every row's own tokens + every prompt's prefix once
                a_bytes = (int(kp.sum()) * (done - steps / 2) + G * P) * kv_tok_bytes
                out[-1].update(attention_us=a_ms * 1e3, attention_GBps=a_bytes / (a_ms * 1e-3) / 1e9)
    d.close()
    return out


def predict_rollout(workload, b, t, seed=0, layers=None, c_kv=0.0):
    """Eq. 4 on this GPU: T = sum over lock-step iterations of PTL(active rows) [+ c_kv x active rows x step index: the
    rows' own KV, see the module docstring], with PTL interpolated from the measured points (prefill not included), against the measured
    device time of the same rollout."""
    import torch
    from . import api, workloads as wl
    c = wl.CONFIGS[workload]
    cfg = dict(c["model"])
    if layers:
        cfg["n_layers"] = layers
    G, P, K, max_new = c["G"], c["P"], c["K"], c["max_new"]
    model = wl.make_model(cfg, seed=seed, device="cuda")
    x = wl.rollout_inputs(workload, seed=seed)
    R = int(x["Kp"].sum())
    page = 64
    kv_page_bytes = cfg["n_layers"] * 2 * cfg["n_kv_heads"] * page * cfg["head_dim"] * 2
    n_pages = min(G * ((P + page - 1) // page) + R * (max_new // page + 1), int(100e9 // kv_page_bytes))
    d = api.Darts(model, page_size=page, n_pages=n_pages, max_rows=R, max_prompts=G, max_prompt_len=P, max_new=max_new)
    toks = torch.from_numpy(x["prompts"]).cuda()
    f_dev = torch.from_numpy(x["forced_len"]).cuda()
    ms = []
    for _ in range(2):                                       # the second run is the measurement
        d.prefill_device(toks, P, x["Kp"], K, temperature=1.0, seed=seed, forced_len_dev=f_dev)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(d.stream)
        d.run_to_completion()
        e1.record(d.stream)
        torch.cuda.synchronize()
        ms.append(e0.elapsed_time(e1))
    lens = d.results()["len"]
    d.close()
    steps = int(lens.max())
    rows = [int((lens > s).sum()) for s in range(1, steps)]
    pred = float(sum(np.interp(r, b, t) for r in rows))      # Eq. 4 written per step: same sum as over sorted length differences
    pred_ctx = pred + float(sum(c_kv * r * (s + 1) for s, r in enumerate(rows)))
    return dict(decode_steps=len(rows), measured_ms=ms[-1], eq4_ms=pred, ratio=ms[-1] / pred, eq4_with_ctx_ms=pred_ctx,
                ratio_with_ctx=ms[-1] / pred_ctx, c_kv_ms_per_row_token=c_kv, mean_len=float(lens.mean()),
                note="eq4_ms: PTL(b) at context = prompt length only (the paper's form); eq4_with_ctx_ms adds c_kv * rows * generated length per step")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="c3")
    ap.add_argument("--rows", default="16,32,64,128,192,256,384,512")
    ap.add_argument("--steps", type=int, default=24)
    ap.add_argument("--P", type=int, default=None)
    ap.add_argument("--layers", type=int, default=None)
    ap.add_argument("--ctx", default="0", help="generated lengths t at which every row count is timed (0 = right after the prefill)")
    ap.add_argument("--attention", action="store_true", help="also report the attention launches of layer 0 per point (time, algorithmic GB/s)")
    ap.add_argument("--predict", action="store_true",
                    help="also run one rollout of the workload and compare its device time with Eq. 4 evaluated on the fitted PTL(b)")
    a = ap.parse_args()
    pts = measure(a.workload, tuple(int(x) for x in a.rows.split(",")), a.steps, a.P, layers=a.layers, ctxs=tuple(int(x) for x in a.ctx.split(",")),
                  attention=a.attention)
    base = [p for p in pts if p["ctx"] == min(q["ctx"] for q in pts)]
    b, t = [p["rows"] for p in base], [p["ms_median"] for p in base]
    res = dict(workload=a.workload, points=pts)
    if len(b) >= 4:
        knots, vals, rmse = fit_piecewise3(b, t)
        res["fit"] = dict(knots=knots, ms_at_knots=vals, rmse_ms=rmse)
    c_kv, resid = fit_ctx_slope(pts) if any(p["ctx"] > 0 for p in pts) and any(p["ctx"] == 0 for p in pts) else (0.0, 0.0)
    res["ctx_fit"] = dict(c_kv_ms_per_row_token=c_kv, worst_rel_residual=resid)
    if a.predict:
        res["eq4"] = predict_rollout(a.workload, b, t, layers=a.layers, c_kv=c_kv)
        res["eq6_k_ms_per_trajectory"] = eq6_k(b, t, c_kv, res["eq4"]["mean_len"], float(np.mean(b)))
    json.dump(res, sys.stdout)
    print()


if __name__ == "__main__":
    main()
