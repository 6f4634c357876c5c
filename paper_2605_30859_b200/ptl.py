"""PTL(b): per-token (= per lock-step decode step) latency as a function of the active batch size b on this GPU,
its 3-stage piecewise-linear fit, and the rollout time Eq. 4 predicts from it.

  PAPER.md:163-169 §4.2.1, Eq. 4:  T = sum_m (l_(m) - l_(m-1)) * PTL(d_TP, M' - m + 1)   (lengths sorted ascending)
  PAPER.md:372-382 App. A:         PTL is profiled per batch size and fitted with a 3-stage piecewise-linear curve.

    python -m paper_2605_30859_b200.ptl --workload c3 [--rows 16,32,...] [--steps 24] [--P 512]

Measurement only (CUDA events around darts_decode_step + darts_select_and_compact through the C-ABI); the fit is an
ordinary least-squares search over two breakpoints.  d_TP = 1 (one GPU).  Context is P + a few tokens, so the curve
isolates the batch-size dependence (weights + launch floor); the KV term grows with context and is reported by bench.py.
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


def measure(workload="c3", rows=(16, 32, 64, 128, 192, 256, 384, 512), steps=24, P=None, seed=0, layers=None):
    import torch
    from . import api, workloads as wl
    c = wl.CONFIGS[workload]
    cfg = dict(c["model"])
    if layers:
        cfg["n_layers"] = layers
    P = c["P"] if P is None else P
    model = wl.make_model(cfg, seed=seed, device="cuda")
    Rmax = max(rows)
    page = 64
    Kp = 16
    d = api.Darts(model, page_size=page, n_pages=(Rmax // Kp + 1) * (P // page + 1) + Rmax * 2 + 64, max_rows=Rmax, max_prompts=Rmax // Kp + 1,
                  max_prompt_len=P, max_new=steps + 8, eos_id=-1)
    out = []
    for R in rows:
        G = max(1, R // Kp)
        kp = np.full(G, R // G, dtype=np.int32)
        prompts = wl.make_prompts(G, P, cfg["vocab"], seed)
        d.prefill(list(prompts), kp, 1, temperature=1.0, seed=seed, forced_len=None, L_long=0, mode=api.MODE_DUAL_END)
        d.select_and_compact()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for a, b in ev:
            a.record(d.stream)
            d.decode_step()
            d.select_and_compact()
            b.record(d.stream)
        torch.cuda.synchronize()
        ms = np.array([a.elapsed_time(b) for a, b in ev][4:])
        assert d.n_active() == int(kp.sum())
        out.append(dict(rows=int(kp.sum()), ms_median=float(np.median(ms)), ms_min=float(ms.min()), ms_max=float(ms.max())))
    d.close()
    return out


def predict_rollout(workload, b, t, seed=0, layers=None):
    """Eq. 4 on this GPU: T = sum over lock-step iterations of PTL(active rows), with PTL interpolated from the measured
    points (prefill not included), against the measured device time of the same rollout.  PTL(b) is measured at context = prompt
    length; Eq. 4 has no context-length term, so the prediction misses the growth of the KV reads — the difference is reported."""
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
    return dict(decode_steps=len(rows), measured_ms=ms[-1], eq4_ms=pred, ratio=ms[-1] / pred,
                note="PTL(b) measured at context = prompt length; the excess is KV traffic growing with the generated length")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="c3")
    ap.add_argument("--rows", default="16,32,64,128,192,256,384,512")
    ap.add_argument("--steps", type=int, default=24)
    ap.add_argument("--P", type=int, default=None)
    ap.add_argument("--layers", type=int, default=None)
    ap.add_argument("--predict", action="store_true",
                    help="also run one rollout of the workload and compare its device time with Eq. 4 evaluated on the fitted PTL(b)")
    a = ap.parse_args()
    pts = measure(a.workload, tuple(int(x) for x in a.rows.split(",")), a.steps, a.P, layers=a.layers)
    b, t = [p["rows"] for p in pts], [p["ms_median"] for p in pts]
    res = dict(workload=a.workload, points=pts)
    if len(b) >= 4:
        knots, vals, rmse = fit_piecewise3(b, t)
        res["fit"] = dict(knots=knots, ms_at_knots=vals, rmse_ms=rmse)
    if a.predict:
        res["eq4"] = predict_rollout(a.workload, b, t, layers=a.layers)
    json.dump(res, sys.stdout)
    print()


if __name__ == "__main__":
    main()
