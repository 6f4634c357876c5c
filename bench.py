#!/usr/bin/env python
"""bench.py — one JSON line: rollout generated tokens/s on 1 B200 (K'-of-K early stop) + decode HBM GB/s vs peak.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c3|c4|c5|c2] [--mode auto|early] [--impl reference]

A "step" is one pass of the whole hot path over one batch of synthetic input:
  workload c3 (default): one full group rollout of BASELINE.json configs[2] (Qwen3-4B-shaped, G=32 x K'=16, keep 8,
      max_new 8192, lognormal forced-EOS lengths): prefill, ~2000 lock-step decode steps, selection/compaction.
  workload c2: one decode-step attention over all 2048 rows of BASELINE.json configs[1].
`value` is measured with inputs resident in HBM (CUDA events on the library's stream); `e2e` goes through the
C-ABI call that takes HOST buffers (pinned) and returns HOST results.  `roofline` is the attention kernel
(the dominant HBM consumer of the decode step): algorithmic KV bytes per launch / CUDA-event duration.
`cpu_baseline` is the oracle (oracle/, numpy fp64) timed on this box's host cores on a bounded sample.
With --gpus N>1 (torchrun) every rank runs an independent replica with its own seed ("replicas only");
`value` is the sum of generated tokens over ranks divided by the max-over-ranks time.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
T_START = time.perf_counter()
EXTRA_EST_S = {"c4": 260, "c5": 290, "c5_early": 130}     # one rollout + building the model (c5: 61 GB of random weights)

KV_BYTES_PER_TOKEN_LAYER = {"c2": 2 * 8 * 128 * 2}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=float(d["hbm_gbs"]), bf16=float(d["bf16_tflops"]), bf16_sustained=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                    source="measured (MEASURED_PEAKS.json)")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sustained=1400.0, source="fallback (B200_PROFILING.md)")


class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        self.p.terminate()
        self.p.wait()
        self.f.flush()
        rows = [l.strip().split(", ") for l in open(self.f.name) if l.strip()]
        os.unlink(self.f.name)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[2:6]):
                if v.strip().lower().startswith("active"):
                    reasons.add(n)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None, reasons=sorted(reasons),
                    samples=len(sm))


def dist_setup(n):
    """One process per GPU (torchrun env).  The ranks are independent replicas: the process group only
    carries the barriers and the max / sum of the timing reduction — NCCL on GPUs, gloo when there is no GPU (CPU tests)."""
    import torch
    rank, world = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))
    local = int(os.environ.get("LOCAL_RANK", 0))
    cuda = torch.cuda.is_available()
    if cuda:
        torch.cuda.set_device(local if world > 1 else 0)
    if world > 1:
        import torch.distributed as dist
        if cuda:
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group("gloo")
    return rank, world, local


def barrier(world):
    import torch
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    if torch.cuda.is_available():
        torch.cuda.synchronize()


def allreduce(world, x, op):
    import torch
    if world == 1:
        return x
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device="cuda" if torch.cuda.is_available() else "cpu")
    dist.all_reduce(t, op=getattr(dist.ReduceOp, op))
    return float(t.item())


def aggregate(world, local_ms, local_units):
    """Whole-job throughput of N independent replicas: units of all ranks / the slowest rank's time (max over ranks)."""
    ms = allreduce(world, float(local_ms), "MAX")
    units = allreduce(world, float(local_units), "SUM")
    return units / (ms * 1e-3), ms, units


# ------------------------------------------------------------------------------------------------ c2: attention step
def attention_microbench(steps, warmup, seed=0, flags=0, G=None):
    import torch
    from paper_2605_30859_b200 import api, workloads as wl
    x = wl.attention_inputs("c2", seed=seed, device="cuda", G=G)
    Gn, P, Kp, R = x["G"], x["P"], x["Kp"], x["R"]
    page = 64
    n_pages = Gn * (P // page) + int(np.sum((x["suffix_len"] + page - 1) // page)) + 8
    d = api.Darts(dict(cfg=dict(wl.CONFIGS["c2"]["model"])), page_size=page, n_pages=max(n_pages, 2 * R + 16), max_rows=R, max_prompts=Gn,
                  max_prompt_len=P, max_new=8192, flags=flags)
    d.attn_load(Gn, P, Kp, x["k_prefix"], x["v_prefix"], x["suffix_len"], x["k_suffix"], x["v_suffix"])
    del x["k_suffix"], x["v_suffix"], x["k_prefix"], x["v_prefix"]
    out = torch.empty_like(x["q"])
    kvb = KV_BYTES_PER_TOKEN_LAYER["c2"]
    shared = not (flags & api.FLAG_NO_PREFIX_SHARING)
    algo_bytes = (int(x["suffix_len"].sum()) + (Gn if shared else R) * P) * kvb + 2 * x["q"].numel() * 2
    for _ in range(max(warmup, 3)):
        d.attention(x["q"], out)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in ev:                      # the working set (12.9 GB of KV) is ~100x the L2: no flush needed
        a.record(d.stream)
        d.attention(x["q"], out)
        b.record(d.stream)
    torch.cuda.synchronize()
    ms = [a.elapsed_time(b) for a, b in ev]
    res = dict(ms=float(np.mean(ms)), ms_min=float(np.min(ms)), algo_bytes=algo_bytes, rows=R, launches=2 * steps,
               kv_tokens=int(x["suffix_len"].sum()) + Gn * P)
    d.close()
    return res, x


def oracle_attention_sample(x_full_seed=0, n_rows=32):
    """cpu_baseline for c2: the oracle's per-row attention on a seeded sample of rows."""
    import torch
    from oracle import attention as oattn
    from paper_2605_30859_b200 import workloads as wl
    x = wl.attention_inputs("c2", seed=x_full_seed, device="cpu", G=max(1, n_rows // 16))
    f = lambda t: t.float().numpy().astype(np.float64)
    t0 = time.perf_counter()
    for r in range(x["R"]):
        a, b = int(x["suffix_offs"][r]), int(x["suffix_offs"][r + 1])
        oattn.attention_row(f(x["q"][r]), f(x["k_prefix"][r // 16]), f(x["v_prefix"][r // 16]), f(x["k_suffix"][a:b]), f(x["v_suffix"][a:b]))
    dt = time.perf_counter() - t0
    return x["R"] / dt, x["R"], torch.get_num_threads()


# ------------------------------------------------------------------------------------------------ full rollouts (c3 / c4 / c5)
# dram__bytes_read.sum + dram__bytes_write.sum of ONE attn_main_k launch from an `ncu --set full` capture (profiles/), with the
# algorithmic bytes of that same launch beside it (launches differ in size over a rollout; `achieved` is the rollout average)
NCU_ATTENTION_TRAFFIC = {"c3": dict(dram_bytes=1.2374e9, algorithmic_bytes=1.1927e9, ratio=1.037,
                                    launch="decode step 1001 of the seed-0 rollout (the first warm-up rollout's inputs): 277 rows x 1001 suffix tokens, 25 open groups",
                                    source="profiles/r2_launches_c3_step1000.md, re-capture on the final kernels (ncu --set full -k attn_main_k, bench.py --profile-step 1000)")}
# the same for ONE launch of the config-2 microbench (seed 0: 3 131 237 suffix tokens + 128 x 1024 prefix tokens = 13.396 GB algorithmic)
NCU_ATTENTION_C2 = dict(ncu_dram_bytes=13.717e9, ncu_traffic_over_algorithmic=1.024, ncu_source="profiles/r2_attention_c2.md (re-capture on the final kernels)")
KV_POOL_CAP_BYTES = {"c3": 64e9, "c4": 100e9, "c5": 36e9}


def build_rollout(name, seed, max_new=None, G=None, n_layers=None, flags=None):
    from paper_2605_30859_b200 import api, workloads as wl
    c = wl.CONFIGS[name]
    cfg = dict(c["model"])
    if n_layers:
        cfg["n_layers"] = n_layers
    G = c["G"] if G is None else G
    max_new = c["max_new"] if max_new is None else max_new
    model = wl.make_model(cfg, seed=seed, device="cuda")
    Kp_max = c["Kp"] if isinstance(c["Kp"], int) else max(c["Kp"])
    R = G * Kp_max
    page = 64
    # pool: every row's worst case is far too much; size for the expected peak with margin
    kv_page_bytes = cfg["n_layers"] * 2 * cfg["n_kv_heads"] * page * cfg["head_dim"] * 2
    n_pages = min(G * ((c["P"] + page - 1) // page) + R * (max_new // page + 1), int(KV_POOL_CAP_BYTES[name] // kv_page_bytes))
    d = api.Darts(model, page_size=page, n_pages=n_pages, max_rows=R, max_prompts=G, max_prompt_len=c["P"], max_new=max_new,
                  flags=api.FLAG_PROFILE_ATTENTION if flags is None else flags)
    return d, model, c, cfg, G, max_new


def rollout_algo_attention_bytes(lens, Kp, P, kvb):
    """Algorithmic KV bytes the attention of ONE layer must read over a whole rollout (prefix once per active group).
    lens: final lengths per row (group-major), Kp: [G] rows per group."""
    lens = np.asarray(lens)
    offs = np.concatenate([[0], np.cumsum(Kp)])
    grp = np.repeat(np.arange(len(Kp)), Kp)
    total, per_step = 0, []
    for s in range(1, int(lens.max())):
        act = lens > s                              # rows that are fed token s-1 at decode step s
        n_groups = len(np.unique(grp[act]))
        b = (int(act.sum()) * s + n_groups * P) * kvb
        per_step.append(b)
        total += b
    return total, per_step


def rollout_algo_step_bytes(cfg, lens, Kp, P):
    """Algorithmic HBM bytes of the whole decode path over a rollout: per lock-step iteration the active weights
    once (MoE: the experts actually hit, in expectation E (1 - (1 - k/E)^R) per layer), every active row's own suffix KV, each open
    group's prefix KV once, and the appended K/V — summed over the steps the final lengths imply.  Activations are ignored."""
    L, d, hd, Hq, Hkv, V = cfg["n_layers"], cfg["d_model"], cfg["head_dim"], cfg["n_q_heads"], cfg["n_kv_heads"], cfg["vocab"]
    attn_w = (Hq + 2 * Hkv) * hd * d + Hq * hd * d
    dense_w = L * (attn_w + 3 * d * cfg["ffn"]) + V * d if not cfg["n_experts"] else L * (attn_w + cfg["n_experts"] * d * 2) + V * d
    expert_w = 3 * d * cfg["expert_ffn"] if cfg["n_experts"] else 0
    kvb = 2 * Hkv * hd * 2 * L
    lens = np.asarray(lens)
    grp = np.repeat(np.arange(len(Kp)), Kp)
    total = 0.0
    for s in range(1, int(lens.max())):
        act = lens > s
        R = int(act.sum())
        w = dense_w * 2
        if cfg["n_experts"]:
            E, k = cfg["n_experts"], cfg["top_k"]
            w += L * E * (1.0 - (1.0 - k / E) ** R) * expert_w * 2
        total += w + (R * s + len(np.unique(grp[act])) * P + R) * kvb
    return total


def oracle_rollout_sample(name, model_gpu, cfg, P, n_tokens=1, seed=0):
    """cpu_baseline / reference arm: the oracle (oracle/, numpy fp64) decoding `n_tokens` tokens of ONE trajectory of
    the workload's model at context P.  The prompt's KV is drawn N(0,1) instead of being prefilled (an oracle prefill
    of P tokens at this size takes minutes); per-token cost is what the sample measures."""
    import torch
    from oracle import transformer as otf
    from oracle.sampling import sample_token
    from paper_2605_30859_b200 import workloads as wl
    host = wl.host_model(model_gpu)                 # bf16 bits copied to the host; up-cast to fp64 inside the oracle
    rng = np.random.default_rng(seed)
    Hkv, hd = cfg["n_kv_heads"], cfg["head_dim"]
    kv = [(rng.standard_normal((P, Hkv, hd)), rng.standard_normal((P, Hkv, hd))) for _ in range(cfg["n_layers"])]
    tok = 1
    t0 = time.perf_counter()
    for s in range(n_tokens):
        z = otf.decode_one(host, kv, tok, P + s)
        tok, _ = sample_token(z, 1.0, seed, 0, 0, s + 1)
    dt = time.perf_counter() - t0
    return n_tokens / dt, dt, os.cpu_count()


def rollout_bench(name, warmup, steps, e2e_steps, args, rank, world, peaks, keep_model):
    """`warmup` untimed rollouts, `steps` device-timed rollouts (inputs resident in HBM) and `e2e_steps` rollouts through darts_rollout_host
    (host buffers in, host results out; the same inputs and seeds as the device phase).  Returns the bench line's keys for this workload."""
    import torch
    from paper_2605_30859_b200 import api, workloads as wl
    d, model, c, cfg, G, max_new = build_rollout(name, seed=0, max_new=args.max_new, G=args.G, n_layers=args.layers)
    K, P = c["K"], c["P"]
    mode = api.MODE_SHORTEST_EARLY_STOP if args.mode == "early" else api.MODE_AUTO
    kvb = 2 * cfg["n_kv_heads"] * cfg["head_dim"] * 2
    n_runs = warmup + steps                               # the e2e phase re-runs the device phase's inputs and seeds: same work, comparable numbers
    host_in = [wl.rollout_inputs(name, seed=1000 * rank + it, G=G, max_new=max_new) for it in range(n_runs)]
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    gen_tokens, kept_tokens, dev_ms, e2e_ms, e2e_tokens, attn_ms, attn_bytes, steps_count, near, step_bytes = [], [], [], [], [], [], [], [], [], []
    launches = 0
    it = 0
    for phase, n in (("warmup", warmup), ("device", steps), ("e2e", e2e_steps)):
        if phase != "warmup":
            barrier(world)
        if phase == "e2e":
            it = warmup
        for _ in range(n):
            xin = host_in[it]; it += 1
            if phase == "e2e":
                p_pin, f_pin = pin(xin["prompts"]), pin(xin["forced_len"])
                t0 = time.perf_counter()
                out = d.rollout_host(p_pin.numpy(), xin["Kp"], K, max_new, 1.0, 7 + it, forced_len=f_pin.numpy(), mode=mode)
                e2e_ms.append((time.perf_counter() - t0) * 1e3)
                e2e_tokens.append(int(out["len"].sum()))
            else:
                toks = torch.from_numpy(np.ascontiguousarray(xin["prompts"])).cuda()
                f_dev = torch.from_numpy(np.ascontiguousarray(xin["forced_len"])).cuda()
                l0 = d.counters()["kernel_launches"]
                torch.cuda.synchronize()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(d.stream)
                d.prefill_device(toks, P, xin["Kp"], K, temperature=1.0, seed=7 + it, forced_len_dev=f_dev, mode=mode, max_len=max_new)
                d.run_to_completion()
                b.record(d.stream)
                torch.cuda.synchronize()
                if phase == "device":
                    dev_ms.append(a.elapsed_time(b))
                    cnt = d.counters()
                    launches += cnt["kernel_launches"] - l0
                    gen_tokens.append(cnt["n_generated_tokens"]); kept_tokens.append(cnt["n_kept_tokens"])
                    steps_count.append(cnt["n_steps"]); near.append(cnt["n_near_ties"])
                    res = d.results()
                    step_bytes.append(rollout_algo_step_bytes(cfg, res["len"], xin["Kp"], P))
                    tot, per_step = rollout_algo_attention_bytes(res["len"], xin["Kp"], P, kvb)
                    t_ms = d.attention_times()
                    m = min(len(t_ms), len(per_step))
                    attn_ms.append(float(np.sum(t_ms[:m])))
                    attn_bytes.append(float(np.sum(per_step[:m])))
        if phase != "warmup":
            barrier(world)
    value, tot_ms, tot_tok = aggregate(world, np.sum(dev_ms), np.sum(gen_tokens))
    e2e_value, tot_e2e_ms, tot_e2e_tok = aggregate(world, max(np.sum(e2e_ms), 1e-9), np.sum(e2e_tokens)) if e2e_steps else (None, 0.0, 0)
    ach = float(np.sum(attn_bytes)) / (float(np.sum(attn_ms)) * 1e-3) / 1e9 if np.sum(attn_ms) > 0 else 0.0
    R = int(host_in[0]["Kp"].sum())
    h2d = int(host_in[0]["prompts"].nbytes + host_in[0]["forced_len"].nbytes + host_in[0]["Kp"].nbytes)
    d2h = int(R * max_new * 12 + R * 5 + G * (K * 4 + 4 * 4))     # tokens, margins, log-probs; len, status; sel, mask, close step, mean, var
    attn_share = float(np.sum(attn_ms)) * cfg["n_layers"] / max(float(np.sum(dev_ms)), 1e-9)
    rule = {"c3": "K'=16 >= 2K: shortest-only + early stop", "c4": "K' in {8,12,16}: early stop only for K'=16 prompts, dual-end otherwise",
            "c5": "K'=12 < 2K: dual-end, no early stop"}[name] if args.mode == "auto" else "forced shortest-only + early stop (variant, DESIGN.md R17)"
    out = dict(metric="rollout generated tokens/s on 1 B200 (K'-of-K early stop)", value=value, unit="tokens/s",
               ms_per_step=tot_ms / max(1, steps),
               config=dict(workload=f"{name}: {cfg['n_layers']} layers d={cfg['d_model']} bf16, G={G} prompts of {P}, K'={c['Kp']}, keep {K}, "
                                    f"max_new={max_new}, forced-EOS {c['forced']['kind']}, rule: {rule}",
                           l2="per-step working set (weights + KV, > 8 GB) >> 126 MB L2, no flush",
                           decode_steps_per_rollout=int(np.mean(steps_count)), generated_tokens_per_rollout=int(np.mean(gen_tokens)),
                           kept_tokens_per_rollout=int(np.mean(kept_tokens)), near_ties_per_rollout=int(np.mean(near)),
                           ms_per_decode_step=float(np.sum(dev_ms) / max(1, np.sum(steps_count))),
                           kv_pool_pages=int(d.rt.n_pages), kv_pages_allocated_last_rollout=int(d.counters()["pages_allocated"]),
                           kv_peak_pages_last_rollout=int(d.counters()["peak_pages"])),
               roofline=dict(bound="hbm", achieved=ach, peak=peaks["hbm"], unit="GB/s", frac=ach / peaks["hbm"],
                             traffic=NCU_ATTENTION_TRAFFIC.get(name, {}).get("dram_bytes"), traffic_detail=NCU_ATTENTION_TRAFFIC.get(name),
                             traffic_note="a rollout's ~2000 x 36 launches differ in size: `achieved` is their byte-weighted average, measured live; `traffic` is "
                                          "ncu's DRAM bytes of ONE of those launches (traffic_detail names it and gives that launch's algorithmic bytes)",
                             kernel="attn_main_k+attn_merge_k (layer 0 of every decode step, CUDA events on the library's stream inside the rollout)",
                             share_of_step=attn_share, peak_source=peaks["source"]),
               gpu_launches=int(launches))
    step_gbps = float(np.sum(step_bytes)) / (float(np.sum(dev_ms)) * 1e-3) / 1e9
    out["decode_path_roofline"] = dict(bound="hbm", achieved=step_gbps, peak=peaks["hbm"], unit="GB/s", frac=step_gbps / peaks["hbm"],
                                       what="algorithmic bytes of ALL kernels of the rollout (active weights once per step, suffix KV per row, "
                                            "prefix KV once per open group, KV appends) / device time of the rollout incl. prefill")
    if e2e_steps:
        out["e2e"] = dict(value=e2e_value if tot_e2e_tok > 0 else None, unit="tokens/s", h2d_bytes_per_step=h2d,
                          d2h_bytes_per_step=d2h, ms_per_step=tot_e2e_ms / max(1, e2e_steps), api="darts_rollout_host (pinned host buffers in, host results out)")
    if args.max_new or args.G or args.layers:
        out["config"]["INVALID"] = "debug flags shrink the workload"
    d.close()
    out["cpu_model"] = None
    if keep_model:
        out["cpu_model"] = dict(cfg=model["cfg"], layers=[{k: v.cpu() for k, v in L.items()} for L in model["layers"]],
                                **{k: model[k].cpu() for k in ("embed", "lm_head", "final_norm")})
    out["cfg"] = cfg
    del model
    torch.cuda.empty_cache()
    return out


def gemm_tensor_bench(peaks, rows_list=(256, 512)):
    """The projection GEMMs of config 3 alone through the C-ABI hook (stream-K tcgen05 kernel, fp32 pieces left in place): CUDA-graph replay
    on the library's stream so the Python call path does not bound the time, weights rotated through copies that together exceed the L2,
    CUDA events around three replays.  TFLOP/s = 2 rows N K / time, against the measured bf16 burst peak (kernels timed alone)."""
    import torch
    from paper_2605_30859_b200 import api, workloads as wl
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        d = api.Darts(dict(cfg=dict(wl.CONFIGS["c2"]["model"])), page_size=64, n_pages=64, max_rows=8, max_prompts=2, max_prompt_len=64, max_new=64, stream=st)
    out = {}
    for gname, N, K in (("qkv", 6144, 2560), ("o", 2560, 4096), ("gate_up", 19456, 2560), ("down", 2560, 9728)):
        ncopy = max(2, int(400e6 // (N * K * 2)) + 1)
        Ws = [(torch.randn(N, K, device="cuda") * 0.02).to(torch.bfloat16) for _ in range(ncopy)]
        for rows in rows_list:
            X = torch.randn(rows, K, device="cuda").to(torch.bfloat16)
            scratch = torch.empty(24 * rows * N, dtype=torch.float32, device="cuda")
            n = 2 * ncopy
            torch.cuda.synchronize()
            with torch.cuda.stream(st):
                for i in range(2):
                    d.debug_gemm_bf16(X, Ws[i % ncopy], split_k=0, scratch=scratch, reduce=False)
            torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=st):
                for i in range(n):
                    d.debug_gemm_bf16(X, Ws[i % ncopy], split_k=0, scratch=scratch, reduce=False)
            g.replay()
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(3):
                g.replay()
            b.record()
            torch.cuda.synchronize()
            us = a.elapsed_time(b) * 1e3 / (3 * n)
            tf = 2.0 * rows * N * K / us / 1e6
            out[f"{gname}_{rows}"] = dict(N=N, K=K, rows=rows, us=us, tflops=tf, frac_of_bf16_burst_peak=tf / peaks["bf16"], weight_GBps=N * K * 2 / us / 1e3)
            del g
        del Ws
    d.close()
    out["peak"] = dict(bf16_tflops_burst=peaks["bf16"], source=peaks["source"], launches=int(sum(1 for _ in out)))
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--workload", default="c3", choices=["c2", "c3", "c4", "c5"])
    ap.add_argument("--mode", default="auto", choices=["auto", "early"], help="early: force shortest-only + early stop (DESIGN.md R17 variant)")
    ap.add_argument("--max-new", type=int, default=None, help="debug only: shorten the rollout (INVALID as a bench number)")
    ap.add_argument("--G", type=int, default=None, help="debug only")
    ap.add_argument("--layers", type=int, default=None, help="debug only")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the extra_workloads leg (configs 4 and 5, one timed rollout each)")
    ap.add_argument("--budget-s", type=float, default=1450.0, help="wall-clock budget of the whole command; an extra workload that would not fit is skipped and says so")
    ap.add_argument("--profile-step", type=int, default=None,
                    help="profiling aid (prints no bench line): run the workload's rollout step by step up to this decode step, then bracket "
                         "two more steps with cudaProfilerStart/Stop (use with `ncu --profile-from-start off`)")
    args = ap.parse_args()

    if args.impl == "reference":
        return reference_arm(args)
    if args.profile_step is not None:
        return profile_steps(args)

    import torch
    from paper_2605_30859_b200 import build as _build
    if not os.path.exists(_build.LIB):                       # build step (nvcc, sm_100a), not a fallback: without the library nothing runs
        _build.build()
    from paper_2605_30859_b200 import api, workloads as wl
    rank, world, local = dist_setup(args.gpus)
    peaks = measured_peaks()
    sampler = ClockSampler(local) if rank == 0 else None
    line = dict(n_gpus=world, steps=args.steps, warmup=args.warmup, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="bf16", data="synthetic")
    cpu_model = None

    if args.workload == "c2":
        barrier(world)
        res, x = attention_microbench(args.steps, args.warmup, seed=rank)
        barrier(world)
        ms = allreduce(world, res["ms"], "MAX")
        rows = allreduce(world, res["rows"], "SUM")
        ach = res["algo_bytes"] / (res["ms"] * 1e-3) / 1e9
        line.update(metric="decode attention rows (generated tokens)/s, one step over all rows", value=rows / (ms * 1e-3), unit="tokens/s",
                    ms_per_step=ms, config=dict(workload="c2: attention-only, 32q/8kv hd128 page64, G=128 x K'=16, P=1024, suffix lognormal(7.0,0.8)",
                                                l2="working set 12.9 GB >> 126 MB L2, no flush"),
                    roofline=dict(bound="hbm", achieved=ach, peak=peaks["hbm"], unit="GB/s", frac=ach / peaks["hbm"], traffic=None,
                                  kernel="attn_main_k+attn_merge_k", peak_source=peaks["source"]),
                    gpu_launches=res["launches"])
    else:
        name = args.workload
        P = wl.CONFIGS[name]["P"]
        res = rollout_bench(name, args.warmup, args.steps, args.steps, args, rank, world, peaks, keep_model=rank == 0 and not args.no_cpu_baseline)
        cpu_model, cfg = res.pop("cpu_model"), res.pop("cfg")
        line.update(res)
        if rank == 0:
            # the dominant kernel timed alone on BASELINE.json configs[1], and the projections alone at 512 rows
            res2, _ = attention_microbench(10, 3)
            a2 = res2["algo_bytes"] / (res2["ms"] * 1e-3) / 1e9
            line["attention_c2"] = dict(ms=res2["ms"], achieved_GBps=a2, frac_of_measured_peak=a2 / peaks["hbm"], rows=res2["rows"],
                                        algorithmic_bytes=res2["algo_bytes"], **NCU_ATTENTION_C2)
            line["gemm_tensor"] = gemm_tensor_bench(peaks)
        # BASELINE.json configs[3] and [4] in the same driver-run line: ONE timed rollout each (16 384 lock-step iterations, minutes), only
        # while the whole command stays clear of the driver's step limit
        if world == 1 and not (args.max_new or args.G or args.layers) and name == "c3" and not args.no_extra:
            line["extra_workloads"] = {}
            for extra in ("c4", "c5", "c5_early"):
                spent = time.perf_counter() - T_START
                if spent + EXTRA_EST_S[extra] > args.budget_s:
                    line["extra_workloads"][extra] = dict(skipped=f"{spent:.0f} s spent, needs ~{EXTRA_EST_S[extra]} s, budget {args.budget_s} s (driver step limit 1800 s)")
                    continue
                # c5_early: config 5 with shortest-only + early stop FORCED (R17: under the paper's rule K' = 12 < 2K is dual-end and
                # never stops early, while BASELINE.json's metric says "K'-of-K early stop"): a labelled variant, not the paper's rule
                xargs = argparse.Namespace(**{**vars(args), "mode": "early"}) if extra == "c5_early" else args
                r = rollout_bench(extra.split("_")[0], 0, 1, 0, xargs, rank, world, peaks, keep_model=False)
                line["extra_workloads"][extra] = dict(value=r["value"], unit="tokens/s", ms_per_rollout=r["ms_per_step"], warmup_rollouts=0, timed_rollouts=1,
                                                      config=r["config"], attention_roofline_frac=r["roofline"]["frac"], attention_share_of_step=r["roofline"]["share_of_step"],
                                                      decode_path_roofline_frac=r["decode_path_roofline"]["frac"], gpu_launches=r["gpu_launches"])

    if rank == 0:
        line["clocks"] = sampler.stop()
        if not args.no_cpu_baseline:
            if args.workload == "c2":
                v, n, cores = oracle_attention_sample()
                line["cpu_baseline"] = dict(value=v, unit="attention rows/s", cores=cores, kind="oracle",
                                            sample=f"{n} rows of config 2 (1 prompt group), oracle.attention.attention_row, numpy fp64")
            else:
                v, dt, cores = oracle_rollout_sample(args.workload, cpu_model, cfg, P)
                line["cpu_baseline"] = dict(value=v, unit="tokens/s", cores=cores, kind="oracle",
                                            sample=f"1 decode token of one {args.workload} trajectory at context {P} (oracle.transformer.decode_one, numpy fp64, "
                                                   f"prompt KV drawn at random instead of prefilled), {dt:.1f} s")
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def profile_steps(args):
    """Rollout of the chosen workload through the step calls of the C-ABI; the two steps after --profile-step are the profiled range."""
    import torch
    from paper_2605_30859_b200 import api, workloads as wl
    torch.cuda.set_device(0)
    name = args.workload
    d, model, c, cfg, G, max_new = build_rollout(name, seed=0, max_new=args.max_new, G=args.G, n_layers=args.layers)
    xin = wl.rollout_inputs(name, seed=0, G=G, max_new=max_new)
    toks = torch.from_numpy(np.ascontiguousarray(xin["prompts"])).cuda()
    f_dev = torch.from_numpy(np.ascontiguousarray(xin["forced_len"])).cuda()
    mode = api.MODE_SHORTEST_EARLY_STOP if args.mode == "early" else api.MODE_AUTO
    d.prefill_device(toks, c["P"], xin["Kp"], c["K"], temperature=1.0, seed=7, forced_len_dev=f_dev, mode=mode)
    d.select_and_compact()
    for _ in range(args.profile_step):
        d.decode_step()
        d.select_and_compact()
    n0 = d.n_active()
    torch.cuda.synchronize()
    torch.cuda.profiler.start()
    for _ in range(2):
        d.decode_step()
        d.select_and_compact()
    torch.cuda.synchronize()
    torch.cuda.profiler.stop()
    res = d.results()
    act = res["status"] == 0
    group_of_row = np.repeat(np.arange(G), np.asarray(xin["Kp"]).reshape(-1))
    print(json.dumps(dict(profiled_steps=[args.profile_step + 1, args.profile_step + 2], active_rows=int(n0),
                          mean_suffix_tokens=float(res["len"][act].mean()) if act.any() else 0.0,
                          active_rows_after=int(act.sum()), open_groups_after=int(len(np.unique(group_of_row[act]))), workload=name)))
    d.close()


def reference_arm(args):
    """The tier's reference arm: the oracle as it stands on the host cores, same metric / config, bounded sample per step."""
    rank = int(os.environ.get("RANK", 0))
    if rank != 0:
        return
    import torch
    from paper_2605_30859_b200 import workloads as wl
    name = args.workload
    if name == "c2":
        v, n, cores = oracle_attention_sample()
        print(json.dumps(dict(impl="reference", metric="decode attention rows (generated tokens)/s, one step over all rows", value=v, unit="tokens/s",
                              n_gpus=args.gpus, steps=args.steps, warmup=args.warmup, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64",
                              data="synthetic", config=dict(workload="c2 (sample of rows)"),
                              cpu_baseline=dict(value=v, unit="tokens/s", kind="oracle", cores=cores, sample=f"{n} rows"),
                              e2e=dict(value=v, unit="tokens/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0))))
        return
    c = wl.CONFIGS[name]
    cfg = dict(c["model"])
    if args.layers:
        cfg["n_layers"] = args.layers
    dev = "cuda" if torch.cuda.is_available() else "cpu"      # the device only draws the seeded weights; the oracle runs on the host
    model = wl.make_model(cfg, seed=0, device=dev)
    cpu_model = dict(cfg=model["cfg"], layers=[{k: v.cpu() for k, v in L.items()} for L in model["layers"]],
                     **{k: model[k].cpu() for k in ("embed", "lm_head", "final_norm")})
    del model
    for _ in range(min(args.warmup, 1)):                       # one untimed token pages the weights in
        oracle_rollout_sample(name, cpu_model, cfg, c["P"])
    tok, secs, cores = 0, 0.0, 0
    for _ in range(args.steps):
        v, dt, cores = oracle_rollout_sample(name, cpu_model, cfg, c["P"])
        tok += 1; secs += dt
    v = tok / secs
    sample = f"each step = 1 decode token of one {name} trajectory at context {c['P']} (oracle.transformer.decode_one, numpy fp64)"
    print(json.dumps(dict(impl="reference", metric="rollout generated tokens/s on 1 B200 (K'-of-K early stop)", value=v, unit="tokens/s", n_gpus=args.gpus,
                          steps=args.steps, warmup=args.warmup, ms_per_step=secs / max(1, args.steps) * 1e3, higher_is_better=True, scaling="weak",
                          vs_baseline=None, dtype="f64", data="synthetic", config=dict(workload=f"{name} (bounded sample: {sample})"),
                          cpu_baseline=dict(value=v, unit="tokens/s", kind="oracle", cores=cores, sample=sample),
                          e2e=dict(value=v, unit="tokens/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0))))


if __name__ == "__main__":
    main()
