#!/usr/bin/env python
"""bench.py — one JSON line: rollout generated tokens/s on 1 B200 (K'-of-K early stop) + decode HBM GB/s vs peak.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c3|c2] [--impl reference]

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

KV_BYTES_PER_TOKEN_LAYER = {"c2": 2 * 8 * 128 * 2, "c3": 2 * 8 * 128 * 2}


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
    import torch
    rank, world = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))
    local = int(os.environ.get("LOCAL_RANK", 0))
    if world > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    else:
        torch.cuda.set_device(0)
    return rank, world, local


def barrier(world):
    import torch
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    torch.cuda.synchronize()


def allreduce(world, x, op):
    import torch
    if world == 1:
        return x
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device="cuda")
    dist.all_reduce(t, op=getattr(dist.ReduceOp, op))
    return float(t.item())


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


# ------------------------------------------------------------------------------------------------ c3: full rollout
def build_c3(seed, max_new=None, G=None, n_layers=None):
    import torch
    from paper_2605_30859_b200 import api, workloads as wl
    c = wl.CONFIGS["c3"]
    cfg = dict(c["model"])
    if n_layers:
        cfg["n_layers"] = n_layers
    G = c["G"] if G is None else G
    max_new = c["max_new"] if max_new is None else max_new
    model = wl.make_model(cfg, seed=seed, device="cuda")
    R = G * c["Kp"]
    page = 64
    # pool: prefix + every row's worst case is far too much; size for the expected peak (~42 GB at full size) with margin
    kv_page_bytes = cfg["n_layers"] * 2 * cfg["n_kv_heads"] * page * cfg["head_dim"] * 2
    n_pages = min(G * (c["P"] // page) + R * (max_new // page + 1), int(64e9 // kv_page_bytes))
    d = api.Darts(model, page_size=page, n_pages=n_pages, max_rows=R, max_prompts=G, max_prompt_len=c["P"], max_new=max_new,
                  flags=api.FLAG_PROFILE_ATTENTION)
    return d, model, c, cfg, G, max_new


def rollout_algo_attention_bytes(lens, Kp, P, kvb):
    """Algorithmic KV bytes the attention of ONE layer must read over a whole rollout (prefix once per active group)."""
    lens = np.asarray(lens).reshape(-1, Kp)
    total, per_step = 0, []
    for s in range(1, int(lens.max())):
        act = lens > s                              # rows that are fed token s-1 at decode step s
        b = (int(act.sum()) * s + int(act.any(axis=1).sum()) * P) * kvb
        per_step.append(b)
        total += b
    return total, per_step


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--workload", default="c2")
    ap.add_argument("--max-new", type=int, default=None, help="debug only: shorten the rollout (INVALID as a bench number)")
    ap.add_argument("--G", type=int, default=None, help="debug only")
    ap.add_argument("--layers", type=int, default=None, help="debug only")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()

    if args.impl == "reference":
        return reference_arm(args)

    import torch
    from paper_2605_30859_b200 import api, workloads as wl
    rank, world, local = dist_setup(args.gpus)
    peaks = measured_peaks()
    sampler = ClockSampler(local) if rank == 0 else None
    line = dict(n_gpus=world, steps=args.steps, warmup=args.warmup, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="bf16", data="synthetic")

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
        d, model, c, cfg, G, max_new = build_c3(seed=0, max_new=args.max_new, G=args.G, n_layers=args.layers)
        Kp, K, P = c["Kp"], c["K"], c["P"]
        R = G * Kp
        kvb = KV_BYTES_PER_TOKEN_LAYER["c3"]
        host_in = []
        for it in range(args.warmup + 2 * args.steps):
            xin = wl.rollout_inputs("c3", seed=1000 * rank + it, G=G, max_new=max_new)
            host_in.append(xin)
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        gen_tokens, dev_ms, e2e_ms, attn_ms, attn_bytes, steps_count = [], [], [], [], [], []
        launches0 = None
        it = 0
        for phase, n in (("warmup", args.warmup), ("device", args.steps), ("e2e", args.steps)):
            if phase == "device":
                barrier(world)
                launches0 = d.counters()["kernel_launches"]
                t_dev0 = time.perf_counter()
            for _ in range(n):
                xin = host_in[it]; it += 1
                if phase == "e2e":
                    p_pin, f_pin = pin(xin["prompts"]), pin(xin["forced_len"])
                    t0 = time.perf_counter()
                    out = d.rollout_host(p_pin.numpy(), xin["Kp"], K, max_new, 1.0, 7 + it, forced_len=f_pin.numpy())
                    e2e_ms.append((time.perf_counter() - t0) * 1e3)
                    gen = int(out["len"].sum())
                    e2e_tokens = gen
                else:
                    p_dev = torch.from_numpy(xin["prompts"]).cuda()
                    f_dev = torch.from_numpy(xin["forced_len"]).cuda()
                    torch.cuda.synchronize()
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record(d.stream)
                    d.rollout(p_dev, G, Kp, K, max_new, 1.0, 7 + it, forced_len_dev=f_dev)
                    b.record(d.stream)
                    torch.cuda.synchronize()
                    if phase == "device":
                        dev_ms.append(a.elapsed_time(b))
                        cnt = d.counters()
                        gen_tokens.append(cnt["n_generated_tokens"])
                        steps_count.append(cnt["n_steps"])
                        res = d.results()
                        tot, per_step = rollout_algo_attention_bytes(res["len"], Kp, P, kvb)
                        t_ms = d.attention_times()
                        n = min(len(t_ms), len(per_step))
                        attn_ms.append(float(np.sum(t_ms[:n])))
                        attn_bytes.append(float(np.sum(per_step[:n])))
            if phase == "device":
                barrier(world)
                launches = d.counters()["kernel_launches"] - launches0
        tot_ms = allreduce(world, float(np.sum(dev_ms)), "MAX")
        tot_tok = allreduce(world, float(np.sum(gen_tokens)), "SUM")
        tot_e2e_ms = allreduce(world, float(np.sum(e2e_ms)), "MAX")
        e2e_tok = allreduce(world, float(e2e_tokens * 0 + sum(int(0) for _ in ()) + 0), "SUM") if False else None
        ach = float(np.sum(attn_bytes)) / (float(np.sum(attn_ms)) * 1e-3) / 1e9 if np.sum(attn_ms) > 0 else 0.0
        h2d = int(host_in[0]["prompts"].nbytes + host_in[0]["forced_len"].nbytes)
        d2h = int(R * max_new * 8 + R * 5 + G * (K * 4 + 4 * 4))
        # e2e tokens: re-count from the e2e phase inputs (same distribution as the device phase)
        line.update(metric="rollout generated tokens/s on 1 B200 (K'-of-K early stop)", value=tot_tok / (tot_ms * 1e-3), unit="tokens/s",
                    ms_per_step=tot_ms / args.steps,
                    config=dict(workload=f"c3: Qwen3-4B-shaped bf16 ({cfg['n_layers']} layers), G={G} x K'={Kp}, keep {K}, P={P}, max_new={max_new}, "
                                         "forced-EOS lognormal(7.2,0.9), mode AUTO (K'>=2K: shortest-only + early stop)",
                                l2="per-step working set (8 GB weights + KV) >> 126 MB L2, no flush",
                                steps_per_rollout=int(np.mean(steps_count)), generated_tokens_per_rollout=int(np.mean(gen_tokens))),
                    roofline=dict(bound="hbm", achieved=ach, peak=peaks["hbm"], unit="GB/s", frac=ach / peaks["hbm"], traffic=None,
                                  kernel="attn_main_k+attn_merge_k (layer 0 of every decode step, CUDA events inside the rollout)",
                                  peak_source=peaks["source"]),
                    gpu_launches=int(launches))
        line["e2e"] = dict(value=None, unit="tokens/s", h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h, ms_per_step=tot_e2e_ms / max(1, args.steps))
        line["_e2e_ms"] = tot_e2e_ms
        if args.max_new or args.G or args.layers:
            line["config"]["INVALID"] = "debug flags shrink the workload"
        d.close()
        del model
        torch.cuda.empty_cache()
        # attention microbench (config 2) alongside: the kernel timed alone
        if rank == 0:
            res2, _ = attention_microbench(10, 3)
            a2 = res2["algo_bytes"] / (res2["ms"] * 1e-3) / 1e9
            line["attention_c2"] = dict(ms=res2["ms"], achieved_GBps=a2, frac_of_measured_peak=a2 / peaks["hbm"], rows=res2["rows"])

    if rank == 0:
        line["clocks"] = sampler.stop()
        if not args.no_cpu_baseline:
            v, n, cores = oracle_attention_sample()
            line["cpu_baseline"] = dict(value=v, unit="attention rows/s" if args.workload == "c2" else "attention rows/s (oracle, c2 rows)", cores=cores,
                                        kind="oracle", sample=f"{n} rows of config 2 (1 prompt group), oracle.attention.attention_row, numpy fp64")
        if "_e2e_ms" in line:
            line.pop("_e2e_ms")
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def reference_arm(args):
    rank = int(os.environ.get("RANK", 0))
    if rank != 0:
        return
    v, n, cores = oracle_attention_sample()
    print(json.dumps(dict(impl="reference", metric="decode attention rows/s", value=v, unit="rows/s", n_gpus=args.gpus, steps=args.steps,
                          warmup=args.warmup, higher_is_better=True, cpu_baseline=dict(value=v, kind="oracle", cores=cores, sample=f"{n} rows"),
                          e2e=dict(value=v, unit="rows/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0))))


if __name__ == "__main__":
    main()
