"""Microbenchmark of the split-KV attention pair (attn_main_k + attn_merge_k) at a FEW live rows — the
tail of a long rollout, where the pair is bound by its two kernel boundaries and not by HBM (DESIGN.md 9 (4c)).

    [DARTS_SKIP=4|8|12] [DARTS_NO_PDL=1] python -m paper_2605_30859_b200.attn_bench [G:Kp:suffix,...]

Config-2 head geometry (32 q / 8 kv heads, head_dim 128, page 64), one 1024-token shared prefix per group, every row with the
same suffix length.  Prints, per case, the time of ONE call between two CUDA events on the library's stream and the time per
call of 20 back-to-back calls (the launch path amortised, the PDL chain as inside a decode step), the same 20 calls replayed from a
CUDA graph (no host launch path: the GPU-side cost alone), with the KV bytes of the call.
DARTS_SKIP=4 drops attn_main_k, 8 drops attn_merge_k (include/darts.h): what is left is the cost of the other kernel alone."""
import os
import sys

import numpy as np
import torch

from . import api, workloads as wl


def main():
    cases = sys.argv[1] if len(sys.argv) > 1 else "1:1:64,1:1:8000,1:1:15000,1:4:8000,16:4:2000"
    tag = "skip=%s pdl=%s" % (os.environ.get("DARTS_SKIP", "0"), "off" if os.environ.get("DARTS_NO_PDL") else "on")
    page = 64
    kvb = 2 * 8 * 128 * 2
    st = torch.cuda.Stream()
    torch.cuda.set_stream(st)                       # graph capture needs a non-default stream; the library launches on this one
    for case in cases.split(","):
        G, Kp, suf = (int(v) for v in case.split(":"))
        x = wl.attention_inputs("c2", seed=1, device="cuda", G=G, Kp=Kp, suffix=dict(kind="lognormal", mu=0.0, sigma=0.1, lo=suf, hi=suf))
        P, R = x["P"], x["R"]
        n_pages = G * (P // page) + int(np.sum((x["suffix_len"] + page - 1) // page)) + 8
        d = api.Darts(dict(cfg=dict(wl.CONFIGS["c2"]["model"])), page_size=page, n_pages=max(n_pages, 2 * R + 16), max_rows=R, max_prompts=G,
                      max_prompt_len=P, max_new=16384, flags=0)
        d.attn_load(G, P, x["Kp"], x["k_prefix"], x["v_prefix"], x["suffix_len"], x["k_suffix"], x["v_suffix"])
        out = torch.empty_like(x["q"])
        for _ in range(5):
            d.attention(x["q"], out)
        torch.cuda.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(50)]
        for a, b in ev:
            a.record(d.stream)
            d.attention(x["q"], out)
            b.record(d.stream)
        torch.cuda.synchronize()
        single = float(np.median([a.elapsed_time(b) for a, b in ev])) * 1e3
        for a, b in ev[:20]:
            a.record(d.stream)
            for _ in range(20):
                d.attention(x["q"], out)
            b.record(d.stream)
        torch.cuda.synchronize()
        chained = float(np.median([a.elapsed_time(b) for a, b in ev[:20]])) * 1e3 / 20
        # the same 20 calls replayed from a CUDA graph: no host launch path at all — what the GPU alone needs per pair
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            for _ in range(20):
                d.attention(x["q"], out)
        g.replay()
        torch.cuda.synchronize()
        a, b = ev[0]
        a.record(st)
        for _ in range(5):
            g.replay()
        b.record(st)
        torch.cuda.synchronize()
        graph = a.elapsed_time(b) * 1e3 / 100
        del g
        mb = (int(x["suffix_len"].sum()) + G * P) * kvb / 1e6
        print(f"{tag}: G={G} Kp={Kp} suffix={suf} ({mb:.1f} MB of KV): single {single:.1f} us, chained {chained:.1f} us per call "
              f"({mb / chained:.2f} TB/s), graph replay {graph:.1f} us per call ({mb / graph:.2f} TB/s)", flush=True)
        d.close()
        del x, d


if __name__ == "__main__":
    main()
