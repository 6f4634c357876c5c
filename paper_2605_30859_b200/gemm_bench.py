"""Microbenchmark of the projection GEMMs alone on the config-3 shapes.

    python -m paper_2605_30859_b200.gemm_bench [rows,rows,...] [qkv,o,gu,down,lm] [splits: 0 = stream-K kernel, S>=1 = split-K tile kernel]

HBM-cold: the weights rotate through copies that together exceed the 126 MB L2.  The launches are replayed from a CUDA graph so
the Python / ctypes call path does not bound the measurement; time = CUDA events around three replays.  Prints us per GEMM,
weight GB/s and TFLOP/s (2 * rows * N * K)."""
import sys

import torch

from . import api, workloads as wl


def main():
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        d = api.Darts(dict(cfg=dict(wl.CONFIGS["c2"]["model"])), page_size=64, n_pages=64, max_rows=8, max_prompts=2, max_prompt_len=64, max_new=64, stream=st)
    shapes = [("qkv", 6144, 2560), ("o", 2560, 4096), ("gu", 19456, 2560), ("down", 2560, 9728), ("lm", 151936, 2560)]
    rows_list = [int(x) for x in (sys.argv[1] if len(sys.argv) > 1 else "16,128,256,512").split(",")]
    sp = [int(x) for x in sys.argv[3].split(",")] if len(sys.argv) > 3 else [0]
    splits = {k: sp for k in ("qkv", "o", "gu", "down", "lm")}
    only = sys.argv[2].split(",") if len(sys.argv) > 2 else None
    for name, N, K in shapes:
        if only and name not in only:
            continue
        ncopy = max(2, int(400e6 // (N * K * 2)) + 1)
        Ws = [(torch.randn(N, K, device="cuda") * 0.02).to(torch.bfloat16) for _ in range(ncopy)]
        for rows in rows_list:
            X = torch.randn(rows, K, device="cuda").to(torch.bfloat16)
            for S in splits[name]:
                scratch = torch.empty((S if S else 16) * rows * N, dtype=torch.float32, device="cuda")
                torch.cuda.synchronize()
                with torch.cuda.stream(st):
                    for i in range(2):
                        d.debug_gemm_bf16(X, Ws[i % ncopy], split_k=S, scratch=scratch, reduce=False)
                torch.cuda.synchronize()
                n = 2 * ncopy
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=st):
                    for i in range(n):
                        d.debug_gemm_bf16(X, Ws[i % ncopy], split_k=S, scratch=scratch, reduce=False)
                g.replay()
                torch.cuda.synchronize()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                for _ in range(3):
                    g.replay()
                b.record()
                torch.cuda.synchronize()
                us = a.elapsed_time(b) * 1e3 / (3 * n)
                print(f"{name:5s} N={N:6d} K={K:5d} rows={rows:4d} S={S:2d}  {us:8.2f} us  {N*K*2/us/1e3:7.1f} GB/s  {2*rows*N*K/us/1e6:7.1f} TF/s", flush=True)
                del g
        del Ws
    d.close()


if __name__ == "__main__":
    main()
