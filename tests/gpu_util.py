"""Helpers shared by the -m gpu tests: build a context for a config, run the oracle teacher-forced."""
import numpy as np

from paper_2605_30859_b200 import workloads as wl


def make_ctx(cfg, seed, G, Kp_max, P, max_new, page=16, flags=0, n_pages=None, std=0.02, norm_std=0.0):
    from paper_2605_30859_b200 import api
    model_cpu = wl.make_model(cfg, seed=seed, std=std, norm_std=norm_std)
    model_gpu = dict(cfg=model_cpu["cfg"], layers=[{k: v.cuda() for k, v in L.items()} for L in model_cpu["layers"]])
    for k in ("embed", "lm_head", "final_norm"):
        model_gpu[k] = model_cpu[k].cuda()
    R = G * Kp_max
    if n_pages is None:
        n_pages = G * ((P + page - 1) // page) + R * ((max_new + page - 1) // page + 1)
    d = api.Darts(model_gpu, page_size=page, n_pages=n_pages, max_rows=R, max_prompts=G, max_prompt_len=P, max_new=max_new, flags=flags)
    return d, wl.host_model(model_cpu)


def rel_inf(a, b):
    """||a-b||_inf / ||b||_inf (the logit error metric)."""
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))
