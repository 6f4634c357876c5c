"""Seeded synthetic inputs shaped like BASELINE.json's configs (serves BOTH the CUDA path
and the oracle; holds none of the method's arithmetic — only random draws and shapes).

Recipe:
  weights   N(0, 0.02^2); norm weights 1 (parity tests: 1 + N(0, 0.2^2), `norm_std`); MoE router N(0, 1/d_model) so router logits of a
            unit-RMS hidden are ~N(0,1) (BASELINE.json c5 "router logits N(0,1)")
  prompts   uniform ints in [0, V-2]  (eos_id = V-1 never appears in a prompt)
  forced    forced-EOS length of trajectory (i,j) = round(lognormal(mu, sigma)) clipped to
            [lo, hi]; c4 uses the 80/20 two-component mixture; values > max_new never fire,
            so those rows run into the length limit (TRUNC)
  Kp        per-prompt K' (c4: uniform over {8,12,16})
  c2        Q, prefix K/V, per-row suffix K/V ~ N(0,1) in bf16; suffix lengths lognormal(7.0, 0.8)
            clipped to [16, 8192]
The paper's measured length distributions (DAPO-MATH with trained Qwen models,
PAPER.md:238, Fig. 1/3) are not in this container; these lognormal draws stand in for them
(tail 5-10x the median).

Everything is drawn with torch generators seeded from (seed, tag); a tensor drawn on
`device` is the single source of truth and the oracle receives a host copy of the same bits.
"""
import math
import zlib

import numpy as np
import torch

CONFIGS = {
    # BASELINE.json configs[0]
    "c1": dict(model=dict(n_layers=2, d_model=128, n_q_heads=4, n_kv_heads=2, head_dim=32, ffn=256,
                          vocab=512, n_experts=0, top_k=0, expert_ffn=0, qk_norm=False,
                          rope_theta=1.0e6, rms_eps=1.0e-6, dtype="f32"),
               G=4, P=32, Kp=8, K=4, max_new=64, temperature=1.0,
               forced=dict(kind="lognormal", mu=3.0, sigma=0.6, lo=4, hi=64)),
    # BASELINE.json configs[1]: attention-only microbench
    "c2": dict(model=dict(n_layers=1, d_model=4096, n_q_heads=32, n_kv_heads=8, head_dim=128, ffn=0,
                          vocab=0, n_experts=0, top_k=0, expert_ffn=0, qk_norm=False,
                          rope_theta=1.0e6, rms_eps=1.0e-6, dtype="bf16"),
               G=128, P=1024, Kp=16, page=64,
               suffix=dict(kind="lognormal", mu=7.0, sigma=0.8, lo=16, hi=8192)),
    # BASELINE.json configs[2]: Qwen3-4B-shaped
    "c3": dict(model=dict(n_layers=36, d_model=2560, n_q_heads=32, n_kv_heads=8, head_dim=128, ffn=9728,
                          vocab=151936, n_experts=0, top_k=0, expert_ffn=0, qk_norm=False,
                          rope_theta=1.0e6, rms_eps=1.0e-6, dtype="bf16"),
               G=32, P=512, Kp=16, K=8, max_new=8192, temperature=1.0,
               forced=dict(kind="lognormal", mu=7.2, sigma=0.9, lo=1, hi=1 << 30)),
    # BASELINE.json configs[3]: Qwen3-8B-shaped
    "c4": dict(model=dict(n_layers=36, d_model=4096, n_q_heads=32, n_kv_heads=8, head_dim=128, ffn=12288,
                          vocab=151936, n_experts=0, top_k=0, expert_ffn=0, qk_norm=False,
                          rope_theta=1.0e6, rms_eps=1.0e-6, dtype="bf16"),
               G=64, P=1024, Kp=(8, 12, 16), K=8, max_new=16384, temperature=1.0,
               forced=dict(kind="mixture", w=(0.8, 0.2), mu=(7.0, 8.8), sigma=(0.7, 0.5), lo=1, hi=1 << 30)),
    # BASELINE.json configs[4]: Qwen3-30B-A3B-shaped MoE
    "c5": dict(model=dict(n_layers=48, d_model=2048, n_q_heads=32, n_kv_heads=4, head_dim=128, ffn=0,
                          vocab=151936, n_experts=128, top_k=8, expert_ffn=768, qk_norm=False,
                          rope_theta=1.0e6, rms_eps=1.0e-6, dtype="bf16"),
               G=16, P=768, Kp=12, K=8, max_new=16384, temperature=1.0,
               forced=dict(kind="lognormal", mu=7.5, sigma=1.0, lo=1, hi=1 << 30)),
}


def _gen(seed, tag, device="cpu"):
    g = torch.Generator(device=device)
    g.manual_seed((int(seed) * 1000003 + zlib.crc32(tag.encode())) & 0x7FFFFFFFFFFFFFFF)
    return g


def _normal(shape, std, seed, tag, dtype, device):
    g = _gen(seed, tag, device)
    x = torch.empty(shape, dtype=torch.float32, device=device)
    x.normal_(0.0, std, generator=g)
    return x.to(dtype).contiguous()


def _gamma(n, norm_std, seed, tag, dtype, device):
    """RMSNorm weight: ones (the configs' recipe) or 1 + N(0, norm_std^2) with its own stream per tensor."""
    if not norm_std:
        return torch.ones(n, dtype=dtype, device=device)
    return (1.0 + _normal((n,), norm_std, seed, tag, torch.float32, device)).to(dtype).contiguous()


def make_model(cfg, seed=0, device="cpu", std=0.02, norm_std=0.0):
    """Random-init weights as torch tensors on `device` (the CUDA path borrows their pointers).
    Layout: every projection is [out_features, in_features] row-major.
    norm_std > 0 draws every RMSNorm weight (attn / mlp / final / q / k, one stream per layer and tensor) from
    1 + N(0, norm_std^2) instead of the recipe's ones: the parity tests use it so that a kernel that drops or
    mis-indexes a norm weight cannot pass."""
    dt = torch.float32 if cfg["dtype"] == "f32" else torch.bfloat16
    d, Hq, Hkv, hd = cfg["d_model"], cfg["n_q_heads"], cfg["n_kv_heads"], cfg["head_dim"]
    V, E = cfg["vocab"], cfg["n_experts"]
    m = dict(cfg=dict(cfg), layers=[])
    if V:
        m["embed"] = _normal((V, d), std, seed, "embed", dt, device)
        m["lm_head"] = _normal((V, d), std, seed, "lm_head", dt, device)
        m["final_norm"] = _gamma(d, norm_std, seed, "final_norm", dt, device)
    for l in range(cfg["n_layers"]):
        L = dict(attn_norm=_gamma(d, norm_std, seed, f"attn_norm{l}", dt, device),
                 mlp_norm=_gamma(d, norm_std, seed, f"mlp_norm{l}", dt, device),
                 wqkv=_normal(((Hq + 2 * Hkv) * hd, d), std, seed, f"wqkv{l}", dt, device),
                 wo=_normal((d, Hq * hd), std, seed, f"wo{l}", dt, device))
        if cfg.get("qk_norm"):
            L["q_norm"] = _gamma(hd, norm_std, seed, f"q_norm{l}", dt, device)
            L["k_norm"] = _gamma(hd, norm_std, seed, f"k_norm{l}", dt, device)
        if E == 0 and cfg["ffn"]:
            L["wgu"] = _normal((2 * cfg["ffn"], d), std, seed, f"wgu{l}", dt, device)
            L["wd"] = _normal((d, cfg["ffn"]), std, seed, f"wd{l}", dt, device)
        elif E:
            F = cfg["expert_ffn"]
            L["wr"] = _normal((E, d), 1.0 / math.sqrt(d), seed, f"wr{l}", torch.float32, device)
            L["wgu_e"] = _normal((E, 2 * F, d), std, seed, f"wgu_e{l}", dt, device)
            L["wd_e"] = _normal((E, d, F), std, seed, f"wd_e{l}", dt, device)
        m["layers"].append(L)
    return m


class HostWeights:
    """Lazy host view of a torch tensor for the oracle: converted to float64 only when used
    (np.asarray(w, dtype=float64) or w[index]) so a 4B-parameter model fits in host memory."""

    def __init__(self, t, lazy=False):
        # lazy: leave the tensor where it is (e.g. a 60 GB MoE model in HBM) and copy only what is indexed
        self.t = t.detach() if lazy else t.detach().cpu()
        self.shape = tuple(self.t.shape)

    def __array__(self, dtype=None, copy=None):
        return self.t.to(torch.float64).cpu().numpy()          # exact widening where the tensor lives, then one copy

    def __getitem__(self, idx):
        if isinstance(idx, np.ndarray):
            idx = torch.from_numpy(idx.astype(np.int64)).to(self.t.device)
        return self.t[idx].to(torch.float64).cpu().numpy()

    def __len__(self):
        return self.shape[0]


def host_model(m, lazy=False):
    """The same weights as `make_model` returned, as host arrays the oracle can consume (lazy: device-backed views)."""
    def conv(v):
        return HostWeights(v, lazy) if torch.is_tensor(v) else v
    out = dict(cfg=dict(m["cfg"]), layers=[{k: conv(v) for k, v in L.items()} for L in m["layers"]])
    for k in ("embed", "lm_head", "final_norm"):
        if k in m:
            out[k] = conv(m[k])
    return out


def make_prompts(G, P, V, seed=0):
    g = _gen(seed, "prompts")
    return torch.randint(0, V - 1, (G, P), generator=g, dtype=torch.int64).to(torch.int32).numpy()


def make_Kp(G, spec, seed=0):
    if isinstance(spec, int):
        return np.full(G, spec, dtype=np.int32)
    g = _gen(seed, "Kp")
    idx = torch.randint(0, len(spec), (G,), generator=g).numpy()
    return np.asarray(spec, dtype=np.int32)[idx]


def _lognormal(n, mu, sigma, g):
    return torch.exp(mu + sigma * torch.randn(n, generator=g, dtype=torch.float64))


def make_lengths(n, spec, seed=0, tag="forced"):
    """n seeded long-tail lengths (int32) per `spec` (kind lognormal | mixture)."""
    g = _gen(seed, tag)
    if spec["kind"] == "lognormal":
        x = _lognormal(n, spec["mu"], spec["sigma"], g)
    else:
        comp = torch.rand(n, generator=g, dtype=torch.float64) >= spec["w"][0]
        a = _lognormal(n, spec["mu"][0], spec["sigma"][0], g)
        b = _lognormal(n, spec["mu"][1], spec["sigma"][1], g)
        x = torch.where(comp, b, a)
    x = torch.clamp(torch.round(x), spec["lo"], spec["hi"])
    return x.to(torch.int32).numpy()


def make_forced_len(Kp, spec, seed=0):
    """forced_len[G, Kp_max] int32 (entries beyond Kp[i] are 0 and unused)."""
    G, Kmax = len(Kp), int(max(Kp))
    flat = make_lengths(G * Kmax, spec, seed).reshape(G, Kmax)
    for i in range(G):
        flat[i, Kp[i]:] = 0
    return flat


def rollout_inputs(name, seed=0, G=None, max_new=None):
    """Prompts, Kp, forced_len and scalars of a rollout config (model built separately)."""
    c = CONFIGS[name]
    G = c["G"] if G is None else G
    V = c["model"]["vocab"]
    Kp = make_Kp(G, c["Kp"], seed)
    return dict(prompts=make_prompts(G, c["P"], V, seed), Kp=Kp, K=c["K"],
                max_new=c["max_new"] if max_new is None else max_new,
                temperature=c["temperature"], forced_len=make_forced_len(Kp, c["forced"], seed),
                eos_id=V - 1)


def attention_inputs(name="c2", seed=0, G=None, device="cpu", P=None, Kp=None, suffix=None):
    """Config-2 inputs: q [R,Hq,hd], prefix K/V [G,P,Hkv,hd], suffix lengths [R], and packed
    suffix K/V [sum t, Hkv, hd] with row offsets; bf16 N(0,1)."""
    c = CONFIGS[name]
    m = c["model"]
    G = c["G"] if G is None else G
    P = c["P"] if P is None else P
    Kp = c["Kp"] if Kp is None else Kp
    R = G * Kp
    Hq, Hkv, hd = m["n_q_heads"], m["n_kv_heads"], m["head_dim"]
    t = make_lengths(R, c["suffix"] if suffix is None else suffix, seed, "suffix")
    offs = np.concatenate([[0], np.cumsum(t)]).astype(np.int64)
    bf = torch.bfloat16
    return dict(G=G, P=P, Kp=Kp, R=R, suffix_len=t, suffix_offs=offs,
                q=_normal((R, Hq, hd), 1.0, seed, "q", bf, device),
                k_prefix=_normal((G, P, Hkv, hd), 1.0, seed, "kp", bf, device),
                v_prefix=_normal((G, P, Hkv, hd), 1.0, seed, "vp", bf, device),
                k_suffix=_normal((int(offs[-1]), Hkv, hd), 1.0, seed, "ks", bf, device),
                v_suffix=_normal((int(offs[-1]), Hkv, hd), 1.0, seed, "vs", bf, device))
