"""Pre-norm GQA decoder in float64 (oracle; test infrastructure only).

The paper defines no model ("Qwen-series models", §5.1); the
architecture is fixed by BASELINE.json's configs ("RMSNorm, RoPE, SwiGLU", GQA
head counts, top-8 MoE) and DESIGN.md R5:

  h_0      = E[token]
  a        = rmsnorm(h, w_attn_norm)                 rmsnorm(x)_k = x_k w_k / sqrt(mean(x^2)+eps)
  q,k,v    = split(a Wqkv^T)                         rows of Wqkv: Hq q-heads, Hkv k-heads, Hkv v-heads
  q,k      = rope(headnorm(q)), rope(headnorm(k))    headnorm only if the model has q_norm/k_norm
  o        = softmax(q K^T / sqrt(hd)) V             q-head h reads kv-head h // (Hq/Hkv), causal
  h        = h + o Wo^T
  b        = rmsnorm(h, w_mlp_norm)
  dense:   m = (silu(b Wg^T) * (b Wu^T)) Wd^T        Wgu = [Wg ; Wu] stacked on rows
  moe:     p = softmax(b Wr^T); top-k by p (ties -> lower expert id); w = p_top / sum(p_top)
           m = sum_e w_e expert_e(b)
  h        = h + m
  logits   = rmsnorm(h_L, w_final_norm) Wlm^T

RoPE: rotate-half pairing (i, i+hd/2), angle = pos * theta^(-2i/hd).

A model is a dict (built by the seeded generator in paper_2605_30859_b200.workloads,
which holds no arithmetic of the method):
  cfg: n_layers, d_model, n_q_heads, n_kv_heads, head_dim, ffn, vocab,
       n_experts, top_k, expert_ffn, qk_norm, rope_theta, rms_eps
  embed [V,d]  final_norm [d]  lm_head [V,d]
  layers[l]: attn_norm [d]  wqkv [(Hq+2Hkv)hd, d]  (q_norm, k_norm [hd])  wo [d, Hq hd]
             mlp_norm [d]   dense: wgu [2 ffn, d], wd [d, ffn]
                            moe:   wr [E, d], wgu_e [E, 2 effn, d], wd_e [E, d, effn]
Arrays may be float32 / bf16-valued float32 / float64; every product is taken
after up-casting to float64 ("the oracle up-casts the same bits and computes
un-rounded in double").

Two entry points:
  forward_full(model, tokens)         the definition: one causal pass over a whole sequence.
  prefill / decode_one                the incremental form the rollout uses, over an explicit
                                      per-row KV list (never shared between rows).
Pin: tests check decode_one position-by-position against forward_full, attention
against torch float64 SDPA, and the special cases listed in oracle/__init__.py.
"""
import numpy as np


def f64(x):
    return np.asarray(x, dtype=np.float64)


# Matched-rounding debug mode (SURVEY.md 8(c) "precision contract": "a second matched-rounding oracle mode that rounds to bf16 at
# the GPU's documented rounding points").  ROUND = None (default): the un-rounded definition, nothing below changes a value.
# ROUND = callable(name, array) -> array: applied where the bf16 CUDA path rounds an input of a tensor-core product
# ("rounding points"): "xn" the normed hidden fed to QKV, "q" / "k" / "v" after RoPE (k, v as stored in the cache),
# "p" the un-normalised attention probabilities exp(s - max) fed to P.V (the denominator sums the un-rounded ones), "ao" the
# attention output fed to Wo, "xn2" the normed hidden fed to the MLP / the experts (the MoE router reads the un-rounded one),
# "act" silu(g) * u fed to Wd, "xnf" the final normed hidden fed to the LM head.  It answers "how far is an ideal bf16 pipeline
# from the definition on this model", which no kernel can beat; the parity tolerance is still stated against the definition.
ROUND = None


def _r(name, x):
    return x if ROUND is None else ROUND(name, x)


def rmsnorm(x, w, eps):
    x = f64(x)
    return x * f64(w) / np.sqrt(np.mean(x * x, axis=-1, keepdims=True) + eps)


def rope(x, pos, theta):
    """x [..., T, H, hd] rotated at integer positions pos [T]."""
    x = f64(x)
    hd = x.shape[-1]
    half = hd // 2
    i = np.arange(half, dtype=np.float64)
    inv_freq = theta ** (-2.0 * i / hd)
    ang = f64(pos)[:, None] * inv_freq[None, :]            # [T, half]
    cos, sin = np.cos(ang)[:, None, :], np.sin(ang)[:, None, :]
    x1, x2 = x[..., :half], x[..., half:]
    return np.concatenate([x1 * cos - x2 * sin, x2 * cos + x1 * sin], axis=-1)


def softmax(z, axis=-1):
    z = f64(z)
    z = z - np.max(z, axis=axis, keepdims=True)
    e = np.exp(z)
    return e / np.sum(e, axis=axis, keepdims=True)


def silu(x):
    return x / (1.0 + np.exp(-x))


def attention_one(q, K, V, n_kv_heads):
    """One query position.  q [Hq, hd]; K, V [T, Hkv, hd] (all keys visible).  Returns [Hq, hd]."""
    q, K, V = f64(q), f64(K), f64(V)
    Hq, hd = q.shape
    rep = Hq // n_kv_heads
    out = np.empty((Hq, hd))
    for h in range(Hq):
        g = h // rep
        s = K[:, g, :] @ q[h] / np.sqrt(hd)                 # [T]
        if ROUND is None:
            p = softmax(s)
            out[h] = p @ V[:, g, :]
        else:                                               # matched rounding: rounded numerator, un-rounded denominator
            e = np.exp(s - np.max(s))
            out[h] = (ROUND("p", e) @ V[:, g, :]) / np.sum(e)
    return out


def qkv_project(layer, cfg, a, pos):
    """a [T, d] -> q [T,Hq,hd], k [T,Hkv,hd], v [T,Hkv,hd], q/k rotated at pos."""
    Hq, Hkv, hd = cfg["n_q_heads"], cfg["n_kv_heads"], cfg["head_dim"]
    T = a.shape[0]
    qkv = a @ f64(layer["wqkv"]).T
    q = qkv[:, : Hq * hd].reshape(T, Hq, hd)
    k = qkv[:, Hq * hd: (Hq + Hkv) * hd].reshape(T, Hkv, hd)
    v = qkv[:, (Hq + Hkv) * hd:].reshape(T, Hkv, hd)
    if cfg.get("qk_norm", False):
        q = rmsnorm(q, layer["q_norm"], cfg["rms_eps"])
        k = rmsnorm(k, layer["k_norm"], cfg["rms_eps"])
    q = rope(q, pos, cfg["rope_theta"])
    k = rope(k, pos, cfg["rope_theta"])
    return _r("q", q), _r("k", k), _r("v", v)


# DESIGN.md R13: when this is a list, every routing decision appends the probability gap between the
# k-th and (k+1)-th expert (tests use it to set aside rows whose discrete expert choice is a near-tie).
# Pure instrumentation: it does not change any value computed here.
ROUTER_GAPS = None

# DESIGN.md R13, teacher-forced routing (the analogue of teacher-forced tokens, R12): when ROUTE_OVERRIDE is an iterator,
# every routing decision takes its expert ids from it (in call order: forward_full walks layers, then positions) instead of
# from its own top-k; the gates are still this oracle's probabilities renormalised over those experts.  When ROUTE_REGRET is a
# list, each such decision appends max p(own choice not taken) - min p(forced choice not own): 0 when the two sets agree, else how
# far, in probability, the forced set is from being the top-k.  Both None: nothing changes.
ROUTE_OVERRIDE = None
ROUTE_REGRET = None


def moe_route(layer, cfg, b):
    """b [d] -> (expert ids [top_k] in selection order, weights [top_k] summing to 1)."""
    p = softmax(f64(layer["wr"]) @ b)
    # top-k by p, ties -> lower expert id: stable sort of -p keeps lower ids first
    order = np.argsort(-p, kind="stable")[: cfg["top_k"]]
    if ROUTER_GAPS is not None and cfg["top_k"] < len(p):
        ps = np.sort(p)[::-1]
        ROUTER_GAPS.append(float(ps[cfg["top_k"] - 1] - ps[cfg["top_k"]]))
    if ROUTE_OVERRIDE is not None:
        forced = np.asarray(next(ROUTE_OVERRIDE), dtype=np.int64)
        assert forced.shape == order.shape and len(set(forced.tolist())) == len(forced) and forced.min() >= 0 and forced.max() < len(p)
        if ROUTE_REGRET is not None:
            own, frc = set(order.tolist()), set(forced.tolist())
            ROUTE_REGRET.append(0.0 if own == frc else float(max(p[list(own - frc)]) - min(p[list(frc - own)])))
        order = forced
    w = p[order] / np.sum(p[order])
    return order, w


def mlp(layer, cfg, b):
    """b [T, d] -> m [T, d]."""
    br = _r("xn2", b)                                        # == b unless the matched-rounding mode is on
    if cfg.get("n_experts", 0) == 0:
        F = cfg["ffn"]
        gu = br @ f64(layer["wgu"]).T
        return _r("act", silu(gu[:, :F]) * gu[:, F:]) @ f64(layer["wd"]).T
    F = cfg["expert_ffn"]
    out = np.zeros_like(b)
    for t in range(b.shape[0]):
        ids, w = moe_route(layer, cfg, b[t])                 # the router always sees the un-rounded hidden (R13)
        for e, we in zip(ids, w):
            gu = f64(layer["wgu_e"][e]) @ br[t]
            out[t] += we * (f64(layer["wd_e"][e]) @ _r("act", silu(gu[:F]) * gu[F:]))
    return out


def logits_from_hidden(model, h):
    cfg = model["cfg"]
    return _r("xnf", rmsnorm(h, model["final_norm"], cfg["rms_eps"])) @ f64(model["lm_head"]).T


def layer_forward(layer, cfg, h, pos):
    """One decoder layer over a whole causal sequence: h [T, d] entering the layer at positions pos [T] -> (h leaving it, k, v).
    (The body of forward_full's loop, callable on its own so that a test can feed it a given residual stream layer by layer.)"""
    T = h.shape[0]
    a = _r("xn", rmsnorm(h, layer["attn_norm"], cfg["rms_eps"]))
    q, k, v = qkv_project(layer, cfg, a, pos)
    o = np.empty((T, cfg["n_q_heads"], cfg["head_dim"]))
    for t in range(T):                                       # causal: position t sees keys 0..t
        o[t] = attention_one(q[t], k[: t + 1], v[: t + 1], cfg["n_kv_heads"])
    h = h + _r("ao", o.reshape(T, -1)) @ f64(layer["wo"]).T
    b = rmsnorm(h, layer["mlp_norm"], cfg["rms_eps"])
    h = h + mlp(layer, cfg, b)
    return h, k, v


def forward_full(model, tokens, return_kv=False, last=None):
    """THE DEFINITION: causal forward over tokens [T] -> logits [T, V] (and per-layer K,V).
    last = n returns the logits of the last n positions only ([n, V]; the rows of the full result, nothing else
    changes): a long teacher-forced history at vocab 151 936 would otherwise need T x V doubles."""
    cfg = model["cfg"]
    tokens = np.asarray(tokens, dtype=np.int64)
    T = tokens.shape[0]
    pos = np.arange(T)
    h = f64(model["embed"])[tokens]                          # [T, d]
    kv = []
    for layer in model["layers"]:
        h, k, v = layer_forward(layer, cfg, h, pos)
        kv.append((k, v))
    logits = logits_from_hidden(model, h if last is None else h[T - last:])
    return (logits, kv) if return_kv else logits


def prefill(model, prompt):
    """Prompt forward (one prompt q_i feeds all M'_i samples).
    Returns (z0 = logits at the last prompt position [V], kv = per-layer (K,V) [P,Hkv,hd])."""
    logits, kv = forward_full(model, prompt, return_kv=True)
    return logits[-1], kv


def decode_one(model, kv, token, pos):
    """Forward of ONE token at position pos over this row's own KV list `kv`
    (list over layers of [K, V] arrays, extended in place).  Returns logits [V]."""
    cfg = model["cfg"]
    h = f64(model["embed"])[int(token)][None, :]             # [1, d]
    for l, layer in enumerate(model["layers"]):
        a = _r("xn", rmsnorm(h, layer["attn_norm"], cfg["rms_eps"]))
        q, k, v = qkv_project(layer, cfg, a, np.array([pos]))
        K = np.concatenate([kv[l][0], k], axis=0)
        V = np.concatenate([kv[l][1], v], axis=0)
        kv[l] = (K, V)
        o = attention_one(q[0], K, V, cfg["n_kv_heads"])
        h = h + _r("ao", o.reshape(1, -1)) @ f64(layer["wo"]).T
        b = rmsnorm(h, layer["mlp_norm"], cfg["rms_eps"])
        h = h + mlp(layer, cfg, b)
    return logits_from_hidden(model, h)[0]
