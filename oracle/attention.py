"""Decode attention for one row over [shared prefix || own suffix] (oracle; test infrastructure only).

BASELINE.json config 2 / SURVEY.md §8(a) row 5: for every row r of prompt i and
every q-head h,
        out[r,h] = softmax( q[r,h] . K^T / sqrt(hd) ) V
over the keys  K = [ K_prefix(i) ; K_suffix(r) ]  (prefix length P, suffix length t_r).
"K' redundant trajectories are generated autoregressively over a shared prompt
KV cache" (north_star; §4.1.1 — the M'_i samples share prompt q_i).

The oracle never shares anything: it concatenates a private copy of the prefix
with the row's suffix and evaluates the textbook formula in float64.  The
split-KV / log-sum-exp merge that the GPU kernel uses is written out separately
(`merge_partials`) only so that tests can pin "split + merge == unsplit".
"""
import numpy as np

from .transformer import attention_one, f64


def attention_row(q, K_prefix, V_prefix, K_suffix, V_suffix):
    """q [Hq,hd]; K_prefix,V_prefix [P,Hkv,hd]; K_suffix,V_suffix [t,Hkv,hd] -> [Hq,hd]."""
    K = np.concatenate([f64(K_prefix), f64(K_suffix)], axis=0)
    V = np.concatenate([f64(V_prefix), f64(V_suffix)], axis=0)
    return attention_one(q, K, V, K.shape[1])


def partial(q, K, V):
    """Un-normalised partial over a chunk of keys for one (q-head, kv-head) pair:
    returns (m = max score, l = sum exp(s-m), acc = sum exp(s-m) v)."""
    q, K, V = f64(q), f64(K), f64(V)
    s = K @ q / np.sqrt(q.shape[-1])
    m = np.max(s)
    e = np.exp(s - m)
    return m, np.sum(e), e @ V


def merge_partials(parts):
    """Log-sum-exp merge of [(m,l,acc), ...] -> normalised output."""
    M = max(p[0] for p in parts)
    l = sum(p[1] * np.exp(p[0] - M) for p in parts)
    acc = sum(p[2] * np.exp(p[0] - M) for p in parts)
    return acc / l
