"""Lock-step group rollout (oracle; test infrastructure only).

Two implementations that must agree (tests/test_oracle_rollout.py):

rollout_stepwise  the algorithm, step by step: every ACTIVE row emits
                  one token per step; after each step every open prompt applies the
                  DARTS rule (oracle.selection.group_rule): EARLY prompts stop as soon as
                  K VALID trajectories exist ("halted immediately once M
                  valid trajectories are collected"), DUAL prompts wait for the whole pool
                  (:224 "the full M'_i pool is required to identify the longest").
rollout_plain     the plain definition: roll every (i,j) out to its own end with no
                  pruning, then select.  With lock-step decoding completion order is
                  length order and the Philox key (seed,i,j,s) makes a trajectory
                  independent of its batch, so for an EARLY prompt the stepwise result is
                  exactly "the K smallest (len, j) among VALID" of the full pool, and the
                  pruned rows are the full trajectories cut at the closing step.

Rows are numbered group-major: row r = sum_{i'<i} Kp[i'] + j.
Each row owns a private copy of its prompt's KV (no prefix sharing here, on purpose:
"prefix-shared == unshared" is then a real check of the GPU path).

Returned dict: tokens [R, max_new] int32 (-1 beyond len), len [R], status [R],
sel [G, K] (sample indices j), sel_mask [G], close_step [G], n_steps,
n_generated_tokens (all rows, incl. pruned), n_kept_tokens, margins [R, max_new],
logprobs [R, max_new] (log softmax(z/T) of the token the sampler drew at each step),
oracle_tokens [R, max_new] (the oracle's own argmax, differs from `tokens` only under
teacher forcing), logits (dict (r,s)->z, only if keep_logits).
"""
import numpy as np

from . import ACTIVE, VALID, TRUNC, PRUNED, MODE_AUTO
from .sampling import sample_token, token_logprob
from .selection import apply_stop, compact, group_mode, group_rule, sel_mask, select_dual
from . import transformer as _tf
from .transformer import decode_one, prefill


def _setup(prompts, Kp):
    G = len(prompts)
    Kp = [int(k) for k in Kp]
    offs = np.concatenate([[0], np.cumsum(Kp)]).astype(np.int64)
    R = int(offs[-1])
    row_i = np.repeat(np.arange(G), Kp)
    row_j = np.concatenate([np.arange(k) for k in Kp]) if R else np.zeros(0, dtype=np.int64)
    return G, Kp, offs, R, row_i, row_j


def _finish(out, G, K, offs):
    kept = 0
    for i in range(G):
        for j in out["sel"][i]:
            kept += int(out["len"][offs[i] + j])
    out["n_generated_tokens"] = int(np.sum(out["len"]))
    out["n_kept_tokens"] = kept
    return out


def rollout_stepwise(model, prompts, Kp, K, max_new, T, seed, forced_len=None, L_long=1,
                     M_up=None, mode=MODE_AUTO, eos_id=None, teacher=None, keep_logits=False,
                     logit_filter=None, routing=None):
    """routing (MoE, optional; R13 teacher-forced routing): dict with ("prefill", i) -> expert ids [L][P_i][top_k]
    and (r, s) -> [L][top_k] for every decode step s >= 1 of row r; the result then carries route_regret[(r, s)], the largest regret
    over the layers of that forward (step 0: over the layers and positions of the prompt's prefill) — see
    oracle.transformer.ROUTE_OVERRIDE."""
    cfg = model["cfg"]
    eos_id = cfg["vocab"] - 1 if eos_id is None else eos_id
    M_up = 2 * K if M_up is None else M_up
    G, Kp, offs, R, row_i, row_j = _setup(prompts, Kp)

    z0, kv0, gap0 = [], [], []
    router_gap = {}                                          # (r, s) -> smallest router gap seen (R13; MoE models only)
    regret0, route_regret = [], {}
    for i in range(G):                                       # one prefill per prompt (:134)
        _tf.ROUTER_GAPS = [] if keep_logits else None
        if routing is not None:
            ids = np.asarray(routing[("prefill", i)])
            _tf.ROUTE_OVERRIDE, _tf.ROUTE_REGRET = iter(ids.reshape(-1, ids.shape[-1])), []
        z, kv = prefill(model, prompts[i])
        if routing is not None:
            regret0.append(max(_tf.ROUTE_REGRET))
            _tf.ROUTE_OVERRIDE = _tf.ROUTE_REGRET = None
        gap0.append(min(_tf.ROUTER_GAPS) if _tf.ROUTER_GAPS else np.inf)
        z0.append(z)
        kv0.append(kv)
    kv = [[(a.copy(), b.copy()) for a, b in kv0[row_i[r]]] for r in range(R)]  # private copies

    tokens = -np.ones((R, max_new), dtype=np.int32)
    otok = -np.ones((R, max_new), dtype=np.int32)
    margins = np.full((R, max_new), np.nan)
    logprobs = np.full((R, max_new), np.nan)                # of the DRAWN token (before a forced EOS or a teacher replaces it)
    length = np.zeros(R, dtype=np.int32)
    status = np.full(R, ACTIVE, dtype=np.uint8)
    sel = -np.ones((G, K), dtype=np.int32)
    mask = np.zeros(G, dtype=np.uint32)
    close_step = -np.ones(G, dtype=np.int32)
    logits = {}

    active = list(range(R))
    s = 0
    n_active_hist = []
    while active:
        n_active_hist.append(len(active))
        for r in active:
            i, j = int(row_i[r]), int(row_j[r])
            if s == 0:
                z = z0[i]
                gap = gap0[i]
                if routing is not None:
                    route_regret[(r, 0)] = regret0[i]
            else:
                _tf.ROUTER_GAPS = [] if keep_logits else None
                if routing is not None:
                    _tf.ROUTE_OVERRIDE, _tf.ROUTE_REGRET = iter(np.asarray(routing[(r, s)])), []
                z = decode_one(model, kv[r], tokens[r, s - 1], len(prompts[i]) + s - 1)
                if routing is not None:
                    route_regret[(r, s)] = max(_tf.ROUTE_REGRET)
                    _tf.ROUTE_OVERRIDE = _tf.ROUTE_REGRET = None
                gap = min(_tf.ROUTER_GAPS) if _tf.ROUTER_GAPS else np.inf
            if keep_logits and (logit_filter is None or logit_filter(r, s)):
                logits[(r, s)] = z.copy()
                router_gap[(r, s)] = gap
            tok, margin = sample_token(z, T, seed, i, j, s)
            otok[r, s], margins[r, s] = tok, margin
            logprobs[r, s] = token_logprob(z, T, tok)
            if teacher is not None:
                tok = int(teacher[r][s])
            length[r] = s + 1
            fl = None if forced_len is None else int(forced_len[i][j])
            tokens[r, s], status[r] = apply_stop(tok, s + 1, fl, eos_id, max_new)
        for i in range(G):
            if close_step[i] >= 0:
                continue
            lo, hi = offs[i], offs[i + 1]
            st = status[lo:hi]                               # view: PRUNED written in place
            chosen = group_rule(length[lo:hi], st, Kp[i], K, L_long, M_up, mode)
            if chosen is not None:
                sel[i], mask[i], close_step[i] = chosen, sel_mask(chosen), s
        active = compact(active, status)
        s += 1

    out = dict(tokens=tokens, len=length, status=status, sel=sel, sel_mask=mask,
               close_step=close_step, n_steps=s, margins=margins, logprobs=logprobs, oracle_tokens=otok,
               logits=logits, router_gap=router_gap, route_regret=route_regret, n_active_hist=n_active_hist)
    _tf.ROUTER_GAPS = None
    return _finish(out, G, K, offs)


def rollout_one(model, prompt, i, j, max_new, T, seed, forced, eos_id):
    """One trajectory to its own end, alone (batch of one)."""
    z, kv0 = prefill(model, prompt)
    kv = [(a.copy(), b.copy()) for a, b in kv0]
    toks, s, st = [], 0, ACTIVE
    while st == ACTIVE:
        if s > 0:
            z = decode_one(model, kv, toks[-1], len(prompt) + s - 1)
        tok, _ = sample_token(z, T, seed, i, j, s)
        tok, st = apply_stop(tok, s + 1, forced, eos_id, max_new)
        toks.append(tok)
        s += 1
    return toks, st


def rollout_plain(model, prompts, Kp, K, max_new, T, seed, forced_len=None, L_long=1,
                  M_up=None, mode=MODE_AUTO, eos_id=None):
    """Full rollout of every trajectory, then the rule as a plain sort."""
    cfg = model["cfg"]
    eos_id = cfg["vocab"] - 1 if eos_id is None else eos_id
    M_up = 2 * K if M_up is None else M_up
    G, Kp, offs, R, row_i, row_j = _setup(prompts, Kp)
    tokens = -np.ones((R, max_new), dtype=np.int32)
    length = np.zeros(R, dtype=np.int32)
    status = np.zeros(R, dtype=np.uint8)
    sel = -np.ones((G, K), dtype=np.int32)
    mask = np.zeros(G, dtype=np.uint32)
    close_step = -np.ones(G, dtype=np.int32)
    for i in range(G):
        full = []
        for j in range(Kp[i]):
            fl = None if forced_len is None else int(forced_len[i][j])
            full.append(rollout_one(model, prompts[i], i, j, max_new, T, seed, fl, eos_id))
        flen = [len(t) for t, _ in full]
        fst = [st for _, st in full]
        valid = sorted((flen[j], j) for j in range(Kp[i]) if fst[j] == VALID)
        if group_mode(Kp[i], K, M_up, mode) == "EARLY" and len(valid) >= K:
            # the K smallest (len, j) among VALID; the group closes when the K-th of them ends
            chosen = [j for _, j in valid[:K]]
            t_close = valid[K - 1][0]
            for j in range(Kp[i]):
                r = offs[i] + j
                if flen[j] <= t_close:
                    length[r], status[r] = flen[j], fst[j]
                else:                                        # stopped by the early-stop signal
                    length[r], status[r] = t_close, PRUNED
                tokens[r, : length[r]] = full[j][0][: length[r]]
            close_step[i] = t_close - 1
        else:
            for j in range(Kp[i]):
                r = offs[i] + j
                length[r], status[r] = flen[j], fst[j]
                tokens[r, : flen[j]] = full[j][0]
            if group_mode(Kp[i], K, M_up, mode) == "EARLY":
                # fewer than K valid: all VALID by (len,j), then TRUNC by (len,j)  (R8)
                trunc = sorted((flen[j], j) for j in range(Kp[i]) if fst[j] == TRUNC)
                chosen = [j for _, j in (valid + trunc)[:K]]
            else:
                chosen = select_dual(flen, fst, K, L_long)
            close_step[i] = max(flen) - 1
        sel[i], mask[i] = chosen, sel_mask(chosen)
    out = dict(tokens=tokens, len=length, status=status, sel=sel, sel_mask=mask,
               close_step=close_step, n_steps=int(np.max(close_step)) + 1 if G else 0)
    return _finish(out, G, K, offs)
